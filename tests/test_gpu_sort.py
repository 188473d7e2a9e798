"""GPU parity for a-3: LSD radix sort + linearisation (Alg. 3) and lt_build_from_keys,
against numpy's sort and the oracle's std::sort + reverse/unique/reverse."""
import numpy as np
import pytest
import torch

import oracle
import parity as P
from paper_2306_06744_b200 import lt

pytestmark = pytest.mark.gpu


def to_dev(k):
    return torch.from_numpy(np.ascontiguousarray(k, np.uint64).view(np.int64)).cuda()


def random_keys(rng, dim, maxl, n, lo_level=0):
    lvl = rng.integers(lo_level, maxl + 1, n)
    out = np.zeros(n, np.uint64)
    for i in range(n):
        x = rng.integers(0, 1 << maxl, 3).astype(np.uint32)
        x[dim:] = 0
        out[i] = oracle.encode(dim, maxl, int(lvl[i]), x)
    return out


@pytest.mark.parametrize("n", [0, 1, 2, 255, 2048, 2049, 100003, 1 << 20])
def test_sort_random(n):
    rng = np.random.default_rng(n)
    dim, maxl = 3, 9
    bits = dim * maxl + 5
    k = rng.integers(0, 1 << bits, n, dtype=np.uint64)
    out = lt.sort_keys(dim, maxl, to_dev(k))
    assert np.array_equal(P.u64(out), np.sort(k))


@pytest.mark.parametrize("dim,maxl", [(2, 29), (3, 19), (2, 3)])
def test_sort_adversarial(dim, maxl):
    bits = dim * maxl + 5
    n = 50000
    rng = np.random.default_rng(bits)
    cases = [
        np.full(n, (1 << bits) - 1, np.uint64),                           # all equal
        np.arange(n, 0, -1).astype(np.uint64),                            # reversed
        (rng.integers(0, 2, n).astype(np.uint64) << np.uint64(bits - 1)),  # only the top bit differs
        rng.integers(0, 2, n).astype(np.uint64),                          # only the bottom bit differs
        (rng.integers(0, 256, n).astype(np.uint64) << np.uint64(8 * ((bits - 1) // 8))),  # top digit only
    ]
    for k in cases:
        k = k & np.uint64((1 << bits) - 1)
        assert np.array_equal(P.u64(lt.sort_keys(dim, maxl, to_dev(k))), np.sort(k))


@pytest.mark.parametrize("dim,maxl", [(2, 6), (3, 4), (3, 9)])
def test_sort_linearise_matches_oracle(dim, maxl):
    rng = np.random.default_rng(dim * 10 + maxl)
    k = random_keys(rng, dim, maxl, 4000)
    k = np.concatenate([k, k[:500]])  # duplicates
    rng.shuffle(k)
    ref = oracle.sort_linearise(dim, maxl, k)
    out = lt.sort_keys(dim, maxl, to_dev(k), linearise=True)
    assert np.array_equal(P.u64(out), ref)


def test_build_from_keys_roundtrip_and_overlaps():
    """A shuffled leaf set plus some of its ancestors and duplicates linearises back to the
    same tree (Alg. 3 drops ancestors and duplicates); an incomplete set is rejected."""
    from paper_2306_06744_b200 import workloads as W
    cfg = W.CONFIGS["c3b"]
    gt, ot = P.new_pair(cfg)
    for c in range(6):
        f = P.host_flags(cfg, c, ot)
        ot.adapt(f); ot.balance()
        gt.adapt(torch.from_numpy(f).cuda()); gt.balance()
    keys = ot.keys()
    rng = np.random.default_rng(5)
    lvl, xyz = ot.leaf_boxes()
    anc = []
    for i in rng.choice(keys.size, 100, replace=False):  # ancestors of random leaves
        l = int(lvl[i])
        if l > cfg["base"]:
            la = int(rng.integers(cfg["base"], l))
            anc.append(oracle.encode(3, cfg["maxl"], la, xyz[i]))
    mixed = np.concatenate([keys, np.array(anc, np.uint64), keys[:50]])
    rng.shuffle(mixed)
    g2 = lt.build_from_keys(3, cfg["base"], cfg["maxl"], to_dev(mixed), None, cfg["periodic"])
    assert np.array_equal(P.u64(g2.keys()), keys)
    o2 = oracle.Tree(3, cfg["base"], cfg["maxl"], cfg["periodic"], keys=mixed)
    assert np.array_equal(o2.keys(), keys)
    P.assert_faces_equal(g2.connect(), ot.connect(), "built from keys")
    assert g2.balance() == 0
    with pytest.raises(lt.LtError) as ei:
        lt.build_from_keys(3, cfg["base"], cfg["maxl"], to_dev(np.delete(keys, 7)), None, cfg["periodic"])
    assert ei.value.status == lt.LT_ERR_INCOMPLETE
