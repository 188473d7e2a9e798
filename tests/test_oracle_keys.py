"""Pins for the oracle's Morton codec and sort/linearise (PAPER.md:82-97 Alg. 1, :122-128 Alg. 3).

None of these re-types the oracle's formula: they check worked values, the paper's
structural statements (Eq. 7 first child = key + 1, siblings consecutive, x lowest) and
the pointer tree's own geometric DFS order against the integer order of the IDs.
"""
import numpy as np
import pytest

import oracle


def test_textbook_interleave_values():
    # Z-order table with x in the low bit ("x^k = x_3^k x_2^k x_1^k"):
    # (x=3, y=5) -> y2 x2 y1 x1 y0 x0 = 1 0 0 1 1 1 = 39 ; (x=7, y=0) -> 010101 = 21
    assert oracle.raw_id(2, 3, 3, (3, 5)) == 39
    assert oracle.raw_id(2, 3, 3, (7, 0)) == 21
    assert oracle.raw_id(2, 3, 3, (0, 7)) == 42
    # 3-D: (1,0,0) -> 1 ; (0,1,0) -> 2 ; (0,0,1) -> 4 ; (1,1,1) at 2 bits (3,3,3) -> 63
    assert oracle.raw_id(3, 1, 1, (1, 0, 0)) == 1
    assert oracle.raw_id(3, 1, 1, (0, 1, 0)) == 2
    assert oracle.raw_id(3, 1, 1, (0, 0, 1)) == 4
    assert oracle.raw_id(3, 2, 2, (3, 3, 3)) == 63
    # (x=2,y=3,z=1) bits: level-1 digit (z1 y1 x1) = 0 1 1 = 3 ; level-0 digit (z0 y0 x0) = 1 1 0 = 6 -> 3*8+6 = 30
    assert oracle.raw_id(3, 2, 2, (2, 3, 1)) == 30


def test_key_layout_padding_and_depth():
    # reading A-1/A-2: key = raw << dim*(Dmax-D) << 5 | D.  Root is key 0.
    assert oracle.encode(2, 8, 0, (0, 0)) == 0
    assert oracle.encode(3, 9, 0, (0, 0, 0)) == 0
    # a level-1 cell at x = half the domain in 2-D, Dmax = 4: raw = 1, padded by 2*3 bits, depth 1
    assert oracle.encode(2, 4, 1, (8, 0)) == ((1 << 6) << 5) | 1
    assert oracle.encode(2, 4, 1, (0, 8)) == ((2 << 6) << 5) | 1
    assert oracle.encode(3, 4, 2, (4, 0, 12)) == (((0b100_101) << 6) << 5) | 2


@pytest.mark.parametrize("dim,maxl", [(2, 8), (2, 29), (3, 12), (3, 19)])
def test_roundtrip_and_structure(dim, maxl):
    rng = np.random.default_rng(7)
    for _ in range(300):
        level = int(rng.integers(0, maxl + 1))
        w = 1 << (maxl - level)
        x = [int(rng.integers(0, 1 << level)) * w for _ in range(dim)]
        k = oracle.encode(dim, maxl, level, x)
        assert k < (1 << (dim * maxl + 5))
        assert oracle.decode(dim, maxl, k) == (level, tuple(x))
        assert (k & 31) == level
        if level < maxl:
            # Eq. 7 case 3: the first child is key + 1
            assert oracle.encode(dim, maxl, level + 1, x) == k + 1
            # siblings: raw-ID increment 1, child c offset bits = c, x lowest (:210)
            h = w >> 1
            raws = []
            for c in range(1 << dim):
                xc = [x[a] + (((c >> a) & 1) * h) for a in range(dim)]
                raws.append(oracle.raw_id(dim, maxl, level + 1, xc))
            assert raws == [raws[0] + c for c in range(1 << dim)]
            # descendants sort after the ancestor and before the ancestor's successor
            xl = [x[a] + w - 1 for a in range(dim)]
            klast = oracle.encode(dim, maxl, maxl, xl)
            assert k < klast
            nxt = k + (1 << (dim * (maxl - level) + 5))
            assert klast < nxt


@pytest.mark.parametrize("dim,base,maxl", [(2, 3, 8), (3, 2, 6), (3, 3, 12)])
def test_uniform_base_tree(dim, base, maxl):
    t = oracle.Tree(dim, base, maxl)
    k = t.keys()
    n = 1 << (dim * base)
    assert k.size == n
    # SURVEY 8(c) pin: key i = (i << dim*(Dmax-base)) << 5 | base
    want = (np.arange(n, dtype=np.uint64) << np.uint64(dim * (maxl - base) + 5)) | np.uint64(base)
    assert np.array_equal(k, want)
    assert t.dfs_is_sorted()


def test_dfs_order_equals_sorted_order_after_adaptation():
    # geometric child order of the pointer tree (anchor + i*Delta/2, x lowest) == integer order of IDs
    rng = np.random.default_rng(3)
    for dim, base, maxl in [(2, 2, 7), (3, 1, 5)]:
        t = oracle.Tree(dim, base, maxl, [1] * dim)
        for _ in range(4):
            f = rng.integers(-1, 2, t.num_leaves()).astype(np.int8)
            t.adapt(f)
            t.balance()
            assert t.dfs_is_sorted()
            k = t.keys()
            assert np.all(k[1:] > k[:-1])


def _boxes(dim, maxl, keys):
    out = []
    for k in keys:
        lvl, x = oracle.decode(dim, maxl, int(k))
        out.append((lvl, x, 1 << (maxl - lvl)))
    return out


def _linearise_bruteforce(dim, maxl, keys):
    """Drop duplicates and every key whose box strictly contains another key's box (O(n^2))."""
    uniq = sorted(set(int(k) for k in keys))
    bx = _boxes(dim, maxl, uniq)
    keep = []
    for i, (li, xi, wi) in enumerate(bx):
        has_desc = False
        for j, (lj, xj, wj) in enumerate(bx):
            if lj > li and all(xi[a] <= xj[a] < xi[a] + wi for a in range(dim)):
                has_desc = True
                break
        if not has_desc:
            keep.append(uniq[i])
    return np.array(keep, dtype=np.uint64)


@pytest.mark.parametrize("dim,maxl", [(2, 6), (3, 4)])
def test_sort_linearise_vs_bruteforce(dim, maxl):
    rng = np.random.default_rng(11)
    for trial in range(6):
        keys = []
        for _ in range(250):
            level = int(rng.integers(0, maxl + 1))
            w = 1 << (maxl - level)
            x = [int(rng.integers(0, 1 << level)) * w for _ in range(dim)]
            keys.append(oracle.encode(dim, maxl, level, x))
        keys += keys[:40]  # duplicates
        keys = np.array(keys, dtype=np.uint64)
        rng.shuffle(keys)
        got = oracle.sort_linearise(dim, maxl, keys)
        want = _linearise_bruteforce(dim, maxl, keys)
        assert np.array_equal(got, want)


def test_sort_linearise_adversarial():
    dim, maxl = 2, 5
    k0 = oracle.encode(dim, maxl, 3, (4, 8))
    # all equal
    assert np.array_equal(oracle.sort_linearise(dim, maxl, np.full(17, k0, np.uint64)), [k0])
    # a chain root -> ... -> finest along the first-child path collapses to the finest
    chain = np.array([oracle.encode(dim, maxl, l, (0, 0)) for l in range(maxl + 1)], np.uint64)
    assert np.array_equal(oracle.sort_linearise(dim, maxl, chain[::-1].copy()), [chain[-1]])
    # reversed sorted uniform level: unchanged set, ascending
    t = oracle.Tree(dim, 3, maxl)
    k = t.keys()
    assert np.array_equal(oracle.sort_linearise(dim, maxl, k[::-1].copy()), k)
    # keys differing only in the top / bottom digit
    a = oracle.encode(dim, maxl, maxl, (0, 0))
    b = oracle.encode(dim, maxl, maxl, (1, 0))
    c = oracle.encode(dim, maxl, maxl, (16, 16))
    assert np.array_equal(oracle.sort_linearise(dim, maxl, np.array([c, b, a], np.uint64)), [a, b, c])
    # empty
    assert oracle.sort_linearise(dim, maxl, np.zeros(0, np.uint64)).size == 0


def test_build_from_keys_roundtrip_and_incomplete():
    rng = np.random.default_rng(5)
    t = oracle.Tree(3, 1, 5, [0, 0, 0])
    for _ in range(3):
        t.adapt(rng.integers(0, 2, t.num_leaves()).astype(np.int8))
    k = t.keys()
    # add ancestors and duplicates, shuffle: linearise must recover the leaf set
    extra = [oracle.encode(3, 5, 0, (0, 0, 0)), oracle.encode(3, 5, 1, (16, 0, 0))]
    mixed = np.concatenate([k, k[:50], np.array(extra, np.uint64)])
    rng.shuffle(mixed)
    t2 = oracle.Tree(3, 1, 5, [0, 0, 0], keys=mixed)
    assert np.array_equal(t2.keys(), k)
    with pytest.raises(oracle.OracleError):
        oracle.Tree(3, 1, 5, [0, 0, 0], keys=k[1:])  # a hole
