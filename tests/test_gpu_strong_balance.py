"""GPU parity for SURVEY 8(f)-3: strong 2:1 balance (connectivity 1 = faces,
2 = + edges, 3 = + corners; reading C-9) against the oracle: keys, leaf order, sweep count and
total splits bit-exact, frontier sweeps == full sweeps, face query on the result."""
import numpy as np
import pytest
import torch

import oracle
import parity as P
from paper_2306_06744_b200 import lt
from paper_2306_06744_b200 import workloads as W

pytestmark = pytest.mark.gpu


def random_pair(dim, base, maxl, periodic, seed, cycles=4, frac=0.25):
    rng = np.random.default_rng(seed)
    dom = [0.0] * dim + [1.0] * dim
    gt = lt.Tree(dim, base, maxl, dom, periodic)
    ot = oracle.Tree(dim, base, maxl, periodic)
    for _ in range(cycles):
        f = (rng.random(ot.num_leaves()) < frac).astype(np.int8)
        ot.adapt(f); ot.drop_snapshot()
        gt.adapt(torch.from_numpy(f).cuda())
    P.assert_keys_equal(gt, ot, "unbalanced input")
    return gt, ot


CASES = [(2, 1, 7, (0, 0), 1), (2, 1, 7, (1, 1), 2), (2, 0, 8, (1, 0), 3),
         (3, 1, 5, (0, 0, 0), 4), (3, 1, 5, (1, 1, 1), 5), (3, 0, 6, (0, 1, 0), 6)]


@pytest.mark.parametrize("dim,base,maxl,periodic,seed", CASES)
@pytest.mark.parametrize("full", [0, 1])
def test_strong_balance_matches_oracle(dim, base, maxl, periodic, seed, full):
    for conn in range(1, dim + 1):
        gt, ot = random_pair(dim, base, maxl, periodic, seed)
        gt.set_option(lt.LT_OPT_BALANCE_FULL_SWEEPS, full)
        it_o = ot.balance(conn)
        it_g = gt.balance(conn)
        P.assert_keys_equal(gt, ot, "conn %d" % conn)
        assert it_g == it_o
        assert gt.balance() == 0  # the option is sticky; a balanced tree is left alone (C-7)
        P.assert_faces_equal(gt.connect(), ot.connect(), "connect after conn %d" % conn)


@pytest.mark.parametrize("dim", [2, 3])
def test_deep_diagonal_ripple(dim):
    # the leaf touching the domain centre from the all-minus side is refined to max level without
    # balancing; ONE strong balance must then cascade through every level (deferred balance)
    maxl = 11 if dim == 2 else 9
    dom = [0.0] * dim + [1.0] * dim
    results = []
    for conn in range(1, dim + 1):
        gt, ot = lt.Tree(dim, 1, maxl, dom), oracle.Tree(dim, 1, maxl)
        for _ in range(maxl - 1):
            lvl, xyz = ot.leaf_boxes()
            w = 1 << (maxl - lvl.astype(np.int64))
            f = np.all(xyz[:, :dim].astype(np.int64) + w[:, None] == (1 << (maxl - 1)), axis=1).astype(np.int8)
            ot.adapt(f); ot.drop_snapshot()
            gt.adapt(torch.from_numpy(f).cuda())
        it_o, it_g = ot.balance(conn), gt.balance(conn)
        P.assert_keys_equal(gt, ot, "diagonal conn %d" % conn)
        assert it_o == it_g and it_g >= maxl - 3
        results.append(gt.num_leaves())
    assert all(a < b for a, b in zip(results, results[1:]))


@pytest.mark.parametrize("conn", [2, 3])
def test_cycles_with_strong_balance(conn):
    # the whole cycle with the paper's strong balance: vortex-tube flags (config 4 shrunk),
    # faces, map and transfer against the oracle every cycle
    cfg = dict(W.CONFIGS["c4"], base=3, maxl=6)
    gt, ot = P.new_pair(cfg)
    p, nvars = cfg["p"], cfg["nvars"]
    uo = P.initial_u(cfg, ot)
    for c in range(4):
        f = P.host_flags(cfg, c, ot)
        ot.adapt(f)
        gt.adapt(torch.from_numpy(f).cuda())
        assert ot.balance(conn) == gt.balance(conn)
        P.assert_keys_equal(gt, ot, "cycle %d" % c)
        P.assert_faces_equal(gt.connect(), ot.connect(), "cycle %d" % c)
        un_o = ot.transfer(uo, p, nvars)
        un_g = gt.transfer(torch.from_numpy(uo).cuda(), p, nvars)
        gt.sync()
        P.assert_u_close(un_g, un_o, "cycle %d" % c)
        uo = un_o


@pytest.mark.parametrize("dim,base,maxl,periodic,conn", [(2, 2, 8, (1, 0), 2), (3, 1, 6, (1, 1, 1), 2),
                                                         (3, 2, 6, (0, 0, 0), 3), (3, 1, 6, (0, 1, 0), 3)])
def test_strong_balance_after_adapt_uses_the_adapt_frontier(dim, base, maxl, periodic, conn):
    # a tree balanced with connectivity `conn` is adapted: the first sweep of the next strong balance looks only
    # at the leaves lt_adapt created -- refined leaves as GROUP entries over the 18 / 26 directions, merged
    # parents from their own side across faces, edges and corners.  Coarsening-heavy and refining-heavy
    # random flags in turn; trees, sweep counts and faces must be the oracle's and the full sweeps'.  A
    # balance with a STRONGER connectivity than the tree was last balanced with must not use the list.
    rng = np.random.default_rng(dim * 1000 + conn * 10 + maxl)
    dom = [0.0] * dim + [1.0] * dim
    gt, gf = lt.Tree(dim, base, maxl, dom, periodic), lt.Tree(dim, base, maxl, dom, periodic)
    gf.set_option(lt.LT_OPT_BALANCE_FULL_SWEEPS, 1)
    ot = oracle.Tree(dim, base, maxl, periodic)
    for c in range(10):
        pr = [0.55, 0.33, 0.12] if c % 2 else [0.25, 0.45, 0.30]
        f = rng.choice(np.array([-1, 0, 1], np.int8), size=ot.num_leaves(), p=pr)
        # cycle 6 balances across faces only, cycle 7 goes back to `conn`: its tree was balanced with
        # connectivity 1, so lt_adapt's list is not enough and the first sweep must be a full one
        k = 1 if c == 6 else conn
        ot.adapt(f); it_o = ot.balance(k); ot.drop_snapshot()
        for g in (gt, gf):
            g.adapt(torch.from_numpy(f).cuda())
            assert g.balance(k) == it_o, "cycle %d" % c
            P.assert_keys_equal(g, ot, "cycle %d" % c)
        if c in (3, 9):
            P.assert_faces_equal(gt.connect(), ot.connect(), "cycle %d" % c)


def test_construct_then_strong_balance():
    cfg = W.POINT_CLOUDS["pc3_small"]
    pts = W.surface_points(cfg).numpy()
    dom = [cfg["lo"]] * 3 + [cfg["hi"]] * 3
    for conn in (2, 3):
        ot = oracle.Tree(3, cfg["base"], cfg["maxl"], cfg["periodic"], points=pts, domain=dom)
        gt = lt.build_from_points(3, cfg["base"], cfg["maxl"], torch.from_numpy(pts).cuda(), dom, cfg["periodic"])
        assert ot.balance(conn) == gt.balance(conn)
        P.assert_keys_equal(gt, ot, "construct + conn %d" % conn)


def test_bad_connectivity():
    gt = lt.Tree(2, 1, 4)
    with pytest.raises(lt.LtError):
        gt.balance(3)
    with pytest.raises(lt.LtError):
        gt.balance(0)
    assert gt.balance(2) == 0
