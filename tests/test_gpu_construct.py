"""GPU parity for SURVEY 8(f)-1: tree construction from scattered points / octants (Alg. 2,
PAPER.md:105-120) and the full-depth 2:1 balance + face query that follow it (Alg. 4, 5),
against the pointer-tree oracle.  Bit-exact: keys, leaf order, balance iteration count, face
tables.  The points are generated ONCE on the host and the same bytes go to both sides."""
import numpy as np
import pytest
import torch

import oracle
import parity as P
from paper_2306_06744_b200 import lt
from paper_2306_06744_b200 import workloads as W

pytestmark = pytest.mark.gpu


def to_dev(k):
    return torch.from_numpy(np.ascontiguousarray(k, np.uint64).view(np.int64)).cuda()


def pair_from_points(cfg, pts):
    dim = cfg["dim"]
    dom = [cfg["lo"]] * dim + [cfg["hi"]] * dim
    ot = oracle.Tree(dim, cfg["base"], cfg["maxl"], cfg["periodic"], points=pts, domain=dom)
    gt = lt.build_from_points(dim, cfg["base"], cfg["maxl"], torch.from_numpy(pts).cuda(), dom, cfg["periodic"])
    return gt, ot


@pytest.mark.parametrize("name", ["pc_tiny", "pc2", "pc3_small"])
def test_points_construct_balance_connect(name):
    cfg = W.POINT_CLOUDS[name]
    pts = W.surface_points(cfg).numpy()
    gt, ot = pair_from_points(cfg, pts)
    P.assert_keys_equal(gt, ot, name + " completion")
    with pytest.raises(lt.LtError):
        gt.connect()  # not balanced yet (reading D-5)
    it_o, it_g = ot.balance(), gt.balance()
    P.assert_keys_equal(gt, ot, name + " balance")
    assert it_g == it_o and it_g >= 1
    P.assert_faces_equal(gt.connect(), ot.connect(), name + " connect")


@pytest.mark.parametrize("dim,base,maxl,n", [(3, 4, 8, 200000), (2, 3, 11, 300000), (3, 0, 7, 50000),
                                             (2, 0, 12, 5)])
def test_points_construct_larger(dim, base, maxl, n):
    # several fill tiles, ragged tail, large base-level gaps (3-D base 4: 4096 base cells)
    cfg = dict(dim=dim, base=base, maxl=maxl, lo=-1.0, hi=1.0, periodic=(0,) * dim,
               surface="torus" if dim == 3 else "sphere", seed=40 + maxl, n=n)
    pts = W.surface_points(cfg).numpy()
    gt, ot = pair_from_points(cfg, pts)
    P.assert_keys_equal(gt, ot, "completion")
    it_o, it_g = ot.balance(), gt.balance()
    P.assert_keys_equal(gt, ot, "balance")
    assert it_g == it_o
    Fg, Fo = gt.connect(), ot.connect()
    for k in ("n_conf", "n_hang", "n_bnd"):
        assert int(Fg[k]) == int(Fo[k])
    assert np.array_equal(Fg["nbr"].cpu().numpy(), Fo["nbr"])


def test_point_cell_edge_cases():
    # boundary, outside, exactly-on-cell-boundary and just-below points: the integer decision is
    # taken in fp64 with the same operation order on both sides (reading G-1)
    dim, base, maxl = 2, 1, 6
    xs = [0.0, 1.0, -0.5, 2.0, 5 / 64, np.nextafter(5 / 64, 0.0), 0.999999999999, 1e-300, 0.3, 1 / 3]
    pts = np.array([[x, y] for x in xs for y in xs[::-1]])
    cfg = dict(dim=dim, base=base, maxl=maxl, lo=0.0, hi=1.0, periodic=(0, 0))
    gt, ot = pair_from_points(cfg, pts)
    P.assert_keys_equal(gt, ot, "edge points")
    # non-dyadic domain
    cfg = dict(dim=dim, base=base, maxl=maxl, lo=-0.7, hi=2.9, periodic=(0, 0))
    rng = np.random.default_rng(9)
    pts = rng.uniform(-0.8, 3.0, (5000, 2))
    gt, ot = pair_from_points(cfg, pts)
    P.assert_keys_equal(gt, ot, "non-dyadic domain")


@pytest.mark.parametrize("dim,base,maxl", [(2, 0, 6), (2, 2, 7), (3, 1, 5), (3, 0, 4), (3, 2, 12)])
def test_octants_mixed_levels(dim, base, maxl):
    rng = np.random.default_rng(7 * dim + maxl)
    for n in (1, 2, 17, 400):
        keys = []
        for _ in range(n):
            l = int(rng.integers(base, maxl + 1))
            x = (rng.integers(0, 1 << l, 3) << (maxl - l)).astype(np.uint32) if l else np.zeros(3, np.uint32)
            x[dim:] = 0
            keys.append(oracle.encode(dim, maxl, l, x))
        keys = np.array(keys + keys[: n // 2], np.uint64)  # duplicates; ancestors arise by chance
        ot = oracle.Tree(dim, base, maxl, keys=keys, complete=True)
        gt = lt.build_complete_from_keys(dim, base, maxl, to_dev(keys))
        P.assert_keys_equal(gt, ot, "octants n=%d" % n)


def test_degenerate_inputs():
    # every point in one cell; max_level == base_level; a full uniform cover
    dom = [0.0, 0.0, 0.0, 1.0, 1.0, 1.0]
    pts = np.tile(np.array([[0.999, 0.999, 0.999]]), (1000, 1))
    gt = lt.build_from_points(3, 2, 9, torch.from_numpy(pts).cuda(), dom)
    ot = oracle.Tree(3, 2, 9, points=pts, domain=dom)
    P.assert_keys_equal(gt, ot, "single cell")
    assert gt.num_leaves() == 64 + 7 * 7
    gt = lt.build_from_points(3, 3, 3, torch.from_numpy(pts).cuda(), dom)
    P.assert_keys_equal(gt, oracle.Tree(3, 3, 3), "base == max")
    n = 32
    g = (np.arange(n) + 0.5) / n
    full = np.stack(np.meshgrid(g, g, indexing="ij"), -1).reshape(-1, 2)
    gt = lt.build_from_points(2, 1, 5, torch.from_numpy(full).cuda(), [0, 0, 1, 1])
    P.assert_keys_equal(gt, oracle.Tree(2, 5, 5), "uniform cover")


def test_bad_arguments():
    dom = [0.0, 0.0, 1.0, 1.0]
    pts = torch.rand(10, 2, dtype=torch.float64).cuda()
    with pytest.raises(lt.LtError):
        lt.build_from_points(2, 1, 5, pts, [0.0, 0.0, 0.0, 1.0])  # hi == lo
    bad = to_dev(np.array([oracle.encode(2, 6, 1, [0, 0])], np.uint64))
    with pytest.raises(lt.LtError):
        lt.build_complete_from_keys(2, 3, 6, bad)  # key above base level


def test_cycle_runs_on_constructed_tree():
    # the adaptation cycle (adapt -> balance -> connect -> transfer) on a tree that came from
    # Alg. 2 + Alg. 4 rather than from a uniform mesh
    cfg = W.POINT_CLOUDS["pc3_small"]
    pts = W.surface_points(cfg).numpy()
    gt, ot = pair_from_points(cfg, pts)
    ot.balance(), gt.balance()
    rng = np.random.default_rng(3)
    p, nvars = 2, 3
    uo = rng.uniform(-1, 1, (ot.num_leaves(), nvars, (p + 1) ** 3))
    for c in range(2):
        f = rng.integers(-1, 2, ot.num_leaves()).astype(np.int8)
        ot.adapt(f)
        gt.adapt(torch.from_numpy(f).cuda())
        assert ot.balance() == gt.balance()
        P.assert_keys_equal(gt, ot, "cycle %d" % c)
        P.assert_faces_equal(gt.connect(), ot.connect(), "cycle %d" % c)
        un_o = ot.transfer(uo, p, nvars)
        un_g = gt.transfer(torch.from_numpy(uo).cuda(), p, nvars)
        gt.sync()
        P.assert_u_close(un_g, un_o, "cycle %d transfer" % c)
        uo = un_o


@pytest.mark.parametrize("dim,maxl", [(2, 29), (3, 19)])
def test_maximum_depth_trees(dim, maxl):
    # key capacity (dim * max_level + 5 = 63 bits): construction, the full-depth ripple (one sweep per
    # level), the face query and one adaptation cycle on a handful of points at the deepest level
    rng = np.random.default_rng(maxl)
    dom = [0.0] * dim + [1.0] * dim
    pts = np.concatenate([rng.uniform(0, 1, (6, dim)), np.full((1, dim), 0.5 - 2.0 ** -30), np.zeros((1, dim)),
                          np.ones((1, dim))])
    ot = oracle.Tree(dim, 0, maxl, points=pts, domain=dom)
    gt = lt.build_from_points(dim, 0, maxl, torch.from_numpy(pts).cuda(), dom)
    P.assert_keys_equal(gt, ot, "deep completion")
    assert int(P.u64(gt.keys()).max() >> np.uint64(dim * maxl + 4)) == 1  # the top key bit is in use
    it_o, it_g = ot.balance(), gt.balance()
    assert it_o == it_g and it_g >= maxl - 4
    P.assert_keys_equal(gt, ot, "deep balance")
    P.assert_faces_equal(gt.connect(), ot.connect(), "deep connect")
    n_before = ot.num_leaves()
    f = rng.integers(-1, 2, n_before).astype(np.int8)
    ot.adapt(f); gt.adapt(torch.from_numpy(f).cuda())
    assert ot.balance() == gt.balance()
    P.assert_keys_equal(gt, ot, "deep cycle")
    p, nvars = 1, 2
    uo = rng.uniform(-1, 1, (n_before, nvars, (p + 1) ** dim))
    un_o = ot.transfer(uo, p, nvars)
    un_g = gt.transfer(torch.from_numpy(uo).cuda(), p, nvars)
    gt.sync()
    P.assert_u_close(un_g, un_o, "deep transfer")


def test_empty_input_is_rejected():
    dom = [0.0, 0.0, 1.0, 1.0]
    with pytest.raises(lt.LtError):
        lt.build_from_points(2, 1, 5, torch.empty((0, 2), dtype=torch.float64, device="cuda"), dom)
    with pytest.raises(lt.LtError):
        lt.build_complete_from_keys(2, 1, 5, torch.empty(0, dtype=torch.int64, device="cuda"))
