"""GPU parity for SURVEY 8(f)-2: mortar operators on nonconforming faces (Alg. 8 steps 2 and 4,
Eq. 14-20) against the oracle's quadrature + dense-solve operators.
Tolerance: max|gpu - ref| <= 1e-12 * max(1, max|ref|) (the fp64 bound of DESIGN.md E-8: sums of
at most 2^(dim-1) (p+1)^(dim-1) products with O(1) operator entries)."""
import numpy as np
import pytest
import torch

import oracle
import parity as P
from paper_2306_06744_b200 import lt
from paper_2306_06744_b200 import workloads as W

pytestmark = pytest.mark.gpu


def adapted_pair(dim, periodic, seed, base, maxl, cycles=3):
    rng = np.random.default_rng(seed)
    gt = lt.Tree(dim, base, maxl, [0.0] * dim + [1.0] * dim, periodic)
    ot = oracle.Tree(dim, base, maxl, periodic)
    for _ in range(cycles):
        f = (rng.random(ot.num_leaves()) < 0.3).astype(np.int8)
        ot.adapt(f); ot.balance(); ot.drop_snapshot()
        gt.adapt(torch.from_numpy(f).cuda()); gt.balance()
    P.assert_keys_equal(gt, ot, "tree")
    return gt, ot, rng


def close(a, b, what):
    a = a.cpu().numpy()
    assert a.shape == b.shape
    assert np.array_equal(np.isnan(a), np.isnan(b)), what + ": touched / untouched slots differ"
    m = ~np.isnan(b)
    scale = max(1.0, float(np.max(np.abs(b[m])))) if m.any() else 1.0
    err = float(np.max(np.abs(a[m] - b[m]))) if m.any() else 0.0
    assert err <= 1e-12 * scale, "%s: error %.3e" % (what, err)


@pytest.mark.parametrize("dim,periodic,base,maxl", [(2, (0, 0), 2, 6), (2, (1, 1), 3, 6), (3, (0, 0, 0), 2, 5),
                                                    (3, (1, 1, 1), 2, 4), (3, (0, 1, 0), 1, 4)])
@pytest.mark.parametrize("p,nvars", [(0, 1), (1, 3), (2, 5), (3, 5), (4, 2), (7, 1)])
def test_mortar_project_and_gather(dim, periodic, base, maxl, p, nvars):
    if dim == 3 and p == 7:
        maxl = min(maxl, 4)
    gt, ot, rng = adapted_pair(dim, periodic, 31 * dim + p, base, maxl)
    Fo = ot.connect()
    P.assert_faces_equal(gt.connect(), Fo, "faces")
    kinds = Fo["kind"] & 15
    assert (kinds == 2).any() and (kinds == 3).any()
    Nf = (p + 1) ** (dim - 1)
    uf = rng.uniform(-1, 1, (ot.num_leaves(), 2 * dim, nvars, Nf))
    close(gt.mortar_project(torch.from_numpy(uf).cuda(), p, nvars), ot.mortar_project(uf, p, nvars), "project")
    close(gt.mortar_gather(torch.from_numpy(uf).cuda(), p, nvars), ot.mortar_gather(uf, p, nvars), "gather")
    gt.sync()  # raises on a sticky device status (a missing fine neighbour)


def test_gather_in_place_and_untouched_slots():
    gt, ot, rng = adapted_pair(3, (1, 1, 1), 5, 2, 4)
    gt.connect(); Fo = ot.connect()
    p, nvars = 2, 4
    fm = rng.uniform(-1, 1, (ot.num_leaves(), 6, nvars, 9))
    want = ot.mortar_gather(fm, p, nvars)
    d = torch.from_numpy(fm).cuda()
    out = gt.mortar_gather(d, p, nvars, f_face=d)  # in place: kind 3 slots overwritten, the rest kept
    assert out.data_ptr() == d.data_ptr()
    m3 = ~np.isnan(want)
    got = out.cpu().numpy()
    assert np.array_equal(got[~m3], fm[~m3])
    assert np.max(np.abs(got[m3] - want[m3])) <= 1e-12
    with pytest.raises(lt.LtError):
        gt.mortar_project(d, p, nvars, u_nb=d)  # project must not alias


def test_needs_connect_on_current_tree():
    gt = lt.Tree(2, 2, 4)
    u = torch.zeros((16, 4, 1, 2), dtype=torch.float64, device="cuda")
    with pytest.raises(lt.LtError):
        gt.mortar_project(u, 1, 1)
    gt.connect()
    gt.mortar_project(u, 1, 1)
    gt.adapt(torch.ones(16, dtype=torch.int8, device="cuda"))
    u = torch.zeros((64, 4, 1, 2), dtype=torch.float64, device="cuda")
    with pytest.raises(lt.LtError):
        gt.mortar_gather(u, 1, 1)  # faces describe the tree before lt_adapt


def test_polynomial_trace_on_cycle_mesh():
    # config-4-shaped mesh (vortex tube flags), p = 2: the neighbour trace of a global polynomial
    # equals the element's own trace on every conforming and hanging face, and the gathered flux
    # equals the coarse face's own samples -- checked on the GPU output alone
    cfg = dict(W.CONFIGS["c4"], base=3, maxl=5, periodic=(0, 0, 0))
    gt, ot = P.new_pair(cfg)
    for c in range(2):
        f = P.host_flags(cfg, c, ot)
        ot.adapt(f); ot.balance(); ot.drop_snapshot()
        gt.adapt(torch.from_numpy(f).cuda()); gt.balance()
    F = gt.connect()
    kind = (F["kind"].cpu().numpy() & 15).reshape(-1, 6)
    lvl, xyz = gt.leaf_boxes()
    lvl, xyz = lvl.cpu().numpy().astype(np.int64), xyz.cpu().numpy().astype(np.float64)
    p, P1 = 2, 3
    z, _ = np.polynomial.legendre.leggauss(P1)
    L = float(1 << cfg["maxl"])
    w = (1 << (cfg["maxl"] - lvl)).astype(np.float64)
    M = len(lvl)
    uf = np.zeros((M, 6, 1, 9))
    for f in range(6):
        ax = f >> 1
        t0, t1 = [a for a in range(3) if a != ax]
        X = np.zeros((M, 9, 3))
        for n in range(9):
            X[:, n, t0] = (xyz[:, t0] + 0.5 * w * (1 + z[n % P1])) / L
            X[:, n, t1] = (xyz[:, t1] + 0.5 * w * (1 + z[n // P1])) / L
            X[:, n, ax] = (xyz[:, ax] + (w if f & 1 else 0.0)) / L
        uf[:, f, 0, :] = (1 + X[..., 0] + 2 * X[..., 0] ** 2) * (2 - X[..., 1] ** 2) * (0.5 + X[..., 2] - X[..., 2] ** 2)
    d = torch.from_numpy(uf).cuda()
    unb = gt.mortar_project(d, p, 1).cpu().numpy()
    m12 = (kind == 1) | (kind == 2)
    assert np.max(np.abs(unb[m12] - uf[m12])) < 1e-12
    ff = gt.mortar_gather(d, p, 1).cpu().numpy()
    assert (kind == 3).any() and np.max(np.abs(ff[kind == 3] - uf[kind == 3])) < 1e-12


@pytest.mark.parametrize("dim,periodic,base,maxl", [(2, (1, 0), 2, 6), (3, (0, 0, 0), 2, 4)])
@pytest.mark.parametrize("p,nvars", [(0, 2), (1, 1), (2, 4), (3, 5), (5, 3), (7, 2)])
def test_face_interp_then_mortars(dim, periodic, base, maxl, p, nvars):
    # Alg. 8 steps 1, 2, 4 chained: solution -> face points -> neighbour traces / gathered fluxes
    gt, ot, rng = adapted_pair(dim, periodic, 17 * dim + p, base, maxl, cycles=2)
    gt.connect(); ot.connect()
    N = (p + 1) ** dim
    u = rng.uniform(-1, 1, (ot.num_leaves(), nvars, N))
    uf_o = ot.face_interp(u, p, nvars)
    uf_g = gt.face_interp(torch.from_numpy(u).cuda(), p, nvars)
    close(uf_g, uf_o, "face_interp")
    close(gt.mortar_project(uf_g, p, nvars), ot.mortar_project(uf_o, p, nvars), "project after interp")
    close(gt.mortar_gather(uf_g, p, nvars), ot.mortar_gather(uf_o, p, nvars), "gather after interp")
    gt.sync()
    with pytest.raises((lt.LtError, ValueError)):
        gt.face_interp(uf_g, p, nvars)  # wrong shape


def test_gather_survives_transfer_host_between_two_meshes():
    """Regression (round-1 advisor finding): lt_transfer_host used to free the hit list that
    lt_mortar_gather keeps on the tree, leaving a dangling pointer for the next gather.  Sequence:
    connect + gather, adapt / balance / transfer_host (its first call on this tree allocates the slab
    bounds), connect + gather on the new tree -- every step against the oracle; then once more with a
    refine-everything cycle so that the hit list has to grow."""
    dim, p, nvars = 3, 2, 3
    gt, ot, rng = adapted_pair(dim, (1, 1, 1), 77, 2, 5, cycles=2)
    N, Nf = (p + 1) ** dim, (p + 1) ** (dim - 1)
    for step in range(3):
        Fo = ot.connect()
        P.assert_faces_equal(gt.connect(), Fo, "faces, step %d" % step)
        assert ((Fo["kind"] & 15) == 3).any()
        fm = rng.uniform(-1, 1, (ot.num_leaves(), 2 * dim, nvars, Nf))
        close(gt.mortar_gather(torch.from_numpy(fm).cuda(), p, nvars), ot.mortar_gather(fm, p, nvars),
              "gather, step %d" % step)
        gt.sync()
        if step == 2:
            break
        uo = rng.uniform(-1, 1, (ot.num_leaves(), nvars, N))
        f = (rng.random(ot.num_leaves()) < (0.3 if step == 0 else 1.0)).astype(np.int8)
        ot.adapt(f); ot.balance()
        gt.adapt(torch.from_numpy(f).cuda()); gt.balance()
        P.assert_keys_equal(gt, ot, "tree, step %d" % step)
        want = ot.transfer(uo, p, nvars)
        h_new = torch.empty((gt.num_leaves(), nvars, N), dtype=torch.float64).pin_memory()
        gt.transfer_host(torch.from_numpy(uo).pin_memory(), h_new, p, nvars)
        P.assert_u_close(h_new, want, "host transfer, step %d" % step)
