"""Parity at BASELINE.json's full size, in the launch configuration bench.py times: config 5
(3-D octree, periodic, base 64^3, max level +3, p = 3, 5 fp64 variables) driven through cycles
0..5 on both sides -- cycles 3, 4 and 5 (8,863,051 -> 13,473,692 -> 18,901,814 -> 26,066,874
leaves) are exactly the steps bench.py times.

For every timed step the trees, balance sweep counts, the face tables and the Alg. 7 map are
compared IN FULL, bit for bit, against the CPU oracle (which builds its own pointer tree of up to
26 M leaves: minutes of host time); the transferred solution is compared on sampled slabs of new
elements that the oracle computes one by one (dense M^-1 S_c, Eq. 12), within the 1e-12 bound of
DESIGN.md reading E-8.  No oracle input comes from the CUDA path: flags and the old solution come
from the shared seeded generators (workloads.py), evaluated on the oracle's own leaf boxes / on
boxes that were compared with the oracle's.
"""
import numpy as np
import pytest
import torch

import oracle
import parity as P
from paper_2306_06744_b200 import lt
from paper_2306_06744_b200 import workloads as W

pytestmark = pytest.mark.gpu

TIMED = (3, 4, 5)    # the cycles bench.py times
SLAB = 96            # new elements per sampled slab
N_SLABS = 40
CENSUS = {3: (8863051, 13473692), 4: (13473692, 18901814), 5: (18901814, 26066874)}


def _analytic_u(cfg, gt, out):
    lvl, xyz = gt.leaf_boxes()
    M = lvl.shape[0]
    step = 1 << 20
    for a in range(0, M, step):
        b = min(a + step, M)
        out[a:b] = W.initial_solution(cfg, lvl[a:b], xyz[a:b])


def _check_transfer_slabs(ot, ug, un_g, src_o, kind_o, p, nvars, seed):
    """Sampled slabs of new elements against the oracle; only the old rows a slab needs are copied
    to the host (transfer_rows takes a window of u_old)."""
    M0, M1 = ug.shape[0], un_g.shape[0]
    rng = np.random.default_rng(seed)
    starts = [0, M1 - SLAB] + [int(v) for v in rng.integers(0, M1 - SLAB, N_SLABS - 2)]
    # make sure every kind is sampled: add slabs that start at a refined / a coarsened element
    for k in (1, 2):
        idx = np.flatnonzero((kind_o & 15) == k)
        assert idx.size > 0
        starts += [int(min(idx[idx.size // 3], M1 - SLAB)), int(min(idx[2 * idx.size // 3], M1 - SLAB))]
    seen = np.zeros(3, np.int64)
    worst = 0.0
    for j0 in starts:
        j1 = j0 + SLAB
        lo = int(src_o[j0:j1].min())
        hi = min(M0, int(src_o[j0:j1].max()) + 8)
        ref = ot.transfer_rows(ug[lo:hi].cpu().numpy(), p, nvars, j0, j1, old_offset=lo)
        got = un_g[j0:j1].cpu().numpy()
        for v in range(nvars):
            tol = 1e-12 * max(1.0, np.abs(ref[:, v]).max())
            err = np.abs(got[:, v] - ref[:, v]).max()
            worst = max(worst, err)
            assert err <= tol, "slab %d var %d: |diff| %.3e > %.3e" % (j0, v, err, tol)
        for k in range(3):
            seen[k] += int(((kind_o[j0:j1] & 15) == k).sum())
    assert (seen > 0).all(), "sampled slabs must cover copy, refine and coarsen: %s" % seen
    return seen, worst


def _check_mortars(gt, ot, p, M1):
    # Alg. 8 steps 2 and 4 on every face slot of the mesh, p = 3 with one variable so that the host
    # arrays stay at 10 GB each
    nf, Nf = 6, (p + 1) ** 2
    uf = np.random.default_rng(11).uniform(-1.0, 1.0, (M1, nf, 1, Nf))
    d_uf = torch.from_numpy(uf).cuda()
    for name in ("mortar_project", "mortar_gather"):
        want = getattr(ot, name)(uf, p, 1)
        got = getattr(gt, name)(d_uf, p, 1).cpu().numpy()
        gt.sync()
        m = ~np.isnan(want)
        assert np.array_equal(np.isnan(got), ~m), name + ": touched slots differ"
        err = float(np.abs(got[m] - want[m]).max())
        assert err <= 1e-12, "%s at full size: |diff| %.3e" % (name, err)
        print("c5 full size %s: %d values, worst |diff| %.2e" % (name, int(m.sum()), err))
        del want, got, m


def test_config5_full_size_timed_cycles():
    cfg = W.CONFIGS["c5"]
    p, nvars = cfg["p"], cfg["nvars"]
    N = (p + 1) ** cfg["dim"]
    free, _ = torch.cuda.mem_get_info()
    if free < 135 * 2 ** 30:
        pytest.skip("needs ~125 GB of device memory (u_old + u_new of cycle 5 are 115 GB)")
    gt, ot = P.new_pair(cfg)
    for c in range(TIMED[-1] + 1):
        tag = "c5 full size, cycle %d" % c
        f = P.host_flags(cfg, c, ot)
        timed = c in TIMED
        ug = None
        if timed:
            # the old solution: analytic vortex on the old tree (the GPU's boxes were compared with the
            # oracle's through the keys of the previous cycle)
            M0 = gt.num_leaves()
            ug = torch.empty((M0, nvars, N), dtype=torch.float64, device="cuda")
            _analytic_u(cfg, gt, ug)
        ot.adapt(f)
        gt.adapt(torch.from_numpy(f).cuda())
        del f
        it_o = ot.balance()
        it_g = gt.balance()
        assert it_g == it_o, "%s: balance iters %d vs oracle %d" % (tag, it_g, it_o)
        P.assert_keys_equal(gt, ot, tag)
        if not timed:
            ot.drop_snapshot()
            continue
        M1 = ot.num_leaves()
        assert (M0, M1) == CENSUS[c], tag
        # ---- connectivity, in full, in the form bench.py times it: the face query on the side stream
        # beside the solution transfer (lt_connect_begin / lt_transfer / lt_connect_end)
        gt.connect_begin()
        un_g = gt.transfer(ug, p, nvars)
        Fg = gt.connect_end()
        Fo = ot.connect()
        P.assert_faces_equal(Fg, Fo, tag + " connect")
        assert 6 * M1 == 2 * Fo["n_conf"] + Fo["n_hang"] + Fo["n_hang"] // 4 + Fo["n_bnd"]
        del Fg, Fo
        # ---- map, in full; transfer on sampled slabs
        src_o, kind_o = ot.build_map()
        gt.sync()
        src_g, kind_g = gt.map()
        assert np.array_equal(src_g.cpu().numpy(), src_o), tag + " map src"
        assert np.array_equal(kind_g.cpu().numpy(), kind_o), tag + " map kind"
        seen, worst = _check_transfer_slabs(ot, ug, un_g, src_o, kind_o, p, nvars, seed=5 + c)
        print("%s: %d -> %d leaves, %d sweeps; sampled %d elements (copy/refine/coarsen %s), worst |diff| %.2e"
              % (tag, M0, M1, it_o, seen.sum(), seen, worst))
        ot.drop_snapshot()
        del src_o, kind_o, src_g, kind_g
        if c == TIMED[0]:
            _check_mortars(gt, ot, p, M1)
        del un_g, ug
        torch.cuda.empty_cache()


def test_construction_full_size_pc9():
    """SURVEY 8(f)-1 at the size bench.py's cpu_baseline uses: 4 M points, D_min 4, D_max 9 ->
    1.19 M leaves after completion, 1.40 M after the full-depth balance; keys, sweep count and
    face tables bit-exact against the oracle."""
    pc = W.POINT_CLOUDS["pc9"]
    dom = [pc["lo"]] * 3 + [pc["hi"]] * 3
    pts = W.surface_points(pc).numpy()
    ot = oracle.Tree(3, pc["base"], pc["maxl"], pc["periodic"], points=pts, domain=dom)
    gt = lt.build_from_points(3, pc["base"], pc["maxl"], torch.from_numpy(pts).cuda(), dom, pc["periodic"])
    P.assert_keys_equal(gt, ot, "pc9 completion")
    assert gt.num_leaves() == 1190953
    it_o, it_g = ot.balance(), gt.balance()
    assert it_o == it_g == 4
    P.assert_keys_equal(gt, ot, "pc9 balance")
    assert gt.num_leaves() == 1402682
    P.assert_faces_equal(gt.connect(), ot.connect(), "pc9 connect")
