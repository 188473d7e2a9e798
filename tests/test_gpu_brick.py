"""GPU parity on bricks of root cubes (lt_build_brick; reading J-1; the paper's 3-D slab,
PAPER.md:410): the whole cycle, strong balance, the paper's append-sort-linearise adapt, the mortar /
FR chain and the slab workload itself, against the oracle's forest (pinned by
tests/test_oracle_brick.py).  Bit-exact for everything integer, 1e-12 for the solution (E-8), the
I-6 bound for the right-hand side."""
import numpy as np
import pytest
import torch

import oracle
import parity as P
from paper_2306_06744_b200 import lt
from paper_2306_06744_b200 import workloads as W
from test_gpu_fr import close_rhs, gpu_pipeline
from test_gpu_mortar import close
from test_oracle_brick import BRICKS

pytestmark = pytest.mark.gpu


def pair(dim, nroot, per, base, maxl, cube=1.0):
    dom = [0.0] * dim + [cube * n for n in nroot]
    return (lt.Tree(dim, base, maxl, dom, per, nroot=nroot), oracle.Tree(dim, base, maxl, per, nroot=nroot))


@pytest.mark.parametrize("dim,nroot,per", BRICKS)
@pytest.mark.parametrize("base", [0, 2])
def test_uniform_bricks(dim, nroot, per, base):
    gt, ot = pair(dim, nroot, per, base, 3)
    assert gt.roots() == tuple(nroot)
    P.assert_keys_equal(gt, ot, "uniform brick")
    glvl, gxyz = gt.leaf_boxes()
    olvl, oxyz = ot.leaf_boxes()
    assert np.array_equal(glvl.cpu().numpy(), olvl) and np.array_equal(gxyz.cpu().numpy().astype(np.uint32), oxyz)
    P.assert_faces_equal(gt.connect(), ot.connect(), "uniform brick faces")
    assert gt.balance() == 0


@pytest.mark.parametrize("dim,nroot,per", BRICKS)
@pytest.mark.parametrize("p,nvars", [(1, 2), (3, 3)])
def test_random_cycles_on_bricks(dim, nroot, per, p, nvars):
    base, maxl = (1, 5) if dim == 2 else (0, 4)
    gt, ot = pair(dim, nroot, per, base, maxl)
    rng = np.random.default_rng(100 * dim + 7 * p + sum(nroot))
    N = (p + 1) ** dim
    uo = rng.uniform(-1, 1, (ot.num_leaves(), nvars, N))
    kinds = set()
    for c in range(6):
        f = rng.choice(np.array([-1, 0, 1], np.int8), ot.num_leaves(), p=[0.5, 0.2, 0.3] if c % 2 else [0.1, 0.5, 0.4])
        if c == 5:
            f[:] = -1                                   # coarsen every complete group above the base level
        ot.adapt(f)
        gt.adapt(torch.from_numpy(f).cuda())
        P.assert_keys_equal(gt, ot, "adapt %d" % c)
        assert gt.balance() == ot.balance()
        P.assert_keys_equal(gt, ot, "balance %d" % c)
        P.assert_faces_equal(gt.connect(), ot.connect(), "connect %d" % c)
        src_o, kind_o = ot.build_map()
        kinds |= set((kind_o & 15).tolist())
        un_o = ot.transfer_rows(uo, p, nvars, 0, ot.num_leaves())
        ot.drop_snapshot()
        un_g = gt.transfer(torch.from_numpy(uo).cuda(), p, nvars)
        gt.sync()
        src_g, kind_g = gt.map()
        assert np.array_equal(src_g.cpu().numpy(), src_o) and np.array_equal(kind_g.cpu().numpy(), kind_o)
        P.assert_u_close(un_g, un_o, "transfer %d" % c)
        uo = un_o
    assert kinds == {0, 1, 2}


@pytest.mark.parametrize("dim,nroot,per,conn", [(2, (3, 2), (1, 0), 2), (3, (2, 2, 1), (1, 1, 1), 2),
                                                (3, (1, 2, 2), (0, 0, 0), 3)])
def test_strong_balance_on_bricks(dim, nroot, per, conn):
    gt, ot = pair(dim, nroot, per, 1, 5 if dim == 2 else 4)
    gt.set_option(lt.LT_OPT_BALANCE_CONNECTIVITY, conn)
    rng = np.random.default_rng(conn + dim)
    for c in range(4):
        f = (rng.random(ot.num_leaves()) < 0.15).astype(np.int8)
        ot.adapt(f); gt.adapt(torch.from_numpy(f).cuda())
        assert gt.balance() == ot.balance(conn)
        P.assert_keys_equal(gt, ot, "strong balance %d" % c)
        ot.drop_snapshot()
    P.assert_faces_equal(gt.connect(), ot.connect(), "faces after strong balance")


def test_adapt_by_append_sort_linearise_on_a_brick():
    """Alg. 6 as printed (path A): the radix sort has to cover the cube index bits as well."""
    dim, nroot, per = 3, (3, 2, 2), (1, 0, 1)
    gt, ot = pair(dim, nroot, per, 1, 4)
    gt.set_option(lt.LT_OPT_ADAPT_SORT, 1)
    rng = np.random.default_rng(9)
    for c in range(4):
        f = rng.integers(-1, 2, ot.num_leaves()).astype(np.int8)
        ot.adapt(f); gt.adapt(torch.from_numpy(f).cuda())
        P.assert_keys_equal(gt, ot, "path A adapt %d" % c)
        assert gt.balance() == ot.balance()
        P.assert_keys_equal(gt, ot, "path A balance %d" % c)
        ot.drop_snapshot()


def test_slab_workload_all_cycles():
    """The paper's slab [-12.5, 12.5]^2 x 1.5625 as 16 x 16 x 1 cubes (Table 5), config 4's
    vortex-tube flags, 20 cycles: every output of every cycle."""
    cfg = W.CONFIGS["slab"]
    log, rec = [], []
    P.run_cycles(cfg, cfg["cycles"], log=log, record=rec)
    assert log[0][1] == 340 and all(r[5] == 0 for r in log)          # periodic: no boundary faces
    assert max(r[1] for r in log) > 40000 and max(r[2] for r in log) >= 3
    P.replay_gpu(cfg, rec, options=[(lt.LT_OPT_BALANCE_FULL_SWEEPS, 1)])


@pytest.mark.parametrize("dim,nroot,per", [(2, (3, 2), (1, 1)), (3, (2, 1, 2), (1, 1, 1))])
@pytest.mark.parametrize("p", [1, 3])
def test_fr_chain_on_a_brick(dim, nroot, per, p):
    """Alg. 8 steps 1-4 + Eq. 2-5 on an adapted periodic brick with cube edge 0.5: the element width
    is width_a / (nroot_a 2^level)."""
    h = 0.5
    gt, ot = pair(dim, nroot, per, 1, 4 if dim == 2 else 3, cube=h)
    rng = np.random.default_rng(5 * dim + p)
    for _ in range(2):
        f = (rng.random(ot.num_leaves()) < 0.3).astype(np.int8)
        ot.adapt(f); ot.balance(); ot.drop_snapshot()
        gt.adapt(torch.from_numpy(f).cuda()); gt.balance()
    F = gt.connect(); ot.connect()
    assert int(F["n_hang"]) > 0
    M, N, nv = ot.num_leaves(), (p + 1) ** dim, dim + 2
    lvl, xyz = ot.leaf_boxes()
    z, _ = np.polynomial.legendre.leggauss(p + 1)
    Lw = float(1 << ot.maxl)
    wd = (1 << (ot.maxl - lvl.astype(np.int64))) / Lw
    X = np.zeros((M, N, dim))
    for n in range(N):
        r = n
        for a in range(dim):
            X[:, n, a] = (xyz[:, a] / Lw + 0.5 * wd * (1 + z[r % (p + 1)])) / nroot[a]   # in [0, 1) over the brick
            r //= p + 1
    ph = 2 * np.pi * X
    rho = 1.0 + 0.2 * np.prod(np.sin(ph), axis=-1)
    vel = np.stack([0.4 + 0.1 * np.cos(ph[..., (a + 1) % dim]) for a in range(dim)], axis=-1)
    pr = 1.0 + 0.1 * np.cos(ph[..., 0])
    u = np.concatenate([rho[:, None], np.moveaxis(rho[..., None] * vel, -1, 1),
                        (pr / 0.4 + 0.5 * rho * np.sum(vel * vel, -1))[:, None]], axis=1).copy()
    uf = ot.face_interp(u, p, nv)
    fs_o = ot.common_flux(uf, ot.mortar_project(uf, p, nv), p)
    fs_o = np.where(np.isnan(fs_o), ot.mortar_gather(fs_o, p, nv), fs_o)
    R_o = ot.fr_rhs(u, fs_o, p, [h * n for n in nroot])
    fs_g, R_g = gpu_pipeline(gt, torch.from_numpy(u).cuda(), p)
    close(fs_g, fs_o, "brick: common fluxes")
    lvl_max = int(lvl.max())
    scale = max(1.0, float(np.abs(R_o).max()), float(2 << lvl_max) / h * float(np.abs(fs_o).max()))
    err = float(np.abs(R_g.cpu().numpy() - R_o).max())
    assert err <= 1e-12 * scale, "brick rhs: %.3e > 1e-12 * %.3g" % (err, scale)
    gt.sync()


def test_bad_bricks():
    for nroot, maxl in (((0, 2), 3), ((2, 2, 1), 19), ((1 << 20, 1 << 20), 2)):
        with pytest.raises(lt.LtError) as ei:
            lt.Tree(len(nroot), 0, maxl, None, None, nroot=nroot)
        assert ei.value.status == lt.LT_ERR_ARG
