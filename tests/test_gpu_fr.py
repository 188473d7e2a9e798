"""GPU parity for the FR pieces around the cycle (Eq. 1-6; Alg. 8 step 3): Rusanov
common flux, the right-hand side with Radau corrections, the SSP-RK3 stages, and the whole chain
face_interp -> mortar_project -> common_flux -> mortar_gather -> fr_rhs, against the oracle.
Tolerance: fluxes max|gpu - ref| <= 1e-12 * max(1, max|ref|); the right-hand side is a sum of terms of size
(2/dx) |operator| |flux| that largely cancel, so its bound is 1e-12 * max(1, max|ref|, (2/dx_min) max|F*|)
(reading I-6)."""
import numpy as np
import pytest
import torch

import oracle
import parity as P
from paper_2306_06744_b200 import lt
from test_gpu_mortar import adapted_pair, close
from test_oracle_fr import random_states

pytestmark = pytest.mark.gpu


def gpu_pipeline(gt, d_u, p):
    nv = gt.dim + 2
    uf = gt.face_interp(d_u, p, nv)
    unb = gt.mortar_project(uf, p, nv)
    fs = gt.common_flux(uf, unb, p)
    gt.mortar_gather(fs, p, nv, f_face=fs)   # in place: the coarse-side hanging slots
    return fs, gt.fr_rhs(d_u, fs, p)


def close_rhs(got, want, fs, ot, what):
    lvl, _ = ot.leaf_boxes()
    scale = max(1.0, float(np.max(np.abs(want))), float(2 << int(lvl.max())) * float(np.nanmax(np.abs(fs))))
    err = float(np.max(np.abs(got.cpu().numpy() - want)))
    assert err <= 1e-12 * scale, "%s: error %.3e > 1e-12 * %.3g" % (what, err, scale)


def oracle_pipeline(ot, u, p):
    nv = ot.dim + 2
    uf = ot.face_interp(u, p, nv)
    unb = ot.mortar_project(uf, p, nv)
    fs = ot.common_flux(uf, unb, p)
    g = ot.mortar_gather(fs, p, nv)
    fs = np.where(np.isnan(fs), g, fs)
    return fs, ot.fr_rhs(u, fs, p, [1.0] * ot.dim)


@pytest.mark.parametrize("dim,base,maxl", [(2, 2, 6), (3, 2, 4)])
@pytest.mark.parametrize("p", [0, 1, 2, 3, 5, 7])
def test_flux_rhs_and_chain_match_oracle(dim, base, maxl, p):
    if dim == 3 and p == 7:
        maxl = 3
    gt, ot, rng = adapted_pair(dim, (1,) * dim, 51 * dim + p, base, maxl, cycles=2)
    gt.connect(); ot.connect()
    M, N, Nf, nv = ot.num_leaves(), (p + 1) ** dim, (p + 1) ** (dim - 1), dim + 2
    # (1) common flux on random admissible traces
    a = np.moveaxis(random_states(rng, (M, 2 * dim, Nf), dim), -1, 2).copy()
    b = np.moveaxis(random_states(rng, (M, 2 * dim, Nf), dim), -1, 2).copy()
    close(gt.common_flux(torch.from_numpy(a).cuda(), torch.from_numpy(b).cuda(), p), ot.common_flux(a, b, p), "common_flux")
    # (2) right-hand side on random states and random common fluxes
    u = np.moveaxis(random_states(rng, (M, N), dim), -1, 1).copy()
    fs = rng.uniform(-1, 1, (M, 2 * dim, nv, Nf))
    close_rhs(gt.fr_rhs(torch.from_numpy(u).cuda(), torch.from_numpy(fs).cuda(), p), ot.fr_rhs(u, fs, p, [1.0] * dim),
              fs, ot, "fr_rhs")
    # (3) the whole chain, on a smooth admissible state (a random one stops being admissible once it
    # is extrapolated to the faces: negative densities, NaN wave speeds)
    lvl, xyz = ot.leaf_boxes()
    z, _ = np.polynomial.legendre.leggauss(p + 1)
    Lw = float(1 << ot.maxl)
    wd = (1 << (ot.maxl - lvl.astype(np.int64))) / Lw
    X = np.zeros((M, N, dim))
    for n in range(N):
        r = n
        for a2 in range(dim):
            X[:, n, a2] = xyz[:, a2] / Lw + 0.5 * wd * (1 + z[r % (p + 1)])
            r //= p + 1
    ph = 2 * np.pi * X
    rho = 1.0 + 0.2 * np.prod(np.sin(ph), axis=-1)
    vel = np.stack([0.4 + 0.1 * np.cos(ph[..., (a2 + 1) % dim]) for a2 in range(dim)], axis=-1)
    pr = 1.0 + 0.1 * np.cos(ph[..., 0])
    u = np.concatenate([rho[:, None], np.moveaxis(rho[..., None] * vel, -1, 1),
                        (pr / 0.4 + 0.5 * rho * np.sum(vel * vel, -1))[:, None]], axis=1).copy()
    fs_g, R_g = gpu_pipeline(gt, torch.from_numpy(u).cuda(), p)
    fs_o, R_o = oracle_pipeline(ot, u, p)
    close(fs_g, fs_o, "chain: common fluxes")
    close_rhs(R_g, R_o, fs_o, ot, "chain: rhs")
    gt.sync()


@pytest.mark.parametrize("dim", [2, 3])
def test_free_stream_and_rk3_on_gpu(dim):
    p = 3 if dim == 2 else 2
    gt, ot, rng = adapted_pair(dim, (1,) * dim, 7, 2, 5 if dim == 2 else 4, cycles=2)
    gt.connect()
    M, N = ot.num_leaves(), (p + 1) ** dim
    state = random_states(np.random.default_rng(2), (), dim)
    u = torch.from_numpy(np.tile(state[None, :, None], (M, 1, N))).cuda()
    _, R = gpu_pipeline(gt, u, p)
    assert float(R.abs().max()) < 1e-9
    # Eq. 6 against the oracle's rk3_stage, arbitrary arrays.  The oracle writes stage 1 as
    # u^n + dt R (its stage vector IS u^n), so stage 1 is called with u_stage = u_n on both sides.
    un_h, us_h, r_h = (rng.uniform(-1, 1, (M, dim + 2, N)) for _ in range(3))
    un, us, r = (torch.from_numpy(a).cuda() for a in (un_h, us_h, r_h))
    dt = 0.37
    for stage in (1, 2, 3):
        st_h, st = (un_h, un) if stage == 1 else (us_h, us)
        want = oracle.rk3_stage(stage, dt, un_h, st_h, r_h)
        got = gt.rk3_stage(stage, dt, un, st, r, p)
        assert float(np.abs(got.cpu().numpy() - want).max()) < 1e-15
    inplace = us.clone()
    gt.rk3_stage(2, dt, un, inplace, r, p, out=inplace)
    assert float(np.abs(inplace.cpu().numpy() - oracle.rk3_stage(2, dt, un_h, us_h, r_h)).max()) < 1e-15


@pytest.mark.parametrize("dim,p", [(2, 3), (3, 2), (3, 3)])
def test_fr_stage_all_stages_match_oracle_chain(dim, p):
    """lt_fr_stage (right-hand side + Eq. 6 in one pass) and the unfused lt_fr_rhs + lt_rk3_stage against
    the ORACLE's chain (Alg. 8 steps 1-4, Eq. 2-5, then oracle.rk3_stage) for all three stages of one
    SSP-RK3 step on an adapted periodic mesh with hanging faces; every stage is fed the oracle's stage
    vector, so no GPU result enters an expected value.  Also in place over u_stage / u_n."""
    gt, ot, rng = adapted_pair(dim, (1,) * dim, 17 + dim, 2, 5 if dim == 2 else 4, cycles=2)
    F = gt.connect(); ot.connect()
    assert int(F["n_hang"]) > 0
    M, N = ot.num_leaves(), (p + 1) ** dim
    lvl, xyz = ot.leaf_boxes()
    z, _ = np.polynomial.legendre.leggauss(p + 1)
    Lw = float(1 << ot.maxl)
    wd = (1 << (ot.maxl - lvl.astype(np.int64))) / Lw
    X = np.zeros((M, N, dim))
    for n in range(N):
        r_ = n
        for a2 in range(dim):
            X[:, n, a2] = xyz[:, a2] / Lw + 0.5 * wd * (1 + z[r_ % (p + 1)])
            r_ //= p + 1
    ph = 2 * np.pi * X
    rho = 1.0 + 0.2 * np.prod(np.sin(ph), axis=-1)
    vel = np.stack([0.4 + 0.1 * np.cos(ph[..., (a2 + 1) % dim]) for a2 in range(dim)], axis=-1)
    pr = 1.0 + 0.1 * np.cos(ph[..., 0])
    u_n = np.concatenate([rho[:, None], np.moveaxis(rho[..., None] * vel, -1, 1),
                          (pr / 0.4 + 0.5 * rho * np.sum(vel * vel, -1))[:, None]], axis=1).copy()
    dt = 2e-3
    d_un = torch.from_numpy(u_n).cuda()
    u_stage = u_n
    for stage in (1, 2, 3):
        fs_o, R_o = oracle_pipeline(ot, u_stage, p)
        want = oracle.rk3_stage(stage, dt, u_n, u_stage, R_o)
        d_us = torch.from_numpy(u_stage).cuda()
        fs_g, R_g = gpu_pipeline(gt, d_us, p)
        close(fs_g, fs_o, "stage %d: common fluxes" % stage)
        close_rhs(R_g, R_o, fs_o, ot, "stage %d: rhs" % stage)
        # dt * (the I-6 bound of R) + E-8's bound on the state
        lvl_max = int(lvl.max())
        tol = 1e-12 * max(1.0, float(np.abs(want).max()), dt * float(2 << lvl_max) * float(np.abs(fs_o).max()))
        unfused = gt.rk3_stage(stage, dt, d_un, d_us, R_g, p)
        fused = gt.fr_stage(stage, dt, d_un, d_us, fs_g, p)
        for name, got in (("rk3_stage(fr_rhs)", unfused), ("fr_stage", fused)):
            err = float(np.abs(got.cpu().numpy() - want).max())
            assert err <= tol, "stage %d %s: |diff| %.3e > %.3e" % (stage, name, err, tol)
        w1 = d_us.clone()
        gt.fr_stage(stage, dt, d_un, w1, fs_g, p, out=w1)          # in place over the stage vector
        assert torch.equal(w1, fused)
        if stage > 1:
            w2 = d_un.clone()
            gt.fr_stage(stage, dt, w2, d_us, fs_g, p, out=w2)      # in place over u^n
            assert torch.equal(w2, fused)
        u_stage = want                                             # the oracle's stage vector feeds the next stage
    gt.sync()
    assert float(np.abs(u_stage - u_n).max()) > 1e-6               # the step did something


def test_full_step_conserves_mass_momentum_energy():
    # one SSP-RK3 step of the isentropic-vortex-like state on an adapted periodic mesh with hanging
    # faces: the mortar projections are conservative, so the domain integrals of all
    # conserved variables are unchanged to round-off
    dim, p = 2, 2
    gt, ot, rng = adapted_pair(dim, (1, 1), 3, 3, 6, cycles=2)
    F = gt.connect()
    assert int(F["n_hang"]) > 0
    lvl, xyz = gt.leaf_boxes()
    M, N = lvl.numel(), (p + 1) ** dim
    z, w = np.polynomial.legendre.leggauss(p + 1)
    L = float(1 << 6)
    wd = (1 << (6 - lvl.cpu().numpy().astype(np.int64))) / L
    X = np.zeros((M, N, 2))
    for n in range(N):
        X[:, n, 0] = xyz[:, 0].cpu().numpy() / L + 0.5 * wd * (1 + z[n % (p + 1)])
        X[:, n, 1] = xyz[:, 1].cpu().numpy() / L + 0.5 * wd * (1 + z[n // (p + 1)])
    rho = 1.0 + 0.2 * np.sin(2 * np.pi * X[..., 0]) * np.cos(2 * np.pi * X[..., 1])
    vx, vy, pr = 0.5 + 0.1 * np.cos(2 * np.pi * X[..., 1]), -0.3 + 0.1 * np.sin(2 * np.pi * X[..., 0]), 1.0
    U = np.stack([rho, rho * vx, rho * vy, pr / 0.4 + 0.5 * rho * (vx ** 2 + vy ** 2)], axis=1)
    un = torch.from_numpy(U).cuda()
    wv = torch.from_numpy(np.kron(w, w)).cuda()
    vol = torch.from_numpy((wd / 2) ** 2).cuda()

    def integral(u):
        return ((u @ wv) * vol[:, None]).sum(0)

    dt = 1e-3
    fs, R = gpu_pipeline(gt, un, p)
    u1 = gt.rk3_stage(1, dt, un, un, R, p)
    fs, _ = gpu_pipeline(gt, u1, p)
    u2 = gt.fr_stage(2, dt, un, u1, fs, p)          # fused right-hand side + stage
    fs, _ = gpu_pipeline(gt, u2, p)
    u3 = gt.fr_stage(3, dt, un, u2, fs, p)
    assert float((u3 - un).abs().max()) > 1e-5                      # the step did something
    assert float((integral(u3) - integral(un)).abs().max()) < 1e-13


@pytest.mark.parametrize("dim,base,maxl", [(2, 2, 6), (3, 2, 4), (3, 4, 6), (2, 7, 9)])
@pytest.mark.parametrize("p", [0, 1, 2, 3, 5, 7])
def test_fused_face_pass_and_stage_with_traces(dim, base, maxl, p):
    """lt_face_flux (Alg. 8 steps 2 + 3 in one pass, a conforming face computed once for both sides) and
    lt_fr_stage_faces (right-hand side + Eq. 6 + the traces of the result) against the oracle's unfused
    chain: common fluxes on every kind 1 / 2 slot, untouched slots untouched, the stage result, and the
    face traces of the stage result = the oracle's face_interp of the oracle's stage result."""
    if dim == 3 and p == 7:
        maxl = 3
    if base > 2 and p not in (1, 3):
        pytest.skip("the larger meshes (many tiles per block of the bulk-copy face pass) run p = 1 and 3 only")
    gt, ot, rng = adapted_pair(dim, (1,) * dim, 71 * dim + p, base, maxl, cycles=2)
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
        for a2 in range(dim):
            X[:, n, a2] = xyz[:, a2] / Lw + 0.5 * wd * (1 + z[r % (p + 1)])
            r //= p + 1
    ph = 2 * np.pi * X
    rho = 1.0 + 0.2 * np.prod(np.sin(ph), axis=-1)
    vel = np.stack([0.4 + 0.1 * np.cos(ph[..., (a2 + 1) % dim]) for a2 in range(dim)], axis=-1)
    pr = 1.0 + 0.1 * np.cos(ph[..., 0])
    u = np.concatenate([rho[:, None], np.moveaxis(rho[..., None] * vel, -1, 1),
                        (pr / 0.4 + 0.5 * rho * np.sum(vel * vel, -1))[:, None]], axis=1).copy()
    u_n = u * (1.0 + 0.01 * rng.uniform(-1, 1, u.shape))
    dt = 1e-3
    # oracle, unfused
    uf_o = ot.face_interp(u, p, nv)
    fs_o = ot.common_flux(uf_o, ot.mortar_project(uf_o, p, nv), p)
    fs_full = np.where(np.isnan(fs_o), ot.mortar_gather(fs_o, p, nv), fs_o)
    R_o = ot.fr_rhs(u, fs_full, p, [1.0] * dim)
    lvl_max = int(lvl.max())
    for stage in (2, 3):
        want = oracle.rk3_stage(stage, dt, u_n, u, R_o)
        want_uf = ot.face_interp(want, p, nv)
        # GPU, fused
        d_u = torch.from_numpy(u).cuda()
        uf = gt.face_interp(d_u, p, nv)
        fs = gt.face_flux(uf, p)
        close(fs, fs_o, "face_flux")                      # NaN (untouched) exactly on the kind 0 / 3 slots
        gt.mortar_gather(fs, p, nv, f_face=fs)
        close(fs, fs_full, "face_flux + gather")
        out, uf2 = gt.fr_stage_faces(stage, dt, torch.from_numpy(u_n).cuda(), d_u, fs, p)
        tol = 1e-12 * max(1.0, float(np.abs(want).max()), dt * float(2 << lvl_max) * float(np.abs(fs_full).max()))
        assert float(np.abs(out.cpu().numpy() - want).max()) <= tol
        assert float(np.abs(uf2.cpu().numpy() - want_uf).max()) <= 4 * tol
        # the traces may overwrite the fluxes (an element touches only its own slots)
        fs2 = fs.clone()
        out2, uf3 = gt.fr_stage_faces(stage, dt, torch.from_numpy(u_n).cuda(), d_u, fs2, p, u_face_out=fs2)
        assert torch.equal(out2, out) and torch.equal(uf3, uf2) and uf3.data_ptr() == fs2.data_ptr()
        # and the plain right-hand side of the re-laid-out kernel
        close_rhs(gt.fr_rhs(d_u, fs, p), R_o, fs_full, ot, "fr_rhs (padded layout)")
        if dim == 3 and p == 3 and stage == 2:
            # the 3-D p = 3 kernel fetches an element's flux blocks by cp.async.bulk when the flux array is
            # 16-byte aligned and by 8-byte cp.async otherwise: a flux array that starts 8 bytes into an
            # allocation takes the second path and must give the same bits
            raw = torch.empty(fs.numel() + 1, dtype=torch.float64, device="cuda")
            fs_odd = raw[1:].view(fs.shape)
            fs_odd.copy_(fs)
            assert fs.data_ptr() % 16 == 0 and fs_odd.data_ptr() % 16 == 8
            assert torch.equal(gt.fr_stage(stage, dt, torch.from_numpy(u_n).cuda(), d_u, fs_odd, p), out)
    gt.sync()
