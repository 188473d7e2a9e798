"""Pins for the oracle's flux-reconstruction pieces around the cycle (Eq. 1-6, and
Alg. 8 step 3; readings I-1..I-5): Euler flux, Rusanov common flux,
the FR right-hand side with Radau correction functions, chained with the Alg. 8 face / mortar calls.

Sources of truth: closed forms of the operators (p = 0, 1), textbook identities of the Rusanov
flux, discrete conservation of the corrected flux derivative (GL quadrature of Eq. 4 is exact), a
first-order finite-volume formula written in numpy for p = 0, free-stream preservation and an
exactly differentiable manufactured state on adapted meshes with hanging faces.
"""
import numpy as np
import pytest

import oracle
from test_oracle_mortar import adapted_tree, face_points, volume_points, gl

G = 1.4


def euler_flux_np(U, a, dim):
    rho, E = U[..., 0], U[..., dim + 1]
    v = U[..., 1:1 + dim] / rho[..., None]
    p = (G - 1) * (E - 0.5 * rho * np.sum(v * v, -1))
    F = np.empty_like(U)
    F[..., 0] = rho * v[..., a]
    for b in range(dim):
        F[..., 1 + b] = U[..., 1 + b] * v[..., a] + (p if b == a else 0.0)
    F[..., dim + 1] = (E + p) * v[..., a]
    return F


def random_states(rng, shape, dim):
    rho = rng.uniform(0.5, 2.0, shape)
    v = rng.uniform(-1.0, 1.0, shape + (dim,))
    p = rng.uniform(0.5, 2.0, shape)
    U = np.empty(shape + (dim + 2,))
    U[..., 0] = rho
    U[..., 1:1 + dim] = rho[..., None] * v
    U[..., dim + 1] = p / (G - 1) + 0.5 * rho * np.sum(v * v, -1)
    return U


# ---------------------------------------------------------------- operators
def test_fr_operator_closed_forms():
    D, lm, lp, gl_, gr_ = oracle.fr_operators(0)
    assert D.shape == (1, 1) and D[0, 0] == 0.0 and lm[0] == lp[0] == 1.0
    assert abs(gl_[0] + 0.5) < 1e-15 and abs(gr_[0] - 0.5) < 1e-15          # g_L = (1 - xi)/2
    D, lm, lp, gl_, gr_ = oracle.fr_operators(1)
    s3 = np.sqrt(3.0)
    assert np.allclose(D, [[-s3 / 2, s3 / 2]] * 2, atol=1e-15)
    assert np.allclose(lm, [(1 + s3) / 2, (1 - s3) / 2], atol=1e-15) and np.allclose(lp, lm[::-1], atol=1e-15)
    assert np.allclose(gl_, [0.5 * (-s3 - 1), 0.5 * (s3 - 1)], atol=1e-15)  # g_L' = (3 xi - 1)/2
    assert np.allclose(gr_, -gl_[::-1], atol=1e-15)
    for p in range(0, 6):
        D, lm, lp, gl_, gr_ = oracle.fr_operators(p)
        z, w = gl(p + 1)
        # differentiation is exact for degree <= p; rows of D sum to zero; the basis sums to one at +-1
        for k in range(p + 1):
            assert np.max(np.abs(D @ z ** k - (k * z ** (k - 1) if k else 0 * z))) < 1e-12
        assert abs(lm.sum() - 1) < 1e-13 and abs(lp.sum() - 1) < 1e-13
        # Radau: int g_L' = g_L(1) - g_L(-1) = -1, int g_R' = +1, and g' is orthogonal to degree <= p - 1
        assert abs(w @ gl_ + 1) < 1e-13 and abs(w @ gr_ - 1) < 1e-13
        for k in range(1, p + 1):
            # int g_L' xi^k = [g_L xi^k] - k int g_L xi^(k-1) = -(-1)^k  (g_L orthogonal to P_(p-1))
            assert abs(w @ (gl_ * z ** k) + (-1.0) ** k) < 1e-12
            assert abs(w @ (gr_ * z ** k) - 1.0) < 1e-12


# ---------------------------------------------------------------- Rusanov flux on the face arrays
@pytest.mark.parametrize("dim", [2, 3])
def test_common_flux_identities(dim):
    p = 2
    t = adapted_tree(dim, (1,) * dim, 5)
    F = t.connect()
    kind = F["kind"].reshape(-1, t.nf) & 15
    rng = np.random.default_rng(dim)
    Nf = (p + 1) ** (dim - 1)
    M = t.num_leaves()
    U = np.moveaxis(random_states(rng, (M, t.nf, Nf), dim), -1, 2)  # [M, nf, nv, Nf]
    m12 = (kind == 1) | (kind == 2)
    # consistency: F*(u, u) = F_a(u)
    fs = t.common_flux(U, U, p)
    assert np.isnan(fs[~m12]).all()
    for f in range(t.nf):
        want = np.moveaxis(euler_flux_np(np.moveaxis(U[:, f], 1, -1), f >> 1, dim), -1, 1)
        sel = m12[:, f]
        assert np.max(np.abs(fs[sel, f] - want[sel])) < 1e-13
    # the textbook formula, with the minus-side state decided by the face parity
    V = np.moveaxis(random_states(rng, (M, t.nf, Nf), dim), -1, 2)
    fs = t.common_flux(U, V, p)
    for f in range(t.nf):
        a = f >> 1
        own, nb = np.moveaxis(U[:, f], 1, -1), np.moveaxis(V[:, f], 1, -1)
        L, R = (own, nb) if f & 1 else (nb, own)

        def speed(W):
            rho = W[..., 0]
            v = W[..., 1:1 + dim] / rho[..., None]
            pr = (G - 1) * (W[..., dim + 1] - 0.5 * rho * np.sum(v * v, -1))
            return np.abs(v[..., a]) + np.sqrt(G * pr / rho)
        lam = np.maximum(speed(L), speed(R))
        want = 0.5 * (euler_flux_np(L, a, dim) + euler_flux_np(R, a, dim)) - 0.5 * lam[..., None] * (R - L)
        sel = m12[:, f]
        assert np.max(np.abs(fs[sel, f] - np.moveaxis(want, -1, 1)[sel])) < 1e-13
    # gas at rest, equal pressure, density jump: F* = (-c_max (rho_R - rho_L)/2, p e_a, -c_max (E_R - E_L)/2)
    L = np.zeros(dim + 2); R = np.zeros(dim + 2)
    L[0], R[0] = 1.0, 0.25
    L[dim + 1] = R[dim + 1] = 1.0 / (G - 1)
    tt = oracle.Tree(dim, 0, 1, (1,) * dim)
    tt.connect()
    own = np.tile(L[None, None, :, None], (1, 2 * dim, 1, 1))
    nb = np.tile(R[None, None, :, None], (1, 2 * dim, 1, 1))
    fs = tt.common_flux(own, nb, 0)[0, 1, :, 0]  # face +x: own = minus side
    c = np.sqrt(G * 1.0 / 0.25)
    assert np.allclose(fs, [-0.5 * c * (0.25 - 1.0), 1.0] + [0.0] * (dim - 1) + [0.0], atol=1e-14)


# ---------------------------------------------------------------- the right-hand side
def pipeline(t, u, p):
    """Alg. 8 steps 1-4 then Eq. 2-5, all on the oracle: returns (f_star, rhs)."""
    nv = t.dim + 2
    uf = t.face_interp(u, p, nv)
    unb = t.mortar_project(uf, p, nv)
    fs = t.common_flux(uf, unb, p)
    g = t.mortar_gather(fs, p, nv)
    fs = np.where(np.isnan(fs), g, fs)      # coarse-side hanging slots receive the projected mortar fluxes
    assert not np.isnan(fs).any()
    return fs, t.fr_rhs(u, fs, p, [1.0] * t.dim)


@pytest.mark.parametrize("dim", [2, 3])
@pytest.mark.parametrize("p", [0, 1, 2, 3])
def test_free_stream_is_preserved_on_adapted_meshes(dim, p):
    t = adapted_tree(dim, (1,) * dim, 20 + p)
    t.connect()
    N = (p + 1) ** dim
    state = random_states(np.random.default_rng(1), (), dim)
    u = np.tile(state[None, :, None], (t.num_leaves(), 1, N))
    _, R = pipeline(t, u, p)
    assert np.max(np.abs(R)) < 1e-10


@pytest.mark.parametrize("dim", [2, 3])
@pytest.mark.parametrize("p", [1, 2, 3])
def test_manufactured_state_is_differentiated_exactly(dim, p):
    # density = polynomial of degree <= p in every coordinate, constant velocity v0 and pressure p0: every
    # flux is linear in rho, the traces are continuous (so the Rusanov flux is the exact flux and, through
    # the mortars, stays exact on hanging faces) and R = -(v0 . grad rho) (1, v0, |v0|^2 / 2).
    # Non-periodic mesh: boundary slots get the exact flux by hand.
    t = adapted_tree(dim, (0,) * dim, 30 + p)
    F = t.connect()
    kind = F["kind"].reshape(-1, t.nf) & 15
    X, XF = volume_points(t, p), face_points(t, p, wrap=False)
    v0 = np.array([0.7, -0.4, 0.3][:dim])
    p0 = 1.3

    def rho_of(Xp):
        r = np.ones(Xp.shape[:-1]) * 2.0
        for a in range(dim):
            r = r + sum((0.2 + 0.1 * a + 0.05 * k) * Xp[..., a] ** k for k in range(1, p + 1))
        return r

    def grad_rho(Xp):
        g = np.zeros(Xp.shape)
        for a in range(dim):
            g[..., a] = sum(k * (0.2 + 0.1 * a + 0.05 * k) * Xp[..., a] ** (k - 1) for k in range(1, p + 1))
        return g

    def state(r):
        U = np.empty(r.shape + (dim + 2,))
        U[..., 0] = r
        U[..., 1:1 + dim] = r[..., None] * v0
        U[..., dim + 1] = p0 / (G - 1) + 0.5 * r * (v0 @ v0)
        return U
    u = np.moveaxis(state(rho_of(X)), -1, 1)                      # [M, nv, N]
    nv = dim + 2
    uf = t.face_interp(u, p, nv)
    assert np.max(np.abs(uf - np.moveaxis(state(rho_of(XF)), -1, 2))) < 1e-12
    unb = t.mortar_project(uf, p, nv)
    fs = t.common_flux(uf, unb, p)
    g = t.mortar_gather(fs, p, nv)
    fs = np.where(np.isnan(fs), g, fs)
    for f in range(t.nf):                                          # boundary slots: the exact flux
        bsel = kind[:, f] == 0
        exact = np.moveaxis(euler_flux_np(np.moveaxis(uf[:, f], 1, -1), f >> 1, dim), -1, 1)
        fs[bsel, f] = exact[bsel]
    assert not np.isnan(fs).any()
    R = t.fr_rhs(u, fs, p, [1.0] * dim)
    adv = -(grad_rho(X) @ v0)                                      # [M, N]
    want = np.stack([adv] + [adv * v0[b] for b in range(dim)] + [adv * 0.5 * (v0 @ v0)], axis=1)
    assert np.max(np.abs(R - want)) < 1e-9 * max(1.0, np.max(np.abs(want)))


@pytest.mark.parametrize("dim", [2, 3])
@pytest.mark.parametrize("p", [0, 1, 2, 3])
def test_rhs_is_conservative_for_arbitrary_data(dim, p):
    # int over the element of R = - sum_a (2/dx) int (corrected flux)' = - sum_a (F*_+ - F*_-) integrated over
    # the face: the (p+1)-point GL rule integrates Eq. 4 (degree p in xi) exactly, whatever u and F* are
    t = adapted_tree(dim, (1,) * dim, 40 + p)
    t.connect()
    rng = np.random.default_rng(p)
    M, N, Nf, nv = t.num_leaves(), (p + 1) ** dim, (p + 1) ** (dim - 1), dim + 2
    u = np.moveaxis(random_states(rng, (M, N), dim), -1, 1)
    fs = rng.uniform(-1, 1, (M, t.nf, nv, Nf))
    R = t.fr_rhs(u, fs, p, [1.0] * dim)
    _, w = gl(p + 1)
    wv = w
    for _ in range(dim - 1):
        wv = np.kron(w, wv)
    wf = w if dim == 2 else np.kron(w, w)
    lvl, _ = t.leaf_boxes()
    dx = 1.0 / (1 << lvl.astype(np.int64))
    lhs = (R @ wv) * (dx[:, None] / 2) ** dim                      # element integral of R, [M, nv]
    rhs = np.zeros((M, nv))
    for a in range(dim):
        rhs -= ((fs[:, 2 * a + 1] - fs[:, 2 * a]) @ wf) * (dx[:, None] / 2) ** (dim - 1)
    assert np.max(np.abs(lhs - rhs)) < 1e-11


def test_p0_is_first_order_finite_volume():
    dim, p = 2, 0
    t = adapted_tree(dim, (1, 1), 9)
    t.connect()
    rng = np.random.default_rng(0)
    M = t.num_leaves()
    u = np.moveaxis(random_states(rng, (M, 1), dim), -1, 1)
    fs, R = pipeline(t, u, p)
    lvl, _ = t.leaf_boxes()
    dx = 1.0 / (1 << lvl.astype(np.int64))
    want = np.zeros((M, 4))
    for a in range(dim):
        want -= (fs[:, 2 * a + 1, :, 0] - fs[:, 2 * a, :, 0]) / dx[:, None]
    assert np.max(np.abs(R[:, :, 0] - want)) < 1e-11


# ---------------------------------------------------------------- pins that do not re-type the flux formula
def _read_fractions(name):
    import os
    from fractions import Fraction
    out = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", name)) as fh:
        for line in fh:
            if line.startswith("#") or not line.strip():
                continue
            k, a, b = line.split()
            out[k] = Fraction(int(a), int(b))
    return out


@pytest.mark.parametrize("dim,axis", [(2, 0), (2, 1), (3, 0), (3, 2)])
def test_rusanov_hand_computed_value(dim, axis):
    """tests/golden/rusanov_hand.txt: both states move, so a dropped '+ p' in (E + p) v_a or a wrong
    sound speed changes the stored numbers.  Other axes / 3-D: the same states with the velocity
    components permuted (the Euler flux is isotropic), w = 0 in 3-D."""
    g = _read_fractions("rusanov_hand.txt")
    uL = np.array([float(g["uL_%d" % k]) for k in range(4)])
    uR = np.array([float(g["uR_%d" % k]) for k in range(4)])
    want = np.array([float(g["Fstar_%d" % k]) for k in range(4)])
    tang = [b for b in range(dim) if b != axis][0]     # the axis that receives the stored vy

    def embed(v4):
        out = np.zeros(dim + 2)
        out[0], out[dim + 1] = v4[0], v4[3]
        out[1 + axis], out[1 + tang] = v4[1], v4[2]
        return out
    t = oracle.Tree(dim, 0, 1, (1,) * dim)
    t.connect()
    own = np.tile(embed(uL)[None, None, :, None], (1, 2 * dim, 1, 1))
    nb = np.tile(embed(uR)[None, None, :, None], (1, 2 * dim, 1, 1))
    fs = t.common_flux(own, nb, 0)[0, 2 * axis + 1, :, 0]      # plus face: own = minus-side state
    assert np.max(np.abs(fs - embed(want))) < 4e-16 * 4
    # seen from the other element (minus face, own = plus-side state) it is the same flux along +a
    fs2 = t.common_flux(nb, own, 0)[0, 2 * axis, :, 0]
    assert np.array_equal(fs, fs2)


@pytest.mark.parametrize("dim", [2, 3])
@pytest.mark.parametrize("p", [1, 2, 3])
def test_manufactured_pressure_field_pins_energy_flux(dim, p):
    """Constant density rho0 and velocity v0, pressure = polynomial of degree <= p per coordinate:
    every flux is affine in the pressure, the traces are continuous (Rusanov = exact flux, exact
    through the mortars) and the divergence is known in closed form,
        R_rho = 0,   R_(rho v_a) = -d p / d x_a,   R_E = -gamma/(gamma-1) v0 . grad p,
    because (E + p) v0 = (gamma/(gamma-1) p + rho0 |v0|^2 / 2) v0.  With E v0 instead of (E + p) v0
    the last component would be -1/(gamma-1) v0 . grad p: the case separates the two."""
    t = adapted_tree(dim, (0,) * dim, 60 + p)
    F = t.connect()
    kind = F["kind"].reshape(-1, t.nf) & 15
    X, XF = volume_points(t, p), face_points(t, p, wrap=False)
    v0 = np.array([0.6, -0.35, 0.45][:dim])
    rho0 = 1.3

    def pr_of(Xp):
        r = np.ones(Xp.shape[:-1]) * 2.5
        for a in range(dim):
            r = r + sum((0.3 - 0.07 * a + 0.04 * k) * Xp[..., a] ** k for k in range(1, p + 1))
        return r

    def grad_pr(Xp):
        g = np.zeros(Xp.shape)
        for a in range(dim):
            g[..., a] = sum(k * (0.3 - 0.07 * a + 0.04 * k) * Xp[..., a] ** (k - 1) for k in range(1, p + 1))
        return g

    def state(pr):
        U = np.empty(pr.shape + (dim + 2,))
        U[..., 0] = rho0
        U[..., 1:1 + dim] = rho0 * v0
        U[..., dim + 1] = pr / (G - 1) + 0.5 * rho0 * (v0 @ v0)
        return U
    nv = dim + 2
    u = np.moveaxis(state(pr_of(X)), -1, 1)
    uf = t.face_interp(u, p, nv)
    assert np.max(np.abs(uf - np.moveaxis(state(pr_of(XF)), -1, 2))) < 1e-12
    unb = t.mortar_project(uf, p, nv)
    fs = t.common_flux(uf, unb, p)
    g = t.mortar_gather(fs, p, nv)
    fs = np.where(np.isnan(fs), g, fs)
    # boundary slots: the exact flux, written out for THIS state (not through a flux routine):
    # F_a = (rho0 v0_a, rho0 v0 v0_a + p e_a, (gamma/(gamma-1) p + rho0 |v0|^2/2) v0_a)
    prF = pr_of(XF)                                                # [M, nf, Nf]
    for f in range(t.nf):
        a = f >> 1
        ex = np.zeros((t.num_leaves(), nv, prF.shape[-1]))
        ex[:, 0] = rho0 * v0[a]
        for b in range(dim):
            ex[:, 1 + b] = rho0 * v0[b] * v0[a] + (prF[:, f] if b == a else 0.0)
        ex[:, dim + 1] = (G / (G - 1) * prF[:, f] + 0.5 * rho0 * (v0 @ v0)) * v0[a]
        bsel = kind[:, f] == 0
        fs[bsel, f] = ex[bsel]
        # and on the interior slots the common flux IS this exact flux (continuous traces)
        isel = ~bsel
        assert np.max(np.abs(fs[isel, f] - ex[isel])) < 1e-11
    assert not np.isnan(fs).any()
    R = t.fr_rhs(u, fs, p, [1.0] * dim)
    gp = grad_pr(X)                                                # [M, N, dim]
    want = np.stack([np.zeros(gp.shape[:2])] + [-gp[..., b] for b in range(dim)] + [-(G / (G - 1)) * (gp @ v0)], axis=1)
    assert np.max(np.abs(R - want)) < 1e-9 * max(1.0, np.max(np.abs(want)))


# ---------------------------------------------------------------- Eq. 6
def test_rk3_amplification_polynomial_and_order():
    """Eq. 6 on u' = lambda u: one step multiplies u by 1 + z + z^2/2 + z^3/6, z = lambda dt
    (the three-stage third-order scheme reproduces the Taylor polynomial of e^z); any swapped or
    misplaced coefficient changes the polynomial.  Then third-order convergence on a nonlinear ODE."""
    rng = np.random.default_rng(0)
    un = rng.uniform(0.5, 1.5, 7)
    for lam, dt in ((-1.3, 0.2), (0.7, 0.5), (-4.0, 0.05)):
        u1 = oracle.rk3_stage(1, dt, un, un, lam * un)
        u2 = oracle.rk3_stage(2, dt, un, u1, lam * u1)
        u3 = oracle.rk3_stage(3, dt, un, u2, lam * u2)
        z = lam * dt
        assert np.max(np.abs(u1 - (1 + z) * un)) < 1e-15
        assert np.max(np.abs(u3 - (1 + z + z * z / 2 + z ** 3 / 6) * un)) < 2e-15
    # u' = -u^2, u(0) = 1 -> u(t) = 1/(1+t): error at t = 1 falls by ~8 when dt is halved
    errs = []
    for nsteps in (20, 40, 80):
        u = np.array([1.0])
        dt = 1.0 / nsteps
        for _ in range(nsteps):
            u1 = oracle.rk3_stage(1, dt, u, u, -u * u)
            u2 = oracle.rk3_stage(2, dt, u, u1, -u1 * u1)
            u = oracle.rk3_stage(3, dt, u, u2, -u2 * u2)
        errs.append(abs(u[0] - 0.5))
    assert 7.0 < errs[0] / errs[1] < 9.0 and 7.0 < errs[1] / errs[2] < 9.0
    with pytest.raises(oracle.OracleError):
        oracle.rk3_stage(4, 0.1, un, un, un)
