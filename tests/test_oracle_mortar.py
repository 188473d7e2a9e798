"""Pins for the oracle's mortar operators (Alg. 8 steps 2 and 4, Eq. 14-20, PAPER.md:265-314;
DESIGN.md readings H-1..H-4).

Sources of truth: Gauss-Legendre closed forms (the Eq. 17 projection of a coarse trace onto a
mortar is interpolation because the trace lies in the mortar space; the Eq. 20 operator is
(1/2) W^-1 I^T W per tangential axis), the values the paper-fixed p = 1 rule gives, partition /
conservation identities, and polynomial traces sampled analytically on every face of an adapted
mesh -- a wrong slot, axis order, face orientation or neighbour index fails the last one.
"""
import numpy as np
import pytest

import oracle


def gl(n):
    z, w = np.polynomial.legendre.leggauss(n)
    return z, w


def interp_1d(p, b):
    z, _ = gl(p + 1)
    xi = 0.5 * (z + 2 * b - 1)
    I = np.ones((p + 1, p + 1))
    for m in range(p + 1):
        for i in range(p + 1):
            for k in range(p + 1):
                if k != i:
                    I[m, i] *= (xi[m] - z[k]) / (z[i] - z[k])
    return I


@pytest.mark.parametrize("dim", [2, 3])
@pytest.mark.parametrize("p", [0, 1, 2, 3, 4])
def test_face_operators_closed_forms(dim, p):
    to_m, from_m = oracle.face_operators(dim, p)
    _, w = gl(p + 1)
    for s in range(1 << (dim - 1)):
        I = [interp_1d(p, (s >> a) & 1) for a in range(dim - 1)]
        R = [0.5 * (I[a].T * w[None, :]) / w[:, None] for a in range(dim - 1)]
        # tangential axes ascending, lower axis fastest: n = n0 + P1 * n1  ->  kron(axis1, axis0)
        Ik = I[0] if dim == 2 else np.kron(I[1], I[0])
        Rk = R[0] if dim == 2 else np.kron(R[1], R[0])
        assert np.max(np.abs(to_m[s] - Ik)) < 5e-15      # Eq. 17 = interpolation
        assert np.max(np.abs(from_m[s] - Rk)) < 5e-15    # Eq. 20 = (1/2) W^-1 I^T W per axis
    # coarse -> mortars -> coarse is the identity; rows of the interpolation sum to one
    N = (p + 1) ** (dim - 1)
    assert np.max(np.abs(sum(from_m[s] @ to_m[s] for s in range(1 << (dim - 1))) - np.eye(N))) < 5e-15
    assert np.max(np.abs(to_m.sum(axis=2) - 1.0)) < 5e-15
    # conservation: the face integral of the projected flux equals the sum of the
    # mortar integrals, each mortar having 2^-(dim-1) of the coarse face's area
    wf = w if dim == 2 else np.kron(w, w)
    for s in range(1 << (dim - 1)):
        assert np.max(np.abs(wf @ from_m[s] - wf / (1 << (dim - 1)))) < 5e-15


def test_p1_values():
    # p = 1, 2-D: the 1-D operators printed in tests/golden/paper_values.txt (SURVEY 8(c) v)
    to_m, from_m = oracle.face_operators(2, 1)
    s3 = np.sqrt(3.0)
    want = np.array([[(3 + s3) / 4, (1 - s3) / 4], [(1 + s3) / 4, (3 - s3) / 4]])
    assert np.max(np.abs(to_m[0] - want)) < 5e-15
    assert np.max(np.abs(to_m[1] - want[::-1, ::-1])) < 5e-15
    assert np.max(np.abs(from_m[0] - 0.5 * want.T)) < 5e-15


def adapted_tree(dim, periodic, seed, base=2, maxl=4):
    rng = np.random.default_rng(seed)
    t = oracle.Tree(dim, base, maxl, periodic)
    for _ in range(2):
        f = (rng.random(t.num_leaves()) < 0.3).astype(np.int8)
        t.adapt(f)
        t.balance()
        t.drop_snapshot()
    return t


def face_points(t, p, wrap=True):
    """Physical coordinates [M, nf, Nf, dim] of every face's Gauss-Legendre points on the unit
    domain; the normal coordinate is the face plane taken modulo the domain (a periodic face and
    its image share it), tangential axes ascending, lower axis fastest (reading H-1)."""
    lvl, xyz = t.leaf_boxes()
    dim, nf, D = t.dim, t.nf, t.maxl
    z, _ = gl(p + 1)
    P1 = p + 1
    Nf = P1 ** (dim - 1)
    L = float(1 << D)
    out = np.zeros((len(lvl), nf, Nf, dim))
    for e in range(len(lvl)):
        w = float(1 << (D - int(lvl[e])))
        for f in range(nf):
            ax = f >> 1
            tang = [a for a in range(dim) if a != ax]
            for n in range(Nf):
                r = n
                for a in tang:
                    out[e, f, n, a] = (xyz[e, a] + 0.5 * w * (1 + z[r % P1])) / L
                    r //= P1
                plane = xyz[e, ax] + (w if f & 1 else 0.0)
                out[e, f, n, ax] = ((plane % L) if wrap else plane) / L
    return out


def poly(X, p, dim):
    # degree <= p in every coordinate, all axes coupled
    v = np.ones(X.shape[:-1])
    for a in range(dim):
        v = v * sum((0.3 + 0.5 * a + k) * X[..., a] ** k for k in range(p + 1))
    return v


@pytest.mark.parametrize("dim,periodic", [(2, (0, 0)), (2, (1, 1)), (3, (0, 0, 0)), (3, (1, 0, 1))])
@pytest.mark.parametrize("p", [1, 2, 3])
def test_polynomial_traces_are_reproduced(dim, periodic, p):
    t = adapted_tree(dim, periodic, 10 * dim + p)
    F = t.connect()
    kind = F["kind"].reshape(-1, t.nf) & 15
    assert (kind == 2).any() and (kind == 3).any()
    X = face_points(t, p)
    # a polynomial of the tangential coordinates and of the (wrapped) face-plane coordinate: both
    # sides of every face, periodic images included, sample the same trace
    nvars = 2
    q = poly(X, p, dim)
    if any(periodic):
        # across a periodic boundary the tangential coordinates are unchanged but the global
        # polynomial is not periodic in them either -- restrict to faces whose neighbour is not
        # a periodic image by making q depend only on coordinates of non-periodic axes
        Xn = X.copy()
        for a in range(dim):
            if periodic[a]:
                Xn[..., a] = 0.0
        q = poly(Xn, p, dim)
    uf = np.stack([q, 2.0 - 3.0 * q], axis=2)  # [M, nf, nvars, Nf]
    unb = t.mortar_project(uf, p, nvars)
    m12 = (kind == 1) | (kind == 2)
    assert np.isnan(unb[~m12]).all()
    tol = 1e-13 * max(1.0, float(np.max(np.abs(uf))))
    assert np.max(np.abs(unb[m12] - uf[m12])) < tol
    ff = t.mortar_gather(uf, p, nvars)
    m3 = kind == 3
    assert np.isnan(ff[~m3]).all()
    assert np.max(np.abs(ff[m3] - uf[m3])) < tol


@pytest.mark.parametrize("dim", [2, 3])
def test_gather_conserves_random_fluxes(dim):
    p, nvars = 2, 3
    t = adapted_tree(dim, (1,) * dim, 77)
    F = t.connect()
    kind = F["kind"].reshape(-1, t.nf)
    nbr = F["nbr"].reshape(-1, t.nf)
    rng = np.random.default_rng(1)
    Nf = (p + 1) ** (dim - 1)
    fm = rng.uniform(-1, 1, (t.num_leaves(), t.nf, nvars, Nf))
    ff = t.mortar_gather(fm, p, nvars)
    _, w = gl(p + 1)
    wf = w if dim == 2 else np.kron(w, w)
    # integral over the coarse face = sum of the integrals over the fine faces that point at it
    coarse_int = {}
    for e, f in zip(*np.nonzero((kind & 15) == 2)):
        key = (int(nbr[e, f]), int(f) ^ 1)
        coarse_int[key] = coarse_int.get(key, 0.0) + (fm[e, f] @ wf) / (1 << (dim - 1))
    assert coarse_int
    for (e, f), val in coarse_int.items():
        assert (kind[e, f] & 15) == 3
        assert np.max(np.abs(ff[e, f] @ wf - val)) < 1e-13


# ---------------------------------------------------------------- Alg. 8 step 1: volume -> face points
def volume_points(t, p):
    """Physical coordinates [M, N, dim] of the solution points (reading E-5: x fastest)."""
    lvl, xyz = t.leaf_boxes()
    dim, D = t.dim, t.maxl
    z, _ = gl(p + 1)
    P1 = p + 1
    N = P1 ** dim
    L = float(1 << D)
    out = np.zeros((len(lvl), N, dim))
    for n in range(N):
        r = n
        for a in range(dim):
            out[:, n, a] = (xyz[:, a] + 0.5 * (1 << (D - lvl.astype(np.int64))) * (1 + z[r % P1])) / L
            r //= P1
    return out


@pytest.mark.parametrize("dim", [2, 3])
@pytest.mark.parametrize("p", [0, 1, 2, 3])
def test_face_interp_reproduces_polynomials(dim, p):
    t = adapted_tree(dim, (0,) * dim, 3 + p)
    XV, XF = volume_points(t, p), face_points(t, p, wrap=False)
    u = np.stack([poly(XV, p, dim), 1.0 - 2.0 * poly(XV, p, dim)], axis=1)       # [M, 2, N]
    want = np.stack([poly(XF, p, dim), 1.0 - 2.0 * poly(XF, p, dim)], axis=2)    # [M, nf, 2, Nf]
    got = t.face_interp(u, p, 2)
    assert np.max(np.abs(got - want)) < 1e-13 * max(1.0, np.max(np.abs(want)))


def test_face_interp_p1_closed_form():
    # p = 1: l_0(-1) = (1 + sqrt 3)/2, l_1(-1) = (1 - sqrt 3)/2 (Lagrange basis on +-1/sqrt 3), mirrored at +1
    t = oracle.Tree(2, 0, 1)
    a, b = (1 + np.sqrt(3.0)) / 2, (1 - np.sqrt(3.0)) / 2
    u = np.arange(4, dtype=np.float64).reshape(1, 1, 4)  # u[iy*2 + ix]
    uf = t.face_interp(u, 1, 1)[0, :, 0, :]
    assert np.allclose(uf[0], [a * 0 + b * 1, a * 2 + b * 3], atol=1e-15)   # -x face, points along y
    assert np.allclose(uf[1], [b * 0 + a * 1, b * 2 + a * 3], atol=1e-15)   # +x
    assert np.allclose(uf[2], [a * 0 + b * 2, a * 1 + b * 3], atol=1e-15)   # -y face, points along x
    assert np.allclose(uf[3], [b * 0 + a * 2, b * 1 + a * 3], atol=1e-15)   # +y
    # constants are reproduced (the basis sums to one)
    assert np.allclose(t.face_interp(np.ones((1, 3, 16)), 3, 3), 1.0, atol=1e-14)
