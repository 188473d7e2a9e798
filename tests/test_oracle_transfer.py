"""Pins for the oracle's old/new map (Alg. 7) and FR data transfer (Eq. 8-13).

The oracle builds dense tensor operators by over-integrated quadrature and Gaussian
elimination; the pins are closed forms (Gauss-Legendre nodes, the p = 1, 2 interpolation
entries, R = 1/2 W^-1 I^T W), algebraic identities (sum_c R_c I_c = Id, mean conservation,
partition of unity), exact transfer of polynomial data through whole cycles, and Alg. 7
restated on the sorted key arrays with Python's bisect (Eq. 7 cases).
"""
import bisect
import math
import os

import numpy as np
import pytest
import torch

import oracle
from paper_2306_06744_b200 import workloads as W

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def paper_values():
    out = {}
    for line in open(os.path.join(GOLD, "paper_values.txt")):
        s = line.split("#")[0].split()
        if len(s) == 2:
            out[s[0]] = float(s[1])
    return out


def test_gauss_legendre_closed_forms():
    z, w = oracle.gauss_legendre(1)
    assert z.tolist() == [0.0] and abs(w[0] - 2.0) < 1e-15
    z, w = oracle.gauss_legendre(2)
    assert np.allclose(z, [-1 / math.sqrt(3), 1 / math.sqrt(3)], atol=1e-15) and np.allclose(w, [1, 1], atol=1e-15)
    z, w = oracle.gauss_legendre(3)
    assert np.allclose(z, [-math.sqrt(0.6), 0, math.sqrt(0.6)], atol=1e-15)
    assert np.allclose(w, [5 / 9, 8 / 9, 5 / 9], atol=1e-15)
    for n in range(1, 14):
        z, w = oracle.gauss_legendre(n)
        assert np.all(np.diff(z) > 0)
        # exact for monomials up to degree 2n-1
        for k in range(2 * n):
            exact = 0.0 if k % 2 else 2.0 / (k + 1)
            assert abs(np.dot(w, z ** k) - exact) < 5e-15
        zl, wl = np.polynomial.legendre.leggauss(n)  # library routine
        assert np.allclose(z, zl, atol=2e-15) and np.allclose(w, wl, atol=2e-15)


def one_d_interp(p, b):
    """Closed form of Eq. 8 in 1-D: I^b[m][i] = l_i((z_m + 2b - 1)/2) on library GL nodes."""
    z = np.polynomial.legendre.leggauss(p + 1)[0]
    I = np.zeros((p + 1, p + 1))
    for m in range(p + 1):
        x = 0.5 * (z[m] + 2 * b - 1)
        for i in range(p + 1):
            I[m, i] = np.prod([(x - z[k]) / (z[i] - z[k]) for k in range(p + 1) if k != i])
    return I


def kron_op(ops1d):
    """Tensor operator with x fastest: n = ix + P1*(iy + P1*iz)  ->  kron(z-op, y-op, x-op)."""
    out = ops1d[0]
    for o in ops1d[1:]:
        out = np.kron(o, out)
    return out


def test_p1_p2_interpolation_values_from_the_paper():
    pv = paper_values()
    I = oracle.operators(2, 1)["interp"]  # [c][n][m], c = bx + 2 by
    # child 0 (bx = by = 0): entries are products of the 1-D closed-form values
    i0 = np.array([[pv["I0_p1_00"], pv["I0_p1_01"]], [pv["I0_p1_10"], pv["I0_p1_11"]]])
    assert np.allclose(i0, [[(3 + math.sqrt(3)) / 4, (1 - math.sqrt(3)) / 4],
                            [(1 + math.sqrt(3)) / 4, (3 - math.sqrt(3)) / 4]], atol=1e-15)
    i1 = i0[::-1, ::-1]  # upper half: both-axes flip
    for c in range(4):
        ox, oy = (i1 if c & 1 else i0), (i1 if c & 2 else i0)
        assert np.allclose(I[c], kron_op([ox, oy]), atol=2e-15), c
    I2 = oracle.operators(2, 2)["interp"][0]
    row0 = np.array([pv["I0_p2_00"], pv["I0_p2_01"], pv["I0_p2_02"]])
    # first row of the x-operator appears in tensor row n = 0 against columns m = 0,1,2 scaled by row0[0] in y
    assert np.allclose(I2[0, :3], row0[0] * row0, atol=2e-15)


@pytest.mark.parametrize("dim,p", [(2, 1), (2, 2), (2, 3), (3, 1), (3, 2), (3, 3)])
def test_operator_identities(dim, p):
    ops = oracle.operators(dim, p)
    nc, N = 1 << dim, (p + 1) ** dim
    z, w = np.polynomial.legendre.leggauss(p + 1)
    I1 = [one_d_interp(p, 0), one_d_interp(p, 1)]
    R1 = [0.5 * np.diag(1 / w) @ I1[b].T @ np.diag(w) for b in (0, 1)]  # reading E-4 closed form
    wt = w
    for _ in range(dim - 1):
        wt = np.kron(w, wt)
    assert np.allclose(ops["mass"], np.diag(wt), atol=1e-14)  # GL collocation: M = diag(w) exactly
    acc = np.zeros((N, N))
    for c in range(nc):
        bits = [(c >> a) & 1 for a in range(dim)]
        assert np.allclose(ops["interp"][c], kron_op([I1[b] for b in bits]), atol=5e-15)
        assert np.allclose(ops["proj"][c], kron_op([R1[b] for b in bits]), atol=1e-14)
        assert np.allclose(ops["interp"][c].sum(axis=1), 1.0, atol=1e-14)       # partition of unity
        assert np.allclose(wt @ ops["proj"][c], wt / nc, atol=1e-14)            # mean conservation
        # S_c = 2^-dim I_c^T W (quadrature of Eq. 13 is exact)
        assert np.allclose(ops["S"][c], (ops["interp"][c].T * wt[None, :]) / nc, atol=1e-14)
        acc += ops["proj"][c] @ ops["interp"][c]
    assert np.allclose(acc, np.eye(N), atol=1e-14)  # refine then coarsen is the identity


def alg7_on_keys(dim, maxl, old, new):
    """Alg. 7 restated on sorted key lists with bisect + Eq. 7."""
    old = [int(k) for k in old]
    src, kind = [], []
    for k in (int(v) for v in new):
        B = bisect.bisect_left(old, k)
        lvl = k & 31
        if B < len(old) and old[B] == k:
            src.append(B); kind.append(0)
        elif B < len(old) and old[B] - k == 1:
            src.append(B); kind.append(2)
        else:
            par = old[B - 1]
            pl = par & 31
            assert pl == lvl - 1
            shift = dim * (maxl - lvl) + 5
            assert (par >> (shift + dim)) == (k >> (shift + dim))  # T_o[B-1] is the parent
            child = (k >> shift) & ((1 << dim) - 1)                # last dim bits of the raw ID
            src.append(B - 1); kind.append(1 | (child << 4))
    return np.array(src, np.int32), np.array(kind, np.uint8)


def sample_poly(cfg, coef, level, xyz):
    """Polynomial of degree <= p per direction, sampled analytically at every leaf's GL nodes."""
    dim, maxl, p = cfg["dim"], cfg["maxl"], cfg["p"]
    P1 = p + 1
    N = P1 ** dim
    z = np.polynomial.legendre.leggauss(P1)[0]
    w = np.ldexp(1.0, (maxl - level.astype(np.int64)))
    L = float(1 << maxl)
    idx = np.arange(N)
    val = np.ones((level.size, N))
    pos = []
    for a in range(dim):
        ia = (idx // P1 ** a) % P1
        pos.append((xyz[:, a].astype(np.float64)[:, None] + 0.5 * w[:, None] * (1.0 + z[ia][None, :])) / L)
    out = np.zeros((level.size, coef.shape[0], N))
    for v in range(coef.shape[0]):
        acc = np.zeros((level.size, N))
        for e in np.ndindex(*([P1] * dim)):
            term = coef[v][e] * np.ones_like(acc)
            for a in range(dim):
                term = term * pos[a] ** e[a]
            acc += term
        out[:, v, :] = acc
    return out


@pytest.mark.parametrize("name,cycles", [("c1", 4), ("c3b", 12)])
def test_polynomial_data_transfers_exactly_and_map_matches_alg7(name, cycles):
    cfg = W.CONFIGS[name]
    dim, p, nvars = cfg["dim"], cfg["p"], cfg["nvars"]
    rng = np.random.default_rng(4)
    coef = rng.uniform(-1, 1, (nvars,) + (p + 1,) * dim)
    t = oracle.Tree(dim, cfg["base"], cfg["maxl"], cfg["periodic"])
    lvl, xyz = t.leaf_boxes()
    u = sample_poly(cfg, coef, lvl, xyz)
    kinds_seen = set()
    for c in range(cycles):
        f = W.flags(cfg, c, torch.from_numpy(lvl), torch.from_numpy(xyz.astype(np.int64))).numpy()
        t.adapt(f)
        t.balance()
        src, kind = t.build_map()
        s2, k2 = alg7_on_keys(dim, cfg["maxl"], t.old_keys(), t.keys())
        assert np.array_equal(src, s2) and np.array_equal(kind, k2)
        kk = kind & 0xF
        kinds_seen |= set(kk.tolist())
        # case counts (SURVEY 8(c) "map"): refine count multiple of nc; every old leaf read exactly once
        assert (kk == 1).sum() % t.nc == 0
        reads = np.zeros(t.old_keys().size, np.int64)
        np.add.at(reads, src[kk == 0], 1)
        np.add.at(reads, src[kk == 1], 1)
        for c2 in range(t.nc):
            np.add.at(reads, src[kk == 2] + c2, 1)
        assert np.all(reads[np.setdiff1d(np.arange(reads.size), src[kk == 1])] == 1)
        assert np.all(reads[src[kk == 1]] == t.nc)
        u = t.transfer(u, p, nvars)
        lvl, xyz = t.leaf_boxes()
        want = sample_poly(cfg, coef, lvl, xyz)
        scale = max(1.0, np.abs(want).max())
        assert np.abs(u - want).max() <= 1e-12 * scale
    assert kinds_seen == {0, 1, 2}


def test_mean_conservation_and_restoration_random_data():
    # config 3: refine 9 times, coarsen 9 times: keys restored, u restored to 1e-12 (BASELINE.json configs[2]);
    # each element's mean (sum_n w_n u_n * volume) is conserved by every transfer
    cfg = W.CONFIGS["c3"]
    dim, p, nvars, maxl = cfg["dim"], cfg["p"], cfg["nvars"], cfg["maxl"]
    t = oracle.Tree(dim, cfg["base"], maxl, cfg["periodic"])
    lvl, xyz = t.leaf_boxes()
    u0 = W.initial_solution(cfg, torch.from_numpy(lvl), torch.from_numpy(xyz.astype(np.int64))).numpy()
    assert u0.shape == (512, nvars, (p + 1) ** dim) and np.abs(u0).max() <= 1.0 and u0.std() > 0.5
    w1 = np.polynomial.legendre.leggauss(p + 1)[1]
    wt = w1
    for _ in range(dim - 1):
        wt = np.kron(w1, wt)

    def integral(u, lv):
        vol = np.ldexp(1.0, dim * (maxl - lv.astype(np.int64)) - dim)  # (w/2)^dim
        return np.einsum("evn,n,e->v", u, wt, vol)

    u = u0
    tot0 = integral(u, lvl)
    for c in range(cfg["cycles"]):
        f = W.flags(cfg, c, torch.from_numpy(lvl), torch.from_numpy(xyz.astype(np.int64))).numpy()
        t.adapt(f)
        t.balance()
        u = t.transfer(u, p, nvars)
        lvl, xyz = t.leaf_boxes()
        assert np.allclose(integral(u, lvl), tot0, rtol=0, atol=1e-9 * np.abs(tot0).max())
    assert t.num_leaves() == 512
    assert np.abs(u - u0).max() <= 1e-12


def test_transfer_without_snapshot_is_identity_and_deferred_balance_is_a_mapping_error():
    cfg = W.CONFIGS["c3b"]
    t = oracle.Tree(3, cfg["base"], cfg["maxl"], cfg["periodic"])
    u = np.random.default_rng(0).uniform(-1, 1, (t.num_leaves(), 2, 8))
    assert np.array_equal(t.transfer(u, 1, 2), u)
    # nine adapts without balance, then one balance: final leaves are > 1 level from the last snapshot
    for c in range(9):
        lvl, xyz = t.leaf_boxes()
        t.adapt(W.flags(cfg, c, torch.from_numpy(lvl), torch.from_numpy(xyz.astype(np.int64))).numpy())
    t.balance()
    with pytest.raises(oracle.OracleError):
        t.build_map()
