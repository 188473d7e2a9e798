"""Pins for the oracle's forest on a brick of root cubes (reading J-1; the paper's 3-D runs
use a slab of 16 x 16 x 1 cubes, one element thick at D_min = 4, while its linear trees
cover "perfect cubes" only).

Sources of truth: the single-cube oracle (a 1 x 1 (x 1) brick must reproduce it bit for bit), closed
forms for uniform bricks, the independent set model of tests/bruteforce.py with per-axis extents
(adapt, Jacobi ripple with sweep and split counts, face census), brute-force O(N^2) box adjacency
across cube boundaries and periodic images, volume tiling, the one-cell-thick periodic axis of reading
D-6, polynomial data through the transfer, and an exactly differentiable state whose right-hand side
depends on the element width dx = width / (nroot * 2^level).
"""
import numpy as np
import pytest

import bruteforce as bf
import oracle
from test_oracle_mortar import face_points, volume_points
from test_oracle_fr import G

BRICKS = [(2, (3, 2), (0, 0)), (2, (2, 3), (1, 0)), (2, (4, 1), (1, 1)),
          (3, (2, 1, 3), (0, 1, 0)), (3, (3, 3, 1), (1, 1, 1)), (3, (1, 2, 2), (0, 0, 0))]


def cells_of(t):
    lvl, xyz = t.leaf_boxes()
    return bf.to_cells(lvl, xyz, t.dim, t.maxl)


def random_cycles(t, rng, ncycles, nroot, periodic, check=True):
    """adapt + balance on both the oracle and the set model, compared after every call"""
    mesh = set(cells_of(t))
    for c in range(ncycles):
        cells = cells_of(t)
        f = rng.choice(np.array([-1, 0, 1], np.int8), len(cells), p=[0.3, 0.4, 0.3] if c % 2 else [0.1, 0.5, 0.4])
        t.adapt(f)
        mesh = bf.adapt(mesh, dict(zip(cells, f.tolist())), t.base, t.maxl)
        if check:
            assert set(cells_of(t)) == mesh, "adapt, cycle %d" % c
        it = t.balance()
        mesh, it_m, sp_m = bf.balance(mesh, periodic, 1, nroot)
        if check:
            assert set(cells_of(t)) == mesh and it == it_m and t.last_balance_splits == sp_m, "balance, cycle %d" % c
        t.drop_snapshot()
    return mesh


# ---------------------------------------------------------------- keys
@pytest.mark.parametrize("dim,base,maxl,per", [(2, 2, 5, (1, 0)), (3, 1, 4, (0, 1, 1))])
def test_one_cube_brick_is_the_single_tree(dim, base, maxl, per):
    a = oracle.Tree(dim, base, maxl, per)
    b = oracle.Tree(dim, base, maxl, per, nroot=(1,) * dim)
    rng = np.random.default_rng(dim)
    for c in range(3):
        assert np.array_equal(a.keys(), b.keys())
        Fa, Fb = a.connect(), b.connect()
        for k in Fa:
            assert np.array_equal(Fa[k], Fb[k]), k
        f = rng.integers(-1, 2, a.num_leaves()).astype(np.int8)
        a.adapt(f); b.adapt(f)
        assert a.balance() == b.balance()
        a.drop_snapshot(); b.drop_snapshot()


@pytest.mark.parametrize("dim,nroot,per", BRICKS)
def test_forest_keys_are_cube_major_morton_ids(dim, nroot, per):
    base, maxl = 1, 3
    t = oracle.Tree(dim, base, maxl, per, nroot=nroot)
    lvl, xyz = t.leaf_boxes()
    keys = t.keys()
    assert np.all(np.diff(keys.astype(np.int64)) > 0)
    ntrees = int(np.prod(nroot))
    assert t.num_leaves() == ntrees << (dim * base)
    mask = (1 << maxl) - 1
    for i in range(t.num_leaves()):
        r, mul = 0, 1
        for a in range(dim):
            r += (int(xyz[i, a]) >> maxl) * mul
            mul *= nroot[a]
        rel = np.array([int(v) & mask for v in xyz[i]], np.uint32)
        # the paper's ID of the octant inside its cube (Alg. 1) with the cube index above the path bits
        assert int(keys[i]) == oracle.encode(dim, maxl, int(lvl[i]), rel) | (r << (dim * maxl + 5))
    # cube-major: all leaves of cube r precede those of cube r + 1
    cube = keys >> np.uint64(dim * maxl + 5)
    assert np.all(np.diff(cube.astype(np.int64)) >= 0) and int(cube[-1]) == ntrees - 1
    assert t.dfs_is_sorted()


# ---------------------------------------------------------------- closed forms on uniform bricks
@pytest.mark.parametrize("dim,nroot,per", BRICKS)
@pytest.mark.parametrize("base", [0, 2])
def test_uniform_brick_face_counts(dim, nroot, per, base):
    t = oracle.Tree(dim, base, 3, per, nroot=nroot)
    N = [nroot[a] << base for a in range(dim)]
    M = int(np.prod(N))
    assert t.num_leaves() == M
    F = t.connect()
    conf = bnd = 0
    for a in range(dim):
        others = M // N[a]
        if per[a]:
            conf += N[a] * others          # also for N[a] == 1: a leaf is its own neighbour (reading D-6)
        else:
            conf += (N[a] - 1) * others
            bnd += 2 * others
    assert (F["n_conf"], F["n_hang"], F["n_bnd"]) == (conf, 0, bnd)
    assert t.balance() == 0
    Fb = t.connect(1)                       # brute force O(N^2)
    for k in F:
        assert np.array_equal(F[k], Fb[k]), k


def test_one_cell_thick_periodic_slab():
    """The paper's slab in miniature: 4 x 4 x 1 cubes, periodic in all directions, one
    element thick: every leaf is its own z-neighbour (reading D-6)."""
    t = oracle.Tree(3, 0, 2, (1, 1, 1), nroot=(4, 4, 1))
    F = t.connect()
    nbr, kind = F["nbr"].reshape(-1, 6), F["kind"].reshape(-1, 6)
    assert np.all(kind == 1) and np.array_equal(nbr[:, 4], np.arange(16)) and np.array_equal(nbr[:, 5], np.arange(16))
    sel = F["conf_axis"] == 2
    assert np.array_equal(F["conf"][sel][:, 0], F["conf"][sel][:, 1])
    # refine one cube: its z-faces now meet its own children across the periodic boundary
    f = np.zeros(16, np.int8); f[5] = 1
    t.adapt(f)
    assert t.balance() == 0
    F = t.connect()
    Fb = t.connect(1)
    for k in F:
        assert np.array_equal(F[k], Fb[k]), k
    # by hand: coarse-coarse faces 14 (x: 16 minus the 2 that became hanging) + 14 (y) + 15 (z: every
    # remaining cube meets itself); inside the refined cube 4 + 4 + 4 internal faces and 4 more where its
    # upper children meet its lower children across the periodic z boundary; hanging: 2 * 4 in x, 2 * 4 in y
    assert (F["n_conf"], F["n_hang"], F["n_bnd"]) == (14 + 14 + 15 + 12 + 4, 16, 0)


# ---------------------------------------------------------------- adapt / balance / connect vs the set model
@pytest.mark.parametrize("dim,nroot,per", BRICKS)
def test_cycles_match_set_model_and_bruteforce_adjacency(dim, nroot, per):
    base, maxl = (1, 4) if dim == 2 else (0, 3)
    t = oracle.Tree(dim, base, maxl, per, nroot=nroot)
    rng = np.random.default_rng(17 + dim + sum(nroot))
    mesh = random_cycles(t, rng, 4, nroot, per)
    assert bf.is_balanced(mesh, per, nroot)
    # volume tiling: the leaves fill ntrees cubes exactly
    assert bf.volume(mesh, maxl) == int(np.prod(nroot)) << (dim * maxl)
    F = t.connect()
    Fb = t.connect(1)
    for k in F:
        assert np.array_equal(F[k], Fb[k]), k
    assert (F["n_conf"], F["n_hang"], F["n_bnd"]) == bf.face_census(mesh, per, nroot)
    nbr, kind = F["nbr"].reshape(-1, t.nf), F["kind"].reshape(-1, t.nf)
    M = t.num_leaves()
    assert t.nf * M == 2 * F["n_conf"] + F["n_hang"] + F["n_hang"] // (1 << (dim - 1)) + F["n_bnd"]
    for e in range(M):                       # reciprocity of conforming faces
        for f in range(t.nf):
            if kind[e, f] == 1:
                assert kind[nbr[e, f], f ^ 1] == 1 and nbr[nbr[e, f], f ^ 1] == e


def test_ripple_crosses_cube_boundaries():
    """Refine towards a corner shared by four cubes: the 2:1 ripple has to run through all of them."""
    nroot, per = (2, 2), (0, 0)
    t = oracle.Tree(2, 1, 6, per, nroot=nroot)
    mesh = set(cells_of(t))
    total = 0
    for c in range(5):
        cells = cells_of(t)
        lvl, xyz = t.leaf_boxes()
        w = 1 << (6 - lvl.astype(np.int64))
        f = ((xyz[:, 0] + w == 64) & (xyz[:, 1] + w == 64)).astype(np.int8)   # the leaf below-left of (1, 1)
        assert f.sum() == 1
        t.adapt(f)
        mesh = bf.adapt(mesh, dict(zip(cells, f.tolist())), 1, 6)
        it = t.balance()
        mesh, it_m, sp = bf.balance(mesh, per, 1, nroot)
        assert it == it_m and set(cells_of(t)) == mesh
        total += sp
        t.drop_snapshot()
    assert total > 0
    other = [c for c in mesh if c[1] >= (1 << c[0]) and c[2] >= (1 << c[0]) and c[0] > 1]
    assert other, "the ripple must have refined the diagonal cube too"


# ---------------------------------------------------------------- transfer and FR on a brick
def _poly(X, p, dim):
    v = np.ones(X.shape[:-1])
    for a in range(dim):
        v = v * sum((0.4 - 0.1 * a + 0.3 * k) * X[..., a] ** k for k in range(p + 1))
    return v


@pytest.mark.parametrize("dim,nroot,per", [(2, (3, 2), (0, 0)), (3, (2, 1, 2), (0, 0, 0))])
@pytest.mark.parametrize("p", [1, 3])
def test_polynomial_data_transfers_exactly_on_a_brick(dim, nroot, per, p):
    t = oracle.Tree(dim, 1, 4, per, nroot=nroot)
    rng = np.random.default_rng(p)
    u = np.stack([_poly(volume_points(t, p), p, dim), 2.0 - _poly(volume_points(t, p), p, dim)], axis=1)
    seen = set()
    for c in range(3):
        # two refining cycles, then coarsen every complete group above the base level
        f = rng.choice(np.array([0, 1], np.int8), t.num_leaves()) if c < 2 else np.full(t.num_leaves(), -1, np.int8)
        t.adapt(f)
        t.balance()
        src, kind = t.build_map()
        seen |= set((kind & 15).tolist())
        u = t.transfer(u, p, 2)
        want = _poly(volume_points(t, p), p, dim)
        assert np.max(np.abs(u[:, 0] - want)) < 1e-11 * np.max(np.abs(want))
        assert np.max(np.abs(u[:, 1] - (2.0 - want))) < 1e-11 * np.max(np.abs(want))
    assert seen == {0, 1, 2}


@pytest.mark.parametrize("dim,nroot", [(2, (3, 1)), (3, (1, 2, 1))])
def test_rhs_on_a_brick_uses_the_cube_width(dim, nroot):
    """Constant density and velocity, polynomial pressure (as in test_oracle_fr): R is known in closed
    form and is proportional to 1/dx, dx = width_a / (nroot_a * 2^level): a wrong element width on the
    long axis of the brick fails.  Cube width 0.5, so the brick is nroot/2 wide."""
    p = 2
    per = (0,) * dim
    h = 0.5
    t = oracle.Tree(dim, 1, 3, per, nroot=nroot)
    rng = np.random.default_rng(3)
    for _ in range(2):
        t.adapt((rng.random(t.num_leaves()) < 0.3).astype(np.int8)); t.balance(); t.drop_snapshot()
    F = t.connect()
    kind = F["kind"].reshape(-1, t.nf) & 15
    assert (kind == 2).any()
    X, XF = h * volume_points(t, p), h * face_points(t, p, wrap=False)
    v0 = np.array([0.6, -0.35, 0.45][:dim])
    rho0 = 1.3
    pr_of = lambda Xp: 2.5 + sum((0.3 - 0.07 * a) * Xp[..., a] + 0.11 * Xp[..., a] ** 2 for a in range(dim))
    grad = lambda Xp: np.stack([(0.3 - 0.07 * a) + 0.22 * Xp[..., a] for a in range(dim)], axis=-1)

    def state(pr):
        U = np.empty(pr.shape + (dim + 2,))
        U[..., 0] = rho0
        U[..., 1:1 + dim] = rho0 * v0
        U[..., dim + 1] = pr / (G - 1) + 0.5 * rho0 * (v0 @ v0)
        return U
    nv = dim + 2
    u = np.moveaxis(state(pr_of(X)), -1, 1)
    uf = t.face_interp(u, p, nv)
    unb = t.mortar_project(uf, p, nv)
    fs = t.common_flux(uf, unb, p)
    g = t.mortar_gather(fs, p, nv)
    fs = np.where(np.isnan(fs), g, fs)
    prF = pr_of(XF)
    for f in range(t.nf):
        a = f >> 1
        ex = np.zeros((t.num_leaves(), nv, prF.shape[-1]))
        ex[:, 0] = rho0 * v0[a]
        for b in range(dim):
            ex[:, 1 + b] = rho0 * v0[b] * v0[a] + (prF[:, f] if b == a else 0.0)
        ex[:, dim + 1] = (G / (G - 1) * prF[:, f] + 0.5 * rho0 * (v0 @ v0)) * v0[a]
        bsel = kind[:, f] == 0
        fs[bsel, f] = ex[bsel]
    R = t.fr_rhs(u, fs, p, [h * n for n in nroot])
    gp = grad(X)
    want = np.stack([np.zeros(gp.shape[:2])] + [-gp[..., b] for b in range(dim)] + [-(G / (G - 1)) * (gp @ v0)], axis=1)
    assert np.max(np.abs(R - want)) < 1e-9 * max(1.0, np.max(np.abs(want)))


def test_bad_bricks_are_rejected():
    with pytest.raises(oracle.OracleError):
        oracle.Tree(2, 0, 3, (0, 0), nroot=(0, 2))
    with pytest.raises(oracle.OracleError):
        oracle.Tree(3, 0, 19, (0, 0, 0), nroot=(2, 2, 1))     # 57 path bits + 5 depth bits + 2 cube bits > 63
