"""Pins for the oracle's adapt (Alg. 6), 2:1 balance (Alg. 4) and connectivity (Alg. 5).

Sources of truth: the independent [survey-calc] censuses (tests/golden/survey_calc_*.txt),
a set-based brute-force model (tests/bruteforce.py), closed-form face counts of uniform
meshes, the paper's worked example and structural invariants.
"""
import os

import numpy as np
import pytest
import torch

import bruteforce as bf
import oracle
from paper_2306_06744_b200 import workloads as W

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def load_table(name):
    rows, extra = [], {}
    for line in open(os.path.join(GOLD, name)):
        s = line.strip()
        if s.startswith("# deferred_"):
            tok = s[2:].split()
            extra.update({tok[i]: int(tok[i + 1]) for i in range(0, len(tok), 2)})
        if not s or s.startswith("#"):
            continue
        rows.append([int(v) for v in s.split()])
    return rows, extra


def flags_for(cfg, cycle, t):
    lvl, xyz = t.leaf_boxes()
    return W.flags(cfg, cycle, torch.from_numpy(lvl), torch.from_numpy(xyz.astype(np.int64))).numpy()


def new_tree(cfg):
    return oracle.Tree(cfg["dim"], cfg["base"], cfg["maxl"], cfg["periodic"])


def volume_ok(t):
    lvl, _ = t.leaf_boxes()
    vol = sum(1 << (t.dim * (t.maxl - int(l))) for l in lvl) if lvl.size < 5000 else \
        int(np.sum(np.ldexp(1.0, t.dim * (t.maxl - lvl.astype(np.int64)))))
    return vol == 1 << (t.dim * t.maxl)


# ---------------------------------------------------------------- golden censuses
def test_config1_deterministic_census():
    cfg = dict(W.CONFIGS["c1"], rand_refine=0.0)
    rows, _ = load_table("survey_calc_c1_deterministic.txt")
    t = new_tree(cfg)
    for c, out, iters, splits, n_conf, n_hang, n_bnd in rows:
        t.adapt(flags_for(cfg, c, t))
        assert t.balance() == iters
        assert t.last_balance_splits == splits
        assert t.num_leaves() == out
        F = t.connect()
        assert (F["n_conf"], F["n_hang"], F["n_bnd"]) == (n_conf, n_hang, n_bnd)
        t.drop_snapshot()


@pytest.mark.parametrize("name", ["c3", "c3b"])
def test_config3_ripple_census(name):
    cfg = W.CONFIGS[name]
    rows, extra = load_table("survey_calc_%s.txt" % name)
    t = new_tree(cfg)
    k0 = t.keys()
    for row in rows:
        c, out, iters = row[0], row[1], row[2]
        t.adapt(flags_for(cfg, c, t))
        assert t.balance() == iters
        if name == "c3b":
            assert t.last_balance_splits == row[3]
        assert t.num_leaves() == out
        want_faces = row[-3:]
        if want_faces[0] >= 0:
            F = t.connect()
            assert [F["n_conf"], F["n_hang"], F["n_bnd"]] == want_faces
        assert volume_ok(t)
        t.drop_snapshot()
    assert np.array_equal(t.keys(), k0)  # coarsen-everything restores the original key array
    if name == "c3b":
        # deferred balance: nine adapts, then ONE balance (reading C-2: same final tree)
        a = new_tree(cfg)
        b = new_tree(cfg)
        for c in range(9):
            a.adapt(flags_for(cfg, c, a))
            a.balance()
            b.adapt(flags_for(cfg, c, b))
        assert b.num_leaves() == extra["deferred_leaves_before"]
        assert b.balance() == extra["deferred_iters"]
        assert b.last_balance_splits == extra["deferred_splits"]
        assert b.num_leaves() == extra["deferred_leaves_after"]
        assert np.array_equal(a.keys(), b.keys())


def test_config2_census_first_cycles():
    cfg = W.CONFIGS["c2"]
    rows, _ = load_table("survey_calc_c2.txt")
    want = {r[0]: r for r in rows}
    t = new_tree(cfg)
    for c in range(6):
        f = flags_for(cfg, c, t)
        lvl, _ = t.leaf_boxes()
        m_in = t.num_leaves()
        n_ref = int(((f > 0) & (lvl < cfg["maxl"])).sum())
        t.adapt(f)
        after = t.num_leaves()
        groups = n_ref - (after - m_in) // 3  # Ma = M0 + (nc-1)(refined - groups), nc-1 = 3
        iters = t.balance()
        F = t.connect()
        got = [c, m_in, n_ref, groups, after, iters, t.last_balance_splits, t.num_leaves(), F["n_conf"], F["n_hang"]]
        assert got == want[c]
        assert F["n_bnd"] == 0
        t.drop_snapshot()


def test_config4_census_first_cycles():
    cfg = W.CONFIGS["c4"]
    rows, _ = load_table("survey_calc_c4.txt")
    t = new_tree(cfg)
    for c, out, iters, splits, n_conf, n_hang in rows[:3]:
        t.adapt(flags_for(cfg, c, t))
        assert t.balance() == iters
        assert t.last_balance_splits == splits
        assert t.num_leaves() == out
        t.drop_snapshot()


# ---------------------------------------------------------------- brute-force model
def random_cycle_compare(dim, base, maxl, periodic, seed, cycles):
    rng = np.random.default_rng(seed)
    t = oracle.Tree(dim, base, maxl, periodic)
    mesh = bf.uniform(dim, base)
    for c in range(cycles):
        lvl, xyz = t.leaf_boxes()
        cells = bf.to_cells(lvl, xyz, dim, maxl)
        assert set(cells) == mesh and len(cells) == len(mesh)
        f = rng.choice([-1, -1, 0, 1], size=len(cells)).astype(np.int8)
        flag_of = {cell: int(fl) for cell, fl in zip(cells, f)}
        t.adapt(f)
        mesh = bf.adapt(mesh, flag_of, base, maxl)
        lvl, xyz = t.leaf_boxes()
        assert set(bf.to_cells(lvl, xyz, dim, maxl)) == mesh
        assert bf.volume(mesh, maxl) == 1 << (dim * maxl)
        iters = t.balance()
        mesh, bi, bs = bf.balance(mesh, periodic)
        assert (iters, t.last_balance_splits) == (bi, bs)
        lvl, xyz = t.leaf_boxes()
        assert set(bf.to_cells(lvl, xyz, dim, maxl)) == mesh
        assert bf.is_balanced(mesh, periodic)
        F = t.connect()
        assert (F["n_conf"], F["n_hang"], F["n_bnd"]) == bf.face_census(mesh, periodic)
        t.drop_snapshot()
    return t


@pytest.mark.parametrize("dim,base,maxl,periodic", [
    (2, 2, 6, (0, 0)), (2, 1, 5, (1, 1)), (2, 2, 5, (1, 0)), (3, 1, 4, (0, 0, 0)), (3, 1, 3, (1, 1, 1)),
])
def test_random_cycles_vs_set_model(dim, base, maxl, periodic):
    random_cycle_compare(dim, base, maxl, periodic, seed=dim * 10 + base, cycles=5)


def test_adapt_rules_small():
    # mixed flags in a group: not coarsened, refine flags honoured (reading B-3);
    # flags at the limits ignored (B-2); count identity Ma = M0 + (nc-1)(#ref - #groups)
    t = oracle.Tree(2, 1, 2)
    assert t.num_leaves() == 4
    t.adapt(np.array([1, 0, 0, 0], np.int8))  # 7 leaves: 4 children at level 2 (= max) + 3
    assert t.num_leaves() == 7
    k = t.keys()
    lvl, _ = t.leaf_boxes()
    assert list(lvl) == [2, 2, 2, 2, 1, 1, 1]
    # refine flags at max level ignored; coarsen at base ignored; mixed group stays
    t.adapt(np.array([1, -1, -1, -1, -1, -1, -1], np.int8))
    assert np.array_equal(t.keys(), k)
    # complete group, all flagged -> parent
    t.adapt(np.array([-1, -1, -1, -1, 0, 0, 1], np.int8))
    lvl, _ = t.leaf_boxes()
    assert list(lvl) == [1, 1, 1, 2, 2, 2, 2]
    # refine-all then coarsen-all restores the key array bit-exactly
    t = oracle.Tree(3, 1, 4, (1, 1, 1))
    k0 = t.keys()
    t.adapt(np.ones(t.num_leaves(), np.int8))
    assert t.num_leaves() == 8 * k0.size
    t.adapt(-np.ones(t.num_leaves(), np.int8))
    assert np.array_equal(t.keys(), k0)


def test_balance_properties_and_minimality():
    rng = np.random.default_rng(21)
    dim, base, maxl, periodic = 2, 1, 6, (0, 1)
    t = oracle.Tree(dim, base, maxl, periodic)
    # several unbalanced refinements, no balance in between
    for _ in range(4):
        f = (rng.random(t.num_leaves()) < 0.25).astype(np.int8)
        t.adapt(f)
    lvl, xyz = t.leaf_boxes()
    before = set(bf.to_cells(lvl, xyz, dim, maxl))
    iters = t.balance()
    assert iters > 0
    lvl, xyz = t.leaf_boxes()
    after = set(bf.to_cells(lvl, xyz, dim, maxl))
    assert bf.is_balanced(after, periodic) and bf.volume(after, maxl) == 1 << (dim * maxl)
    # every output leaf is a descendant-or-equal of an input leaf
    for cell in after:
        assert bf.containing_leaf(before, cell) is not None
    # idempotent (reading C-7)
    k = t.keys()
    assert t.balance() == 0 and np.array_equal(t.keys(), k)
    # minimality: merging any complete sibling group that was not already in the input breaks 2:1
    seen = set()
    n_checked = 0
    for cell in after:
        if cell[0] == 0:
            continue
        par = bf.parent(cell)
        if par in seen:
            continue
        seen.add(par)
        sib = bf.children(par)
        if not all(s in after for s in sib) or all(s in before for s in sib):
            continue
        trial = (after - set(sib)) | {par}
        assert not bf.is_balanced(trial, periodic)
        n_checked += 1
    assert n_checked > 0


# ---------------------------------------------------------------- connectivity
@pytest.mark.parametrize("dim,level", [(2, 3), (3, 2)])
def test_uniform_mesh_face_counts(dim, level):
    n = 1 << level
    M = n ** dim
    t = oracle.Tree(dim, level, level + 2, [1] * dim)
    F = t.connect()
    assert (F["n_conf"], F["n_hang"], F["n_bnd"]) == (dim * M, 0, 0)
    t = oracle.Tree(dim, level, level + 2, [0] * dim)
    F = t.connect()
    assert (F["n_conf"], F["n_hang"], F["n_bnd"]) == (dim * n ** (dim - 1) * (n - 1), 0, 2 * dim * n ** (dim - 1))


def check_face_invariants(t, F):
    dim, nf, M = t.dim, t.nf, t.num_leaves()
    nbr = F["nbr"].reshape(M, nf)
    kind = F["kind"].reshape(M, nf)
    k = kind & 0xF
    slot = kind >> 4
    half = 1 << (dim - 1)
    # slot equation of SURVEY 8(c): nf*M = 2 n_conf + n_hang (1 + 2^-(dim-1)) + n_bnd
    assert nf * M * half == 2 * F["n_conf"] * half + F["n_hang"] * (half + 1) + F["n_bnd"] * half
    assert (k == 0).sum() == F["n_bnd"] and (k == 2).sum() == F["n_hang"] and (k == 1).sum() == 2 * F["n_conf"]
    assert (k == 3).sum() * half == F["n_hang"]
    lvl, _ = t.leaf_boxes()
    for e in range(M):
        for f in range(nf):
            if k[e, f] == 0:
                assert nbr[e, f] == -1
            elif k[e, f] == 1:  # reciprocated by (nbr, f^1)
                g = nbr[e, f]
                assert k[g, f ^ 1] == 1 and nbr[g, f ^ 1] == e and lvl[g] == lvl[e]
            elif k[e, f] == 2:
                g = nbr[e, f]
                assert k[g, f ^ 1] == 3 and lvl[g] == lvl[e] - 1
            else:
                g = nbr[e, f]
                assert k[g, f ^ 1] == 2 and slot[g, f ^ 1] == 0 and nbr[g, f ^ 1] == e
    # every kind-3 slot is pointed at by exactly 2^(dim-1) kind-2 slots with distinct slot numbers
    fine = {}
    for e in range(M):
        for f in range(nf):
            if k[e, f] == 2:
                fine.setdefault((int(nbr[e, f]), f ^ 1), []).append(int(slot[e, f]))
    assert len(fine) == (k == 3).sum()
    for (g, f), slots in fine.items():
        assert k[g, f] == 3 and sorted(slots) == list(range(half))
    # tables are the canonical emission order of the slots (reading D-4)
    conf = [(e, int(nbr[e, f]), f >> 1) for e in range(M) for f in range(nf) if k[e, f] == 1 and (f & 1)]
    assert [tuple(r) for r in np.column_stack([F["conf"], F["conf_axis"]]).tolist()] == conf
    hang = [(e, int(nbr[e, f]), f | (int(slot[e, f]) << 3)) for e in range(M) for f in range(nf) if k[e, f] == 2]
    assert [tuple(r) for r in np.column_stack([F["hang"], F["hang_info"]]).tolist()] == hang
    bnd = [(e, f) for e in range(M) for f in range(nf) if k[e, f] == 0]
    assert list(zip(F["bnd"].tolist(), F["bnd_face"].tolist())) == bnd


@pytest.mark.parametrize("dim,base,maxl,periodic", [
    (2, 2, 6, (0, 0)), (2, 2, 6, (1, 1)), (3, 1, 4, (0, 1, 0)), (3, 2, 4, (1, 1, 1)),
])
def test_descent_equals_bruteforce_and_invariants(dim, base, maxl, periodic):
    t = random_cycle_compare(dim, base, maxl, periodic, seed=99, cycles=3)
    A = t.connect(method=0)
    B = t.connect(method=1)
    for key in A:
        assert np.array_equal(A[key], B[key]), key
    check_face_invariants(t, A)


def test_worked_example_fig5():
    # in a quadtree the children with raw low bits 0 and 2 share Face 0 of
    # their parent's -x neighbour (child 0 is the first contributor, child 2 the second);
    # children 0 and 1 share Face 2 towards the -y neighbour.  Face numbering reading D-1.
    t = oracle.Tree(2, 1, 3)            # 2x2 base: leaves 0:(0,0) 1:(1,0) 2:(0,1) 3:(1,1)
    t.adapt(np.array([0, 0, 0, 1], np.int8))   # refine the (+x,+y) cell -> leaves 3..6 are its children 0..3
    F = t.connect()
    nbr = F["nbr"].reshape(-1, 4)
    kind = F["kind"].reshape(-1, 4)
    c0, c1, c2, c3 = 3, 4, 5, 6
    # Face 0 (-x) of children 0 and 2 meets coarse leaf 2 = (0,1); slots 0 and 1
    assert (nbr[c0, 0], kind[c0, 0]) == (2, 2 | (0 << 4))
    assert (nbr[c2, 0], kind[c2, 0]) == (2, 2 | (1 << 4))
    # Face 2 (-y) of children 0 and 1 meets coarse leaf 1 = (1,0); slots 0 and 1
    assert (nbr[c0, 2], kind[c0, 2]) == (1, 2 | (0 << 4))
    assert (nbr[c1, 2], kind[c1, 2]) == (1, 2 | (1 << 4))
    # the coarse side: Face 1 (+x) of leaf 2 is 'finer', pointing at the first contributor
    assert (nbr[2, 1], kind[2, 1]) == (c0, 3)
    assert (nbr[1, 3], kind[1, 3]) == (c0, 3)
    # siblings are conforming with each other: child 0 +x -> child 1, +y -> child 2
    assert (nbr[c0, 1], kind[c0, 1]) == (c1, 1) and (nbr[c0, 3], kind[c0, 3]) == (c2, 1)
    assert (nbr[c3, 0], kind[c3, 0]) == (c2, 1) and (nbr[c3, 2], kind[c3, 2]) == (c1, 1)
    # domain boundary on +x/+y of child 3
    assert kind[c3, 1] == 0 and kind[c3, 3] == 0 and nbr[c3, 1] == -1
    assert list(map(tuple, F["hang"])) == [(3, 2), (3, 1), (4, 1), (5, 2)]
    assert list(F["hang_info"]) == [0 | 0, 2 | 0, 2 | (1 << 3), 0 | (1 << 3)]


def test_periodic_thin_domains():
    # reading D-6: one cell wide -> a leaf is its own neighbour; two cells wide -> both faces
    # meet the same neighbour
    t = oracle.Tree(2, 0, 2, (1, 1))
    F = t.connect()
    assert F["nbr"].tolist() == [0, 0, 0, 0] and F["kind"].tolist() == [1, 1, 1, 1]
    assert F["conf"].tolist() == [[0, 0], [0, 0]] and F["conf_axis"].tolist() == [0, 1]
    t = oracle.Tree(2, 1, 2, (1, 0))
    F = t.connect()
    nbr = F["nbr"].reshape(4, 4)
    assert nbr[0, 0] == 1 and nbr[0, 1] == 1 and nbr[1, 0] == 0 and nbr[1, 1] == 0
    assert F["n_conf"] == 4 + 2 and F["n_bnd"] == 4


def test_unbalanced_connect_is_an_error():
    t = oracle.Tree(2, 1, 4)
    t.adapt(np.array([1, 0, 0, 0], np.int8))
    f = np.zeros(t.num_leaves(), np.int8)
    f[3] = 1  # child 3 of leaf 0 touches leaves 1 and 2 -> level jump 2
    t.adapt(f)
    with pytest.raises(oracle.OracleError):
        t.connect()
    assert t.balance() == 1
    t.connect()
