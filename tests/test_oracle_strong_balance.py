"""Pins for the oracle's strong 2:1 balance ("any two adjacent octants that share
either an edge or a face must not have tree-depth difference larger than 1"; DESIGN.md reading
C-9: connectivity 1 = faces, 2 = + edges, 3 = + corners; 2-D: 1 = faces, 2 = + corners).

Sources of truth: the set-model Jacobi ripple over offset directions (tests/bruteforce.py, no
Morton IDs, no pointer tree), a purely geometric O(N^2) box-adjacency check that uses no
neighbour keys at all, minimality by brute force, and a constructed case in which leaves are
adjacent ONLY across an edge / a corner, so each connectivity level must change the result.
"""
import numpy as np
import pytest

import bruteforce as bf
import oracle


def cells_of(t):
    lvl, xyz = t.leaf_boxes()
    return bf.to_cells(lvl, xyz, t.dim, t.maxl)


def random_tree(dim, base, maxl, periodic, seed, cycles=4, frac=0.25):
    rng = np.random.default_rng(seed)
    t = oracle.Tree(dim, base, maxl, periodic)
    for _ in range(cycles):
        f = (rng.random(t.num_leaves()) < frac).astype(np.int8)
        t.adapt(f)
        t.drop_snapshot()
    return t


CASES = [(2, 1, 5, (0, 0), 1), (2, 1, 5, (1, 1), 2), (2, 0, 6, (1, 0), 3),
         (3, 1, 4, (0, 0, 0), 4), (3, 1, 4, (1, 1, 1), 5), (3, 0, 4, (0, 1, 0), 6)]


@pytest.mark.parametrize("dim,base,maxl,periodic,seed", CASES)
def test_strong_balance_equals_set_model(dim, base, maxl, periodic, seed):
    for conn in range(1, dim + 1):
        t = random_tree(dim, base, maxl, periodic, seed)
        before = set(cells_of(t))
        it = t.balance(conn)
        want, it_bf, sp_bf = bf.balance(before, periodic, conn)
        got = cells_of(t)
        assert set(got) == want and len(got) == len(want)
        assert it == it_bf and t.last_balance_splits == sp_bf
        # idempotent
        assert t.balance(conn) == 0 and set(cells_of(t)) == want


@pytest.mark.parametrize("dim,base,maxl,periodic,seed", [c for c in CASES if c[2] <= 5])
def test_result_passes_geometric_check_and_is_minimal(dim, base, maxl, periodic, seed):
    for conn in range(1, dim + 1):
        t = random_tree(dim, base, maxl, periodic, seed, cycles=3, frac=0.15)
        before = set(cells_of(t))
        t.balance(conn)
        mesh = set(cells_of(t))
        if len(mesh) > 900:
            pytest.skip("too large for the O(N^2) check")
        assert bf.is_balanced_boxes(mesh, periodic, conn, maxl)
        assert bf.volume(mesh, maxl) == 1 << (dim * maxl)
        # every output leaf descends from (or is) an input leaf
        for c in mesh:
            assert bf.containing_leaf(before, c) is not None
        # minimality: merging any complete sibling group that was not in the input breaks 2:1
        groups = {}
        for c in mesh:
            if c[0] > 0:
                groups.setdefault(bf.parent(c), []).append(c)
        tried = 0
        for par, kids in groups.items():
            if len(kids) != 1 << dim or all(k in before for k in kids):
                continue
            coarser = (mesh - set(kids)) | {par}
            assert not bf.is_balanced_boxes(coarser, periodic, conn, maxl)
            tried += 1
            if tried >= 12:
                break


def diagonal_case(dim, maxl):
    """Refine, level by level, the leaf that touches the domain centre from the all-minus side.
    The leaf diagonally opposite across the centre shares only a corner (2-D) / only an edge or a
    corner (3-D) with it, so face balance never refines that neighbour."""
    t = oracle.Tree(dim, 1, maxl)
    for _ in range(maxl - 1):
        lvl, xyz = t.leaf_boxes()
        half = 1 << (maxl - 1)
        w = 1 << (maxl - lvl.astype(np.int64))
        f = np.all(xyz[:, :dim].astype(np.int64) + w[:, None] == half, axis=1).astype(np.int8)
        assert f.sum() == 1
        t.adapt(f)
        t.drop_snapshot()
    return t


def test_connectivity_levels_differ_2d():
    maxl = 6
    n = []
    for conn in (1, 2):
        t = diagonal_case(2, maxl)
        t.balance(conn)
        mesh = set(cells_of(t))
        assert bf.is_balanced_boxes(mesh, (0, 0), conn, maxl)
        n.append(len(mesh))
        if conn == 1:
            assert not bf.is_balanced_boxes(mesh, (0, 0), 2, maxl)  # face balance leaves a corner jump
        # the leaf touching the centre from the all-plus side: only corner-adjacent to the finest leaf
        opp = bf.containing_leaf(mesh, (maxl, 1 << (maxl - 1), 1 << (maxl - 1)))
        assert opp[0] == (maxl - 1 if conn == 2 else maxl - 2)
    assert n[0] < n[1]


def test_connectivity_levels_differ_3d():
    maxl = 5
    n, meshes = [], []
    for conn in (1, 2, 3):
        t = diagonal_case(3, maxl)
        t.balance(conn)
        mesh = set(cells_of(t))
        assert bf.is_balanced_boxes(mesh, (0, 0, 0), conn, maxl)
        n.append(len(mesh))
        meshes.append(mesh)
        t.connect()  # every strong balance is also a face balance
    assert n[0] < n[1] < n[2]
    assert not bf.is_balanced_boxes(meshes[0], (0, 0, 0), 2, maxl)
    assert not bf.is_balanced_boxes(meshes[1], (0, 0, 0), 3, maxl)
    # the leaf across the (x,y) edge / across the corner from the finest leaf (level maxl): one level
    # coarser once its adjacency counts, two levels coarser when it is reached only through the
    # ripple of the neighbours that do count
    h = 1 << (maxl - 1)
    edge_lv = [bf.containing_leaf(m, (maxl, h, h, h - 1))[0] for m in meshes]
    corner_lv = [bf.containing_leaf(m, (maxl, h, h, h))[0] for m in meshes]
    assert edge_lv == [maxl - 2, maxl - 1, maxl - 1]
    assert corner_lv[2] == maxl - 1 and corner_lv[1] < maxl - 1 and corner_lv[0] <= corner_lv[1]
    # stronger connectivity refines the weaker result
    for weak, strong in ((meshes[0], meshes[1]), (meshes[1], meshes[2])):
        for c in strong:
            assert bf.containing_leaf(weak, c) is not None


def test_bad_connectivity_rejected():
    t = oracle.Tree(2, 1, 3)
    with pytest.raises(oracle.OracleError):
        t.balance(3)
    with pytest.raises(oracle.OracleError):
        t.balance(0)
