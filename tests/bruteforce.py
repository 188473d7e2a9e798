"""Set-based brute-force model of the tree operations, for pinning the oracle on tiny inputs.

Independent of oracle/lto.cpp in form: no pointer tree, no Morton IDs, no descent.  A mesh
is a Python set of cells ``(level, ix, iy[, iz])`` with integer coordinates in units of the
cell's OWN level; neighbours are found by testing set membership of a cell and its
ancestors; balance is the Jacobi ripple of SURVEY 8(c) written on sets.  Only usable for a
few thousand cells.
"""
from itertools import product


def uniform(dim, level, nroot=None):
    """nroot: the domain is a brick of nroot[a] root cubes along axis a (cells of level l then have
    coordinates in [0, nroot[a] << l)); None = one cube."""
    nr = nroot or (1,) * dim
    return {(level,) + c for c in product(*[range(nr[a] << level) for a in range(dim)])}


def children(cell):
    l, c = cell[0], cell[1:]
    return [(l + 1,) + tuple(2 * ci + b for ci, b in zip(c, bits))
            for bits in product((0, 1), repeat=len(c))]


def parent(cell):
    return (cell[0] - 1,) + tuple(ci >> 1 for ci in cell[1:])


def containing_leaf(mesh, cell):
    """The leaf equal to `cell` or an ancestor of it, else None (cell is refined or outside)."""
    while cell[0] >= 0:
        if cell in mesh:
            return cell
        if cell[0] == 0:
            return None
        cell = parent(cell)
    return None


def face_neighbour(cell, axis, sign, periodic, nroot=None):
    l, c = cell[0], list(cell[1:])
    c[axis] += sign
    n = (nroot[axis] if nroot else 1) << l
    if c[axis] < 0 or c[axis] >= n:
        if not periodic[axis]:
            return None
        c[axis] %= n
    return (l,) + tuple(c)


def adapt(mesh, flag_of, base, maxl):
    """flag_of: dict cell -> -1/0/+1.  One level per call (Alg. 6)."""
    out = set(mesh)
    for cell in mesh:
        if flag_of.get(cell, 0) > 0 and cell[0] < maxl:
            out.discard(cell)
            out.update(children(cell))
    seen = set()
    for cell in mesh:
        if cell[0] <= base:
            continue
        par = parent(cell)
        if par in seen:
            continue
        seen.add(par)
        sib = children(par)
        if all(s in mesh and flag_of.get(s, 0) < 0 for s in sib):
            for s in sib:
                out.discard(s)
            out.add(par)
    return out


def offset_neighbour(cell, offs, periodic, nroot=None):
    """Same-level cell at integer offset `offs` (one entry per axis), periodic wrap per axis."""
    l, c = cell[0], list(cell[1:])
    for a, o in enumerate(offs):
        n = (nroot[a] if nroot else 1) << l
        c[a] += o
        if c[a] < 0 or c[a] >= n:
            if not periodic[a]:
                return None
            c[a] %= n
    return (l,) + tuple(c)


def directions(dim, conn):
    """Offsets with between 1 and `conn` non-zero entries: faces, + edges, + corners."""
    return [o for o in product((-1, 0, 1), repeat=dim) if 1 <= sum(1 for v in o if v) <= conn]


def balance(mesh, periodic, conn=1, nroot=None):
    """Jacobi ripple; returns (mesh, iters, splits).  conn: see directions()."""
    mesh = set(mesh)
    dim = len(next(iter(mesh))) - 1
    dirs = directions(dim, conn)
    iters = splits = 0
    while True:
        marked = set()
        for cell in mesh:
            for o in dirs:
                    nb = offset_neighbour(cell, o, periodic, nroot)
                    if nb is None:
                        continue
                    leaf = containing_leaf(mesh, nb)
                    if leaf is not None and leaf[0] < cell[0] - 1:
                        marked.add(leaf)
        if not marked:
            return mesh, iters, splits
        for m in marked:
            mesh.discard(m)
            mesh.update(children(m))
        iters += 1
        splits += len(marked)


def is_balanced(mesh, periodic, nroot=None):
    dim = len(next(iter(mesh))) - 1
    for cell in mesh:
        for axis in range(dim):
            for sign in (-1, 1):
                nb = face_neighbour(cell, axis, sign, periodic, nroot)
                if nb is None:
                    continue
                leaf = containing_leaf(mesh, nb)
                if leaf is not None and leaf[0] < cell[0] - 1:
                    return False
    return True


def is_balanced_boxes(mesh, periodic, conn, maxl):
    """Geometric 2:1 check with no neighbour keys at all: two leaves are adjacent when their
    closed boxes (any periodic image) touch in a set of dimension >= dim - conn, i.e. on every
    axis the intervals overlap or touch, and they touch on between 1 and conn axes.  O(N^2)."""
    cells = sorted(mesh)
    dim = len(cells[0]) - 1
    L = 1 << maxl
    boxes = []
    for c in cells:
        w = 1 << (maxl - c[0])
        boxes.append((c[0], [ci * w for ci in c[1:]], w))
    for i, (la, xa, wa) in enumerate(boxes):
        for lb, xb, wb in boxes[i + 1:]:
            if abs(la - lb) < 2:
                continue
            shifts = [(-L, 0, L) if periodic[a] else (0,) for a in range(dim)]
            for sh in product(*shifts):
                touch = 0
                ok = True
                for a in range(dim):
                    lo = max(xa[a], xb[a] + sh[a])
                    hi = min(xa[a] + wa, xb[a] + sh[a] + wb)
                    if hi < lo:
                        ok = False
                        break
                    if hi == lo:
                        touch += 1
                if ok and 1 <= touch <= conn:
                    return False
    return True


def face_census(mesh, periodic, nroot=None):
    """(n_conf, n_hang, n_bnd) counted from every cell's own faces."""
    dim = len(next(iter(mesh))) - 1
    conf2 = hang = bnd = 0
    for cell in mesh:
        for axis in range(dim):
            for sign in (-1, 1):
                nb = face_neighbour(cell, axis, sign, periodic, nroot)
                if nb is None:
                    bnd += 1
                    continue
                leaf = containing_leaf(mesh, nb)
                if leaf is None:
                    continue  # finer neighbours: counted from their side
                if leaf[0] == cell[0]:
                    conf2 += 1
                else:
                    hang += 1
    assert conf2 % 2 == 0
    return conf2 // 2, hang, bnd


def volume(mesh, maxl):
    dim = len(next(iter(mesh))) - 1
    return sum(1 << (dim * (maxl - c[0])) for c in mesh)


def to_cells(level, xyz, dim, maxl):
    """oracle/GPU leaf boxes (anchor in finest units) -> list of set-model cells, array order."""
    return [(int(l),) + tuple(int(x) >> (maxl - int(l)) for x in X[:dim]) for l, X in zip(level, xyz)]


def complete(cells, dim, base):
    """Alg. 2's result by set algebra (readings G-2, G-3): the
    coarsest complete mesh that refines the uniform level-`base` mesh and in which every input
    cell is a leaf or an interior node.  interior = every strict ancestor of an input cell
    plus every cell above `base`; leaves = children of interior cells that are not interior."""
    interior = set()
    for l in range(base):
        interior |= uniform(dim, l)
    for cell in cells:
        c = cell
        while c[0] > 0:
            c = parent(c)
            if c in interior:
                break
            interior.add(c)
    if not interior:
        return {(0,) + (0,) * dim}
    leaves = set()
    for c in interior:
        for ch in children(c):
            if ch not in interior:
                leaves.add(ch)
    return leaves
