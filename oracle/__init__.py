"""CPU oracle for the linear-tree h-adaptation cycle -- TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  The product
(``paper_2306_06744_b200``) never does, and the two share no code.

The arithmetic lives in ``oracle/lto.cpp`` (plain sequential C++17, pointer tree);
this file only compiles it with g++ and marshals numpy arrays through ctypes.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lto.cpp")
_LIB = os.path.join(_HERE, "liblto.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile oracle/lto.cpp -> oracle/liblto.so (g++, no CUDA)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-shared", "-fPIC", _SRC, "-o", tmp])
        os.replace(tmp, _LIB)
    return _LIB


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t))


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.lto_encode.restype = C.c_uint64
        L.lto_encode.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(C.c_uint32)]
        L.lto_raw_id.restype = C.c_uint64
        L.lto_raw_id.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(C.c_uint32)]
        L.lto_decode.restype = None
        L.lto_decode.argtypes = [C.c_int, C.c_int, C.c_uint64, C.POINTER(C.c_int), C.POINTER(C.c_uint32)]
        L.lto_sort_linearise.restype = C.c_int64
        L.lto_sort_linearise.argtypes = [C.c_int, C.c_int, C.POINTER(C.c_uint64), C.c_int64]
        L.lto_build.restype = C.c_void_p
        L.lto_build.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(C.c_int)]
        L.lto_build_brick.restype = C.c_void_p
        L.lto_build_brick.argtypes = [C.c_int, C.POINTER(C.c_int), C.c_int, C.c_int, C.POINTER(C.c_int)]
        L.lto_build_from_keys.restype = C.c_void_p
        L.lto_build_from_keys.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(C.c_int),
                                          C.POINTER(C.c_uint64), C.c_int64]
        L.lto_build_complete.restype = C.c_void_p
        L.lto_build_complete.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(C.c_int),
                                         C.POINTER(C.c_uint64), C.c_int64]
        L.lto_build_from_points.restype = C.c_void_p
        L.lto_build_from_points.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(C.c_int),
                                            C.POINTER(C.c_double), C.POINTER(C.c_double), C.c_int64]
        L.lto_point_cell.restype = C.c_uint32
        L.lto_point_cell.argtypes = [C.c_double, C.c_double, C.c_double, C.c_int]
        L.lto_free.restype = None
        L.lto_free.argtypes = [C.c_void_p]
        L.lto_num_leaves.restype = C.c_int64
        L.lto_num_leaves.argtypes = [C.c_void_p]
        L.lto_keys.restype = None
        L.lto_keys.argtypes = [C.c_void_p, C.POINTER(C.c_uint64)]
        L.lto_leaf_boxes.restype = None
        L.lto_leaf_boxes.argtypes = [C.c_void_p, C.POINTER(C.c_int32), C.POINTER(C.c_uint32)]
        L.lto_dfs_is_sorted.restype = C.c_int
        L.lto_dfs_is_sorted.argtypes = [C.c_void_p]
        L.lto_adapt.restype = None
        L.lto_adapt.argtypes = [C.c_void_p, C.POINTER(C.c_int8)]
        L.lto_balance.restype = C.c_int
        L.lto_balance.argtypes = [C.c_void_p, C.POINTER(C.c_int64)]
        L.lto_balance_conn.restype = C.c_int
        L.lto_balance_conn.argtypes = [C.c_void_p, C.POINTER(C.c_int64), C.c_int]
        L.lto_connect.restype = C.c_int
        L.lto_connect.argtypes = [C.c_void_p, C.c_int]
        L.lto_face_counts.restype = None
        L.lto_face_counts.argtypes = [C.c_void_p, C.POINTER(C.c_int64)]
        L.lto_faces.restype = None
        L.lto_faces.argtypes = [C.c_void_p, C.POINTER(C.c_int32), C.POINTER(C.c_uint8),
                                C.POINTER(C.c_int32), C.POINTER(C.c_uint8),
                                C.POINTER(C.c_int32), C.POINTER(C.c_uint8),
                                C.POINTER(C.c_int32), C.POINTER(C.c_uint8)]
        L.lto_build_map.restype = C.c_int
        L.lto_build_map.argtypes = [C.c_void_p]
        L.lto_map.restype = None
        L.lto_map.argtypes = [C.c_void_p, C.POINTER(C.c_int32), C.POINTER(C.c_uint8)]
        L.lto_num_old_leaves.restype = C.c_int64
        L.lto_num_old_leaves.argtypes = [C.c_void_p]
        L.lto_old_keys.restype = None
        L.lto_old_keys.argtypes = [C.c_void_p, C.POINTER(C.c_uint64)]
        L.lto_transfer_rows.restype = C.c_int
        L.lto_transfer_rows.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_double),
                                        C.c_int, C.c_int, C.c_int64, C.c_int64]
        L.lto_drop_snapshot.restype = None
        L.lto_drop_snapshot.argtypes = [C.c_void_p]
        L.lto_operators.restype = C.c_int
        L.lto_operators.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(C.c_double)]
        L.lto_mortar_project.restype = C.c_int
        L.lto_mortar_project.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_double), C.c_int, C.c_int]
        L.lto_mortar_gather.restype = C.c_int
        L.lto_mortar_gather.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_double), C.c_int, C.c_int]
        L.lto_common_flux.restype = C.c_int
        L.lto_common_flux.argtypes = [C.c_void_p] + [C.POINTER(C.c_double)] * 3 + [C.c_int]
        L.lto_fr_rhs.restype = C.c_int
        L.lto_fr_rhs.argtypes = [C.c_void_p] + [C.POINTER(C.c_double)] * 4 + [C.c_int]
        L.lto_rk3_stage.restype = C.c_int
        L.lto_rk3_stage.argtypes = [C.c_int, C.c_double, C.c_int64] + [C.POINTER(C.c_double)] * 4
        L.lto_fr_operators.restype = C.c_int
        L.lto_fr_operators.argtypes = [C.c_int, C.c_int, C.POINTER(C.c_double)]
        L.lto_face_interp.restype = C.c_int
        L.lto_face_interp.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_double), C.c_int, C.c_int]
        L.lto_face_operators.restype = C.c_int
        L.lto_face_operators.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(C.c_double)]
        L.lto_gauss_legendre.restype = None
        L.lto_gauss_legendre.argtypes = [C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        _lib = L
    return _lib


# ------------------------------------------------------------------ free functions
def encode(dim, maxl, level, x):
    xx = np.zeros(3, np.uint32)
    xx[:dim] = x[:dim]
    return int(lib().lto_encode(dim, maxl, level, _p(xx, C.c_uint32)))


def raw_id(dim, maxl, level, x):
    xx = np.zeros(3, np.uint32)
    xx[:dim] = x[:dim]
    return int(lib().lto_raw_id(dim, maxl, level, _p(xx, C.c_uint32)))


def decode(dim, maxl, key):
    lvl = C.c_int(0)
    xx = np.zeros(3, np.uint32)
    lib().lto_decode(dim, maxl, C.c_uint64(int(key)), C.byref(lvl), _p(xx, C.c_uint32))
    return lvl.value, tuple(int(v) for v in xx[:dim])


def point_cell(x, lo, hi, maxl):
    """Reading G-1: depth-D_max integer cell of a scattered coordinate."""
    return int(lib().lto_point_cell(float(x), float(lo), float(hi), int(maxl)))


def sort_linearise(dim, maxl, keys):
    k = np.ascontiguousarray(keys, dtype=np.uint64).copy()
    m = lib().lto_sort_linearise(dim, maxl, _p(k, C.c_uint64), k.size)
    return k[:m].copy()


def gauss_legendre(n):
    z = np.zeros(n)
    w = np.zeros(n)
    lib().lto_gauss_legendre(n, _p(z, C.c_double), _p(w, C.c_double))
    return z, w


def operators(dim, p):
    """Dense transfer operators: dict(interp[nc,N,N], proj[nc,N,N], mass[N,N], S[nc,N,N])."""
    nc, N = 1 << dim, (p + 1) ** dim
    out = {}
    for which, name, shape in ((0, "interp", (nc, N, N)), (1, "proj", (nc, N, N)),
                               (2, "mass", (N, N)), (3, "S", (nc, N, N))):
        a = np.zeros(shape)
        rc = lib().lto_operators(dim, p, which, _p(a, C.c_double))
        assert rc == 0
        out[name] = a
    return out


def face_operators(dim, p):
    """(to_mortar [ns,N,N] of Eq. 17, from_mortar [ns,N,N] = M^-1 S^s of Eq. 20) for the
    (dim-1)-dimensional faces; ns = 2^(dim-1), N = (p+1)^(dim-1)."""
    ns, N = 1 << (dim - 1), (p + 1) ** (dim - 1)
    out = []
    for which in (0, 1):
        a = np.zeros((ns, N, N))
        if lib().lto_face_operators(dim, p, which, _p(a, C.c_double)) != 0:
            raise OracleError("oracle face operators: bad arguments")
        out.append(a)
    return tuple(out)


def fr_operators(p):
    """(D [P1,P1] = l_j'(z_i), l(-1) [P1], l(+1) [P1], g_L'(z) [P1], g_R'(z) [P1]) of Eq. 3-4 with Radau g."""
    P1 = p + 1
    out = []
    for which, shape in enumerate([(P1, P1), (P1,), (P1,), (P1,), (P1,)]):
        a = np.zeros(shape)
        lib().lto_fr_operators(p, which, _p(a, C.c_double))
        out.append(a)
    return tuple(out)


def rk3_stage(stage, dt, u_n, u_stage, rhs):
    """Eq. 6, one stage: stage 1 u^n + dt R; stage 2 3/4 u^n + 1/4 u^1 + 1/4 dt R(u^1);
    stage 3 1/3 u^n + 2/3 u^2 + 2/3 dt R(u^2).  u_stage is the vector R was evaluated at."""
    un = np.ascontiguousarray(u_n, dtype=np.float64)
    us = np.ascontiguousarray(u_stage, dtype=np.float64)
    R = np.ascontiguousarray(rhs, dtype=np.float64)
    assert un.shape == us.shape == R.shape
    out = np.zeros(un.shape)
    if lib().lto_rk3_stage(int(stage), float(dt), un.size, _p(un, C.c_double), _p(us, C.c_double),
                           _p(R, C.c_double), _p(out, C.c_double)) != 0:
        raise OracleError("oracle rk3_stage: stage must be 1, 2 or 3")
    return out


class OracleError(RuntimeError):
    pass


class Tree:
    """Pointer-based linear-tree oracle.  Same verbs as the product's C ABI."""

    def __init__(self, dim, base_level, max_level, periodic=None, keys=None, complete=False, points=None,
                 domain=None, nroot=None):
        """keys: unsorted IDs that must tile the domain (sort + linearise, Alg. 3);
        keys + complete=True: Alg. 2 completion of the octants over the uniform base tree;
        points [n][dim] fp64 + domain (lo.., hi..): Alg. 2 from scattered points;
        nroot (n_x, n_y[, n_z]): a brick of root cubes (forest), uniform at base_level."""
        self.dim, self.base, self.maxl = dim, base_level, max_level
        self.nc, self.nf = 1 << dim, 2 * dim
        self.nroot = tuple(int(v) for v in nroot[:dim]) if nroot is not None else (1,) * dim
        per = np.zeros(3, np.int32)
        if periodic is not None:
            per[:dim] = np.asarray(periodic, np.int32)[:dim]
        if nroot is not None:
            assert keys is None and points is None, "construction is defined on a single cube"
            nr = np.ones(3, np.int32)
            nr[:dim] = np.asarray(nroot, np.int32)[:dim]
            self._h = lib().lto_build_brick(dim, _p(nr, C.c_int), base_level, max_level, _p(per, C.c_int))
        elif points is not None:
            pts = np.ascontiguousarray(points, dtype=np.float64).reshape(-1, dim)
            dom = np.ascontiguousarray(domain, dtype=np.float64)
            assert dom.size == 2 * dim
            self._h = lib().lto_build_from_points(dim, base_level, max_level, _p(per, C.c_int),
                                                  _p(dom, C.c_double), _p(pts, C.c_double), pts.shape[0])
        elif keys is not None and complete:
            k = np.ascontiguousarray(keys, dtype=np.uint64)
            self._h = lib().lto_build_complete(dim, base_level, max_level, _p(per, C.c_int),
                                               _p(k, C.c_uint64), k.size)
        elif keys is None:
            self._h = lib().lto_build(dim, base_level, max_level, _p(per, C.c_int))
        else:
            k = np.ascontiguousarray(keys, dtype=np.uint64)
            self._h = lib().lto_build_from_keys(dim, base_level, max_level, _p(per, C.c_int),
                                                _p(k, C.c_uint64), k.size)
        if not self._h:
            raise OracleError("oracle: bad arguments or incomplete key set")

    def __del__(self):
        if getattr(self, "_h", None) and _lib is not None:
            try:
                _lib.lto_free(self._h)
            except Exception:  # interpreter shutdown
                pass
            self._h = None

    # -- state
    def num_leaves(self):
        return int(lib().lto_num_leaves(self._h))

    def keys(self):
        k = np.zeros(self.num_leaves(), np.uint64)
        lib().lto_keys(self._h, _p(k, C.c_uint64))
        return k

    def leaf_boxes(self):
        """(level[M] int32, xyz[M,3] uint32 integer anchors in finest-cell units)."""
        M = self.num_leaves()
        lvl = np.zeros(M, np.int32)
        xyz = np.zeros((M, 3), np.uint32)
        lib().lto_leaf_boxes(self._h, _p(lvl, C.c_int32), _p(xyz, C.c_uint32))
        return lvl, xyz

    def dfs_is_sorted(self):
        return bool(lib().lto_dfs_is_sorted(self._h))

    # -- the cycle
    def adapt(self, flags):
        f = np.ascontiguousarray(flags, dtype=np.int8)
        assert f.size == self.num_leaves()
        lib().lto_adapt(self._h, _p(f, C.c_int8))

    def balance(self, conn=1):
        """conn: 1 faces (default), 2 + edges (3-D: the paper's strong balance; 2-D: corners),
        3 + corners (3-D)."""
        ns = C.c_int64(0)
        it = lib().lto_balance_conn(self._h, C.byref(ns), int(conn))
        if it < 0:
            raise OracleError("oracle balance: bad connectivity %r" % (conn,))
        self.last_balance_splits = ns.value
        return int(it)

    def connect(self, method=0):
        rc = lib().lto_connect(self._h, method)
        if rc != 0:
            raise OracleError("oracle connect: rc=%d (unbalanced or incomplete tree)" % rc)
        cnt = np.zeros(3, np.int64)
        lib().lto_face_counts(self._h, _p(cnt, C.c_int64))
        M, nf = self.num_leaves(), self.nf
        F = dict(
            nbr=np.zeros(M * nf, np.int32), kind=np.zeros(M * nf, np.uint8),
            conf=np.zeros((int(cnt[0]), 2), np.int32), conf_axis=np.zeros(int(cnt[0]), np.uint8),
            hang=np.zeros((int(cnt[1]), 2), np.int32), hang_info=np.zeros(int(cnt[1]), np.uint8),
            bnd=np.zeros(int(cnt[2]), np.int32), bnd_face=np.zeros(int(cnt[2]), np.uint8),
        )
        lib().lto_faces(self._h, _p(F["nbr"], C.c_int32), _p(F["kind"], C.c_uint8),
                        _p(F["conf"], C.c_int32), _p(F["conf_axis"], C.c_uint8),
                        _p(F["hang"], C.c_int32), _p(F["hang_info"], C.c_uint8),
                        _p(F["bnd"], C.c_int32), _p(F["bnd_face"], C.c_uint8))
        F["n_conf"], F["n_hang"], F["n_bnd"] = (int(c) for c in cnt)
        return F

    def build_map(self):
        rc = lib().lto_build_map(self._h)
        if rc != 0:
            raise OracleError("oracle map: a new leaf is more than one level from the old tree")
        M = self.num_leaves()
        src = np.zeros(M, np.int32)
        kind = np.zeros(M, np.uint8)
        lib().lto_map(self._h, _p(src, C.c_int32), _p(kind, C.c_uint8))
        return src, kind

    def _map_window(self, j0, j1):
        M = self.num_leaves()
        src = np.zeros(M, np.int32)
        kind = np.zeros(M, np.uint8)
        lib().lto_map(self._h, _p(src, C.c_int32), _p(kind, C.c_uint8))
        return src[j0:j1], kind[j0:j1]

    def old_keys(self):
        k = np.zeros(int(lib().lto_num_old_leaves(self._h)), np.uint64)
        lib().lto_old_keys(self._h, _p(k, C.c_uint64))
        return k

    def transfer_rows(self, u_old, p, nvars, j0, j1, old_offset=0):
        """Rows [j0, j1) of u_new (requires build_map()).  u_old holds the old rows
        [old_offset, old_offset + len(u_old)): a window is enough when only those rows are sources
        (marshalling only: the base pointer handed to the C++ side is shifted back by old_offset rows)."""
        N = (p + 1) ** self.dim
        u_old = np.ascontiguousarray(u_old, dtype=np.float64)
        out = np.zeros((j1 - j0, nvars, N))
        if old_offset or u_old.shape[0] < int(lib().lto_num_old_leaves(self._h)):
            src, kind = self._map_window(j0, j1)
            last = src.astype(np.int64) + np.where((kind & 15) == 2, self.nc - 1, 0)
            assert src.min() >= old_offset and last.max() < old_offset + u_old.shape[0], \
                "transfer_rows: the window does not cover the sources of rows [%d, %d)" % (j0, j1)
        base = C.cast(C.c_void_p(u_old.ctypes.data - int(old_offset) * nvars * N * 8), C.POINTER(C.c_double))
        rc = lib().lto_transfer_rows(self._h, base, _p(out, C.c_double), p, nvars, j0, j1)
        if rc != 0:
            raise OracleError("oracle transfer: rc=%d" % rc)
        return out

    def transfer(self, u_old, p, nvars):
        """Alg. 7 map + copy / interpolate / project; consumes the snapshot."""
        self.build_map()
        out = self.transfer_rows(u_old, p, nvars, 0, self.num_leaves())
        lib().lto_drop_snapshot(self._h)
        return out

    def face_interp(self, u, p, nvars):
        """Alg. 8 step 1: u [M, nvars, N] -> u_face [M, nf, nvars, Nf] (solution at the face points)."""
        N, Nf = (p + 1) ** self.dim, (p + 1) ** (self.dim - 1)
        u = np.ascontiguousarray(u, dtype=np.float64)
        assert u.shape == (self.num_leaves(), nvars, N)
        out = np.zeros((self.num_leaves(), self.nf, nvars, Nf))
        if lib().lto_face_interp(self._h, _p(u, C.c_double), _p(out, C.c_double), p, nvars) != 0:
            raise OracleError("oracle face_interp: bad arguments")
        return out

    def common_flux(self, u_face, u_nb, p):
        """Alg. 8 step 3 (Rusanov, Euler): own and neighbour traces -> F* along +axis on kind 1 / 2 slots
        (NaN elsewhere).  nvars = dim + 2."""
        uf = np.ascontiguousarray(u_face, dtype=np.float64)
        un = np.ascontiguousarray(u_nb, dtype=np.float64)
        assert uf.shape == un.shape == (self.num_leaves(), self.nf, self.dim + 2, (p + 1) ** (self.dim - 1))
        out = np.full(uf.shape, np.nan)
        if lib().lto_common_flux(self._h, _p(uf, C.c_double), _p(un, C.c_double), _p(out, C.c_double), p) != 0:
            raise OracleError("oracle common_flux: connect first")
        return out

    def fr_rhs(self, u, f_star, p, width):
        """Eq. 2-5: u [M, dim+2, N], f_star [M, nf, dim+2, Nf] -> R [M, dim+2, N]."""
        u = np.ascontiguousarray(u, dtype=np.float64)
        fs = np.ascontiguousarray(f_star, dtype=np.float64)
        wd = np.ascontiguousarray(width, dtype=np.float64)
        assert u.shape == (self.num_leaves(), self.dim + 2, (p + 1) ** self.dim) and wd.size == self.dim
        out = np.zeros(u.shape)
        lib().lto_fr_rhs(self._h, _p(wd, C.c_double), _p(u, C.c_double), _p(fs, C.c_double), _p(out, C.c_double), p)
        return out

    def mortar_project(self, u_face, p, nvars):
        """Alg. 8 step 2: u_face [M, nf, nvars, Nf] -> neighbour traces on kind 1 / 2 slots
        (other slots are returned as NaN)."""
        Nf = (p + 1) ** (self.dim - 1)
        uf = np.ascontiguousarray(u_face, dtype=np.float64)
        assert uf.shape == (self.num_leaves(), self.nf, nvars, Nf)
        out = np.full(uf.shape, np.nan)
        rc = lib().lto_mortar_project(self._h, _p(uf, C.c_double), _p(out, C.c_double), p, nvars)
        if rc != 0:
            raise OracleError("oracle mortar_project: rc=%d (connect first)" % rc)
        return out

    def mortar_gather(self, f_mortar, p, nvars):
        """Alg. 8 step 4: f_mortar [M, nf, nvars, Nf] -> coarse-face fluxes on kind 3 slots
        (other slots are returned as NaN)."""
        Nf = (p + 1) ** (self.dim - 1)
        fm = np.ascontiguousarray(f_mortar, dtype=np.float64)
        assert fm.shape == (self.num_leaves(), self.nf, nvars, Nf)
        out = np.full(fm.shape, np.nan)
        rc = lib().lto_mortar_gather(self._h, _p(fm, C.c_double), _p(out, C.c_double), p, nvars)
        if rc != 0:
            raise OracleError("oracle mortar_gather: rc=%d" % rc)
        return out

    def drop_snapshot(self):
        lib().lto_drop_snapshot(self._h)
