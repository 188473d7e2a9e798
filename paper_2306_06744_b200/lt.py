"""Thin ctypes binding over the C ABI of liblt (include/lt.h).

Argument marshalling only: every step of the adaptation cycle runs in the CUDA kernels of
``csrc/``.  There is no CPU fallback -- if ``liblt.so`` is missing or no CUDA device is
present the calls raise ``LtError``.  PyTorch is used for device memory and streams only.

The functions carry the names of the C entry points (``lt_build`` -> ``Tree(...)`` /
``build``, ``lt_adapt`` -> ``Tree.adapt`` ...).
"""
from __future__ import annotations

import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
# LT_DEBUG_LIB=1 loads the checked build (python -m paper_2306_06744_b200.build --debug)
LIB_PATH = os.path.join(_HERE, "liblt_debug.so" if os.environ.get("LT_DEBUG_LIB") == "1" else "liblt.so")
_lib = None

LT_OK, LT_ERR_ARG, LT_ERR_CUDA, LT_ERR_OOM, LT_ERR_CAPACITY = 0, -1, -2, -3, -4
LT_ERR_UNBALANCED, LT_ERR_MAPPING, LT_ERR_INCOMPLETE = -5, -6, -7
LT_OPT_ADAPT_SORT, LT_OPT_BALANCE_FULL_SWEEPS, LT_OPT_DEBUG_BALANCE_SLACK = 1, 2, 3
LT_OPT_HOST_SLAB_LEAVES, LT_OPT_BALANCE_CONNECTIVITY = 4, 5


class LtError(RuntimeError):
    def __init__(self, status, where=""):
        self.status = status
        msg = lib().lt_strerror(status).decode() if _lib is not None else "liblt not loaded"
        super().__init__("%s: %s (status %d, cuda error %d)" % (where, msg, status,
                                                                 _lib.lt_last_cuda_error() if _lib else -1))


class lt_faces(C.Structure):
    _fields_ = [("n_leaves", C.c_int64), ("n_conf", C.c_int64), ("n_hang", C.c_int64), ("n_bnd", C.c_int64),
                ("nbr", C.c_void_p), ("kind", C.c_void_p), ("conf", C.c_void_p), ("conf_axis", C.c_void_p),
                ("hang", C.c_void_p), ("hang_info", C.c_void_p), ("bnd", C.c_void_p), ("bnd_face", C.c_void_p)]


# every symbol include/lt.h declares: name -> (restype, argtypes)
_P, _I, _I64 = C.c_void_p, C.c_int, C.c_int64
SIGNATURES = {
    "lt_build": (_I, [_I, _I, _I, _P, _P, _P, C.POINTER(_P)]),
    "lt_build_from_keys": (_I, [_I, _I, _I, _P, _P, _P, _P, _I64, C.POINTER(_P)]),
    "lt_build_complete_from_keys": (_I, [_I, _I, _I, _P, _P, _P, _P, _I64, C.POINTER(_P)]),
    "lt_build_from_points": (_I, [_I, _I, _I, _P, _P, _P, _P, _I64, C.POINTER(_P)]),
    "lt_free": (None, [_P]),
    "lt_reserve": (_I, [_P, _I64]),
    "lt_adapt": (_I, [_P, _P]),
    "lt_balance": (_I, [_P, C.POINTER(_I)]),
    "lt_connect": (_I, [_P, C.POINTER(lt_faces)]),
    "lt_connect_begin": (_I, [_P]),
    "lt_connect_end": (_I, [_P, C.POINTER(lt_faces)]),
    "lt_transfer": (_I, [_P, _P, _P, _I, _I]),
    "lt_transfer_host": (_I, [_P, _P, _P, _I, _I]),
    "lt_mortar_project": (_I, [_P, _P, _P, _I, _I]),
    "lt_face_interp": (_I, [_P, _P, _P, _I, _I]),
    "lt_common_flux": (_I, [_P, _P, _P, _P, _I]),
    "lt_fr_rhs": (_I, [_P, _P, _P, _P, _I]),
    "lt_face_flux": (_I, [_P, _P, _P, _I]),
    "lt_fr_stage_faces": (_I, [_P, _I, C.c_double, _P, _P, _P, _P, _P, _I]),
    "lt_rk3_stage": (_I, [_P, _I, C.c_double, _P, _P, _P, _P, _I]),
    "lt_fr_stage": (_I, [_P, _I, C.c_double, _P, _P, _P, _P, _I]),
    "lt_mortar_gather": (_I, [_P, _P, _P, _I, _I]),
    "lt_num_leaves": (_I64, [_P]),
    "lt_num_old_leaves": (_I64, [_P]),
    "lt_last_balance_iters": (_I, [_P]),
    "lt_keys": (_P, [_P]),
    "lt_old_keys": (_P, [_P]),
    "lt_map": (_I, [_P, C.POINTER(_P), C.POINTER(_P)]),
    "lt_leaf_boxes": (_I, [_P, _P, _P]),
    "lt_encode": (_I, [_I, _I, _P, _P, _I64, _P, _P]),
    "lt_decode": (_I, [_I, _I, _P, _I64, _P, _P, _P]),
    "lt_sort_keys": (_I, [_I, _I, _P, _I64, _I, C.POINTER(_I64), _P]),
    "lt_sort_keys_static": (_I, [_I, _I, _P, _I64, _P]),
    "lt_domain": (_I, [_P, _P]),
    "lt_info": (_I, [_P, C.POINTER(_I), C.POINTER(_I), C.POINTER(_I), _P]),
    "lt_sync": (_I, [_P]),
    "lt_set_option": (_I, [_P, _I, _I]),
    "lt_timings": (_I, [_P, _P]),
    "lt_launch_count": (_I64, [_P]),
    "lt_host_syncs": (_I64, [_P]),
    "lt_build_brick": (_I, [_I, _P, _I, _I, _P, _P, _P, C.POINTER(_P)]),
    "lt_roots": (_I, [_P, _P]),
    "lt_balance_phases": (_I, [_P, _P]),
    "lt_strerror": (C.c_char_p, [_I]),
    "lt_last_cuda_error": (_I, []),
    "lt_version": (_I, []),
    "lt_debug_build": (_I, []),
}


def lib():
    """Load liblt.so (raises if it has not been built: there is no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError("liblt.so is missing: run `python -m paper_2306_06744_b200.build` "
                               "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(L, name)
            fn.restype = res
            fn.argtypes = args
        _lib = L
    return _lib


def _check(rc, where):
    if rc != LT_OK:
        raise LtError(rc, where)


class _DevView:
    """Zero-copy view of tree-owned device memory through __cuda_array_interface__."""

    def __init__(self, ptr, shape, typestr):
        self.__cuda_array_interface__ = {"shape": tuple(shape), "typestr": typestr, "data": (int(ptr), False),
                                         "version": 2, "strides": None}


_TYPESTR = {torch.int32: "<i4", torch.uint8: "|u1", torch.int64: "<i8", torch.float64: "<f8"}


def _view(ptr, shape, dtype, device):
    n = 1
    for s in shape:
        n *= s
    if n == 0 or not ptr:
        return torch.empty(shape, dtype=dtype, device=device)
    return torch.as_tensor(_DevView(ptr, shape, _TYPESTR[dtype]), device=device)


def _stream_ptr(device):
    return C.c_void_p(torch.cuda.current_stream(device).cuda_stream)


def _dptr(t: torch.Tensor, dtype, where):
    if not t.is_cuda or t.dtype != dtype or not t.is_contiguous():
        raise TypeError("%s: expected a contiguous CUDA tensor of dtype %s" % (where, dtype))
    return C.c_void_p(t.data_ptr())


class Tree:
    """One linear quadtree / octree on the current CUDA device (handle of lt_build)."""

    def __init__(self, dim, base_level, max_level, domain=None, periodic=None, keys=None, device=None,
                 complete=False, points=None, nroot=None):
        self.device = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
        self.dim, self.base, self.maxl = dim, base_level, max_level
        self.nc, self.nf = 1 << dim, 2 * dim
        dom = (C.c_double * (2 * dim))(*domain) if domain is not None else None
        per = (C.c_int * dim)(*[int(bool(v)) for v in periodic]) if periodic is not None else None
        h = C.c_void_p()
        with torch.cuda.device(self.device):
            self._stream = torch.cuda.current_stream(self.device)
            if points is not None:
                x = points.contiguous()
                if x.dim() != 2 or x.shape[1] != dim:
                    raise ValueError("lt_build_from_points: points must be [n, dim]")
                rc = lib().lt_build_from_points(dim, base_level, max_level, dom, per, _stream_ptr(self.device),
                                                _dptr(x, torch.float64, "points"), x.shape[0], C.byref(h))
            elif keys is not None and complete:
                k = keys.contiguous()
                rc = lib().lt_build_complete_from_keys(dim, base_level, max_level, dom, per,
                                                       _stream_ptr(self.device),
                                                       _dptr(k.view(torch.int64), torch.int64, "keys"), k.numel(),
                                                       C.byref(h))
            elif keys is None and nroot is not None:
                nr = (C.c_int * dim)(*[int(v) for v in nroot[:dim]])
                rc = lib().lt_build_brick(dim, nr, base_level, max_level, dom, per, _stream_ptr(self.device),
                                          C.byref(h))
            elif keys is None:
                rc = lib().lt_build(dim, base_level, max_level, dom, per, _stream_ptr(self.device), C.byref(h))
            else:
                k = keys.contiguous()
                rc = lib().lt_build_from_keys(dim, base_level, max_level, dom, per, _stream_ptr(self.device),
                                              _dptr(k.view(torch.int64), torch.int64, "keys"), k.numel(), C.byref(h))
        _check(rc, "lt_build")
        self._h = h

    def __del__(self):
        self.free()

    def free(self):
        h = getattr(self, "_h", None)
        if h and _lib is not None:
            try:
                _lib.lt_free(h)
            except Exception:  # interpreter shutdown
                pass
            self._h = None

    # ---- the cycle
    def adapt(self, flags: torch.Tensor):
        """lt_adapt: flags int8 [num_leaves] on the device."""
        if flags.numel() != self.num_leaves():
            raise ValueError("lt_adapt: flags must have one entry per leaf")
        _check(lib().lt_adapt(self._h, _dptr(flags, torch.int8, "flags")), "lt_adapt")

    def balance(self, connectivity=None, want_iters=True):
        """lt_balance; connectivity (sticky option LT_OPT_BALANCE_CONNECTIVITY): 1 faces,
        2 + edges (the paper's strong balance in 3-D), 3 + corners.  want_iters=False passes
        iters = NULL, which lets the call return without waiting (see lt.h); last_balance_iters()
        gives the sweep count afterwards."""
        if connectivity is not None:
            self.set_option(LT_OPT_BALANCE_CONNECTIVITY, int(connectivity))
        if not want_iters:
            _check(lib().lt_balance(self._h, None), "lt_balance")
            return None
        it = C.c_int(0)
        _check(lib().lt_balance(self._h, C.byref(it)), "lt_balance")
        return it.value

    def last_balance_iters(self) -> int:
        it = lib().lt_last_balance_iters(self._h)
        if it < 0:
            raise LtError(int(it), "lt_last_balance_iters")
        return int(it)

    def transfer_into(self, u_old: torch.Tensor, u_new: torch.Tensor, p: int, nvars: int):
        """lt_transfer into a caller-sized buffer (>= num_leaves rows) without asking for the leaf count,
        so that the call does not wait for a pending lt_adapt / lt_balance."""
        _check(lib().lt_transfer(self._h, _dptr(u_old, torch.float64, "u_old"), _dptr(u_new, torch.float64, "u_new"),
                                 p, nvars), "lt_transfer")
        return u_new

    def connect(self) -> dict:
        """lt_connect: dict of zero-copy views (valid until the next mutating call)."""
        F = lt_faces()
        _check(lib().lt_connect(self._h, C.byref(F)), "lt_connect")
        return self._faces_dict(F)

    def connect_begin(self):
        """lt_connect_begin: enqueue the face query on the tree's side stream (overlaps lt_transfer)."""
        _check(lib().lt_connect_begin(self._h), "lt_connect_begin")

    def connect_end(self) -> dict:
        """lt_connect_end: join the side stream and return the same dict as connect()."""
        F = lt_faces()
        _check(lib().lt_connect_end(self._h, C.byref(F)), "lt_connect_end")
        return self._faces_dict(F)

    def _faces_dict(self, F) -> dict:
        M, nf, dev = F.n_leaves, self.nf, self.device
        return dict(
            n_leaves=M, n_conf=F.n_conf, n_hang=F.n_hang, n_bnd=F.n_bnd,
            nbr=_view(F.nbr, (M * nf,), torch.int32, dev), kind=_view(F.kind, (M * nf,), torch.uint8, dev),
            conf=_view(F.conf, (F.n_conf, 2), torch.int32, dev),
            conf_axis=_view(F.conf_axis, (F.n_conf,), torch.uint8, dev),
            hang=_view(F.hang, (F.n_hang, 2), torch.int32, dev),
            hang_info=_view(F.hang_info, (F.n_hang,), torch.uint8, dev),
            bnd=_view(F.bnd, (F.n_bnd,), torch.int32, dev), bnd_face=_view(F.bnd_face, (F.n_bnd,), torch.uint8, dev))

    def transfer(self, u_old: torch.Tensor, p: int, nvars: int, u_new: torch.Tensor = None) -> torch.Tensor:
        """lt_transfer: u_old [n_old, nvars, N] fp64 -> u_new [num_leaves, nvars, N] fp64."""
        N = (p + 1) ** self.dim
        n_old = self.num_old_leaves() or self.num_leaves()
        if tuple(u_old.shape) != (n_old, nvars, N):
            raise ValueError("lt_transfer: u_old must be [%d, %d, %d]" % (n_old, nvars, N))
        if u_new is None:
            u_new = torch.empty((self.num_leaves(), nvars, N), dtype=torch.float64, device=self.device)
        elif tuple(u_new.shape) != (self.num_leaves(), nvars, N):
            raise ValueError("lt_transfer: u_new has the wrong shape")
        _check(lib().lt_transfer(self._h, _dptr(u_old, torch.float64, "u_old"), _dptr(u_new, torch.float64, "u_new"),
                                 p, nvars), "lt_transfer")
        return u_new

    def _face_shape(self, p, nvars):
        return (self.num_leaves(), self.nf, nvars, (p + 1) ** (self.dim - 1))

    def face_interp(self, u: torch.Tensor, p: int, nvars: int, u_face: torch.Tensor = None) -> torch.Tensor:
        """lt_face_interp (Alg. 8 step 1): u [M, nvars, N] -> u_face [M, nf, nvars, Nf]."""
        if tuple(u.shape) != (self.num_leaves(), nvars, (p + 1) ** self.dim):
            raise ValueError("lt_face_interp: u must be [%d, %d, %d]" % (self.num_leaves(), nvars, (p + 1) ** self.dim))
        if u_face is None:
            u_face = torch.empty(self._face_shape(p, nvars), dtype=torch.float64, device=self.device)
        _check(lib().lt_face_interp(self._h, _dptr(u, torch.float64, "u"), _dptr(u_face, torch.float64, "u_face"),
                                    p, nvars), "lt_face_interp")
        return u_face

    def common_flux(self, u_face: torch.Tensor, u_nb: torch.Tensor, p: int, f_star: torch.Tensor = None):
        """lt_common_flux (Alg. 8 step 3, Rusanov / Euler): kind 1 / 2 slots of f_star (NaN-filled when
        allocated here)."""
        shp = self._face_shape(p, self.dim + 2)
        if tuple(u_face.shape) != shp or tuple(u_nb.shape) != shp:
            raise ValueError("lt_common_flux: face arrays must be %s" % (shp,))
        if f_star is None:
            f_star = torch.full_like(u_face, float("nan"))
        _check(lib().lt_common_flux(self._h, _dptr(u_face, torch.float64, "u_face"), _dptr(u_nb, torch.float64, "u_nb"),
                                    _dptr(f_star, torch.float64, "f_star"), p), "lt_common_flux")
        return f_star

    def face_flux(self, u_face: torch.Tensor, p: int, f_star: torch.Tensor = None):
        """lt_face_flux (Alg. 8 steps 2 + 3 fused): kind 1 / 2 slots of f_star (NaN-filled when allocated here)."""
        shp = self._face_shape(p, self.dim + 2)
        if tuple(u_face.shape) != shp:
            raise ValueError("lt_face_flux: u_face must be %s" % (shp,))
        if f_star is None:
            f_star = torch.full_like(u_face, float("nan"))
        _check(lib().lt_face_flux(self._h, _dptr(u_face, torch.float64, "u_face"),
                                  _dptr(f_star, torch.float64, "f_star"), p), "lt_face_flux")
        return f_star

    def fr_rhs(self, u: torch.Tensor, f_star: torch.Tensor, p: int, rhs: torch.Tensor = None) -> torch.Tensor:
        """lt_fr_rhs (Eq. 2-5): u [M, dim+2, N], f_star face array -> R [M, dim+2, N]."""
        if tuple(u.shape) != (self.num_leaves(), self.dim + 2, (p + 1) ** self.dim):
            raise ValueError("lt_fr_rhs: u must be [M, dim+2, (p+1)^dim]")
        if tuple(f_star.shape) != self._face_shape(p, self.dim + 2):
            raise ValueError("lt_fr_rhs: f_star must be %s" % (self._face_shape(p, self.dim + 2),))
        if rhs is None:
            rhs = torch.empty_like(u)
        _check(lib().lt_fr_rhs(self._h, _dptr(u, torch.float64, "u"), _dptr(f_star, torch.float64, "f_star"),
                               _dptr(rhs, torch.float64, "rhs"), p), "lt_fr_rhs")
        return rhs

    def rk3_stage(self, stage: int, dt: float, u_n, u_stage, rhs, p: int, out=None):
        """lt_rk3_stage (Eq. 6)."""
        if out is None:
            out = torch.empty_like(u_n)
        _check(lib().lt_rk3_stage(self._h, stage, dt, _dptr(u_n, torch.float64, "u_n"),
                                  _dptr(u_stage, torch.float64, "u_stage"), _dptr(rhs, torch.float64, "rhs"),
                                  _dptr(out, torch.float64, "out"), p), "lt_rk3_stage")
        return out

    def fr_stage(self, stage: int, dt: float, u_n, u_stage, f_star, p: int, out=None):
        """lt_fr_stage: right-hand side + RK stage of Eq. 6 in one pass."""
        if out is None:
            out = torch.empty_like(u_n)
        _check(lib().lt_fr_stage(self._h, stage, dt, _dptr(u_n, torch.float64, "u_n"),
                                 _dptr(u_stage, torch.float64, "u_stage"), _dptr(f_star, torch.float64, "f_star"),
                                 _dptr(out, torch.float64, "out"), p), "lt_fr_stage")
        return out

    def fr_stage_faces(self, stage: int, dt: float, u_n, u_stage, f_star, p: int, out=None, u_face_out=None):
        """lt_fr_stage_faces: lt_fr_stage + the traces of the result at the face points; returns (u_out, u_face)."""
        if out is None:
            out = torch.empty_like(u_n)
        if u_face_out is None:
            u_face_out = torch.empty_like(f_star)
        _check(lib().lt_fr_stage_faces(self._h, stage, dt, _dptr(u_n, torch.float64, "u_n"),
                                       _dptr(u_stage, torch.float64, "u_stage"), _dptr(f_star, torch.float64, "f_star"),
                                       _dptr(out, torch.float64, "out"), _dptr(u_face_out, torch.float64, "u_face_out"),
                                       p), "lt_fr_stage_faces")
        return out, u_face_out

    def mortar_project(self, u_face: torch.Tensor, p: int, nvars: int, u_nb: torch.Tensor = None) -> torch.Tensor:
        """lt_mortar_project (Alg. 8 step 2): u_face [M, nf, nvars, Nf] -> neighbour traces; slots
        of kind 0 / 3 keep what u_nb held (NaN when it is allocated here)."""
        if tuple(u_face.shape) != self._face_shape(p, nvars):
            raise ValueError("lt_mortar_project: u_face must be %s" % (self._face_shape(p, nvars),))
        if u_nb is None:
            u_nb = torch.full_like(u_face, float("nan"))
        _check(lib().lt_mortar_project(self._h, _dptr(u_face, torch.float64, "u_face"),
                                       _dptr(u_nb, torch.float64, "u_nb"), p, nvars), "lt_mortar_project")
        return u_nb

    def mortar_gather(self, f_mortar: torch.Tensor, p: int, nvars: int, f_face: torch.Tensor = None) -> torch.Tensor:
        """lt_mortar_gather (Alg. 8 step 4): f_mortar [M, nf, nvars, Nf] -> coarse-face fluxes on kind 3
        slots of f_face (default: a NaN-filled array; pass f_mortar itself to work in place)."""
        if tuple(f_mortar.shape) != self._face_shape(p, nvars):
            raise ValueError("lt_mortar_gather: f_mortar must be %s" % (self._face_shape(p, nvars),))
        if f_face is None:
            f_face = torch.full_like(f_mortar, float("nan"))
        _check(lib().lt_mortar_gather(self._h, _dptr(f_mortar, torch.float64, "f_mortar"),
                                      _dptr(f_face, torch.float64, "f_face"), p, nvars), "lt_mortar_gather")
        return f_face

    def transfer_host(self, u_old: torch.Tensor, u_new: torch.Tensor, p: int, nvars: int):
        """lt_transfer_host: HOST tensors (pinned or pageable), copies inside the call."""
        if u_old.is_cuda or u_new.is_cuda or u_old.dtype != torch.float64 or u_new.dtype != torch.float64:
            raise TypeError("lt_transfer_host: host float64 tensors expected")
        _check(lib().lt_transfer_host(self._h, C.c_void_p(u_old.data_ptr()), C.c_void_p(u_new.data_ptr()), p, nvars),
               "lt_transfer_host")

    # ---- accessors
    def num_leaves(self) -> int:
        n = lib().lt_num_leaves(self._h)
        if n < 0:
            raise LtError(int(n), "lt_num_leaves")
        return int(n)

    def num_old_leaves(self) -> int:
        return int(lib().lt_num_old_leaves(self._h))

    def keys(self) -> torch.Tensor:
        """lt_keys: zero-copy int64 view of the uint64 keys (all keys are < 2^63)."""
        return _view(lib().lt_keys(self._h), (self.num_leaves(),), torch.int64, self.device)

    def old_keys(self) -> torch.Tensor:
        return _view(lib().lt_old_keys(self._h), (self.num_old_leaves(),), torch.int64, self.device)

    def map(self):
        src, kind = C.c_void_p(), C.c_void_p()
        _check(lib().lt_map(self._h, C.byref(src), C.byref(kind)), "lt_map")
        M = self.num_leaves()
        return _view(src.value, (M,), torch.int32, self.device), _view(kind.value, (M,), torch.uint8, self.device)

    def leaf_boxes(self):
        """lt_leaf_boxes: (level int32 [M], xyz int32 [M,3]) decoded on the device."""
        M = self.num_leaves()
        lvl = torch.empty(M, dtype=torch.int32, device=self.device)
        xyz = torch.empty((M, 3), dtype=torch.int32, device=self.device)
        _check(lib().lt_leaf_boxes(self._h, C.c_void_p(lvl.data_ptr()), C.c_void_p(xyz.data_ptr())), "lt_leaf_boxes")
        return lvl, xyz

    def roots(self):
        out = (C.c_int * 3)()
        _check(lib().lt_roots(self._h, out), "lt_roots")
        return tuple(out[: self.dim])

    def reserve(self, n):
        _check(lib().lt_reserve(self._h, int(n)), "lt_reserve")

    def sync(self):
        _check(lib().lt_sync(self._h), "lt_sync")

    def set_option(self, option, value):
        _check(lib().lt_set_option(self._h, option, value), "lt_set_option")

    def timings(self):
        out = (C.c_float * 8)()
        _check(lib().lt_timings(self._h, out), "lt_timings")
        return dict(adapt=out[0], balance=out[1], connect=out[2], transfer=out[3], k_map=out[4], k_transfer=out[5],
                    k_connect=out[6], k_mortar=out[7])

    def launch_count(self) -> int:
        return int(lib().lt_launch_count(self._h))

    def balance_phases(self):
        out = (C.c_float * 4)()
        _check(lib().lt_balance_phases(self._h, out), "lt_balance_phases")
        return dict(examine=out[0], offsets=out[1], split=out[2], map=out[3])

    def host_syncs(self) -> int:
        return int(lib().lt_host_syncs(self._h))


def build(dim, base_level, max_level, domain=None, periodic=None) -> Tree:
    """lt_build"""
    return Tree(dim, base_level, max_level, domain, periodic)


def build_brick(dim, nroot, base_level, max_level, domain=None, periodic=None) -> Tree:
    """lt_build_brick: a forest on nroot[0] x nroot[1] (x nroot[2]) root cubes."""
    return Tree(dim, base_level, max_level, domain, periodic, nroot=nroot)


def build_from_keys(dim, base_level, max_level, keys, domain=None, periodic=None) -> Tree:
    """lt_build_from_keys: keys = int64 CUDA tensor holding the uint64 IDs."""
    return Tree(dim, base_level, max_level, domain, periodic, keys=keys)


def build_complete_from_keys(dim, base_level, max_level, keys, domain=None, periodic=None) -> Tree:
    """lt_build_complete_from_keys (Alg. 2 on octants): keys = int64 CUDA tensor of uint64 IDs."""
    return Tree(dim, base_level, max_level, domain, periodic, keys=keys, complete=True)


def build_from_points(dim, base_level, max_level, points, domain, periodic=None) -> Tree:
    """lt_build_from_points (Alg. 2): points = float64 CUDA tensor [n, dim]."""
    return Tree(dim, base_level, max_level, domain, periodic, points=points)


def encode(dim, max_level, xyz: torch.Tensor, level: torch.Tensor) -> torch.Tensor:
    """lt_encode: xyz int32 [n,3], level int32 [n] (CUDA) -> keys int64 [n]."""
    n = level.numel()
    keys = torch.empty(n, dtype=torch.int64, device=level.device)
    _check(lib().lt_encode(dim, max_level, _dptr(xyz, torch.int32, "xyz"), _dptr(level, torch.int32, "level"), n,
                           C.c_void_p(keys.data_ptr()), _stream_ptr(level.device)), "lt_encode")
    return keys


def decode(dim, max_level, keys: torch.Tensor):
    """lt_decode: keys int64 [n] (CUDA) -> (level int32 [n], xyz int32 [n,3])."""
    n = keys.numel()
    lvl = torch.empty(n, dtype=torch.int32, device=keys.device)
    xyz = torch.empty((n, 3), dtype=torch.int32, device=keys.device)
    _check(lib().lt_decode(dim, max_level, _dptr(keys, torch.int64, "keys"), n, C.c_void_p(lvl.data_ptr()),
                           C.c_void_p(xyz.data_ptr()), _stream_ptr(keys.device)), "lt_decode")
    return lvl, xyz


def sort_keys(dim, max_level, keys: torch.Tensor, linearise=False) -> torch.Tensor:
    """lt_sort_keys: returns the sorted (and optionally linearised) copy of `keys`."""
    k = keys.clone().contiguous()
    n_out = C.c_int64(0)
    _check(lib().lt_sort_keys(dim, max_level, _dptr(k, torch.int64, "keys"), k.numel(), int(bool(linearise)),
                              C.byref(n_out), _stream_ptr(k.device)), "lt_sort_keys")
    return k[: n_out.value]


SORT_STATIC_MAX_KEYS = 1 << 20  # LT_SORT_STATIC_MAX_KEYS of include/lt.h


def sort_keys_static_(dim, max_level, keys: torch.Tensor) -> None:
    """lt_sort_keys_static: sorts `keys` (contiguous int64 device tensor, at most SORT_STATIC_MAX_KEYS) IN
    PLACE with the library's static scratch: no allocation here or in the library; asynchronous on the
    current stream.  Calls that overlap on the GPU race (one shared scratch array per GPU)."""
    if not keys.is_contiguous():
        raise ValueError("lt_sort_keys_static: keys must be contiguous")
    _check(lib().lt_sort_keys_static(dim, max_level, _dptr(keys, torch.int64, "keys"), keys.numel(),
                                     _stream_ptr(keys.device)), "lt_sort_keys_static")
