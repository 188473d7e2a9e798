"""Seeded synthetic inputs for the h-adaptation cycle (flags and solution values).

This module serves BOTH the CPU oracle (tests) and the CUDA library (tests, bench)
and therefore holds none of the method's arithmetic: no Morton codes, no tree
operations, no transfer operators.  It sees leaves only as integer boxes
``level[M]`` and ``xyz[M,3]`` (anchor in units of the finest cell), which each side
obtains from its own decoder, and it returns ``int8`` flags / ``float64`` values.
Everything is plain ``torch`` tensor algebra, so it runs on CPU tensors (tests) and
on CUDA tensors (bench) alike.

Recipes follow BASELINE.json's five configs with the readings of DESIGN.md
("Input recipe"): the paper's workload is the isentropic vortex of PAPER.md:344-347
(Eq. 21; alpha = 5, phi = 1/2); BASELINE.json replaces the paper's point-counting
criterion by thresholds on the analytic vorticity magnitude.
"""
from __future__ import annotations

import math

import numpy as np
import torch

# name -> recipe.  "cN" is BASELINE.json configs[N-1]; c3b is the supplementary
# ripple stress of SURVEY.md 8(c).
CONFIGS = {
    "c1": dict(dim=2, base=3, maxl=8, lo=0.0, hi=1.0, periodic=(0, 0), cycles=4, p=2, nvars=4,
               flags="disc", seed=0, rand_refine=0.05, rand_coarsen=0.0, u0="random"),
    "c2": dict(dim=2, base=7, maxl=11, lo=-10.0, hi=10.0, periodic=(1, 1), cycles=50, p=3, nvars=4,
               flags="vortex", seed=0, rand_refine=0.0, rand_coarsen=0.0, u0="vortex"),
    "c3": dict(dim=3, base=3, maxl=12, lo=0.0, hi=1.0, periodic=(0, 0, 0), cycles=18, p=1, nvars=5,
               flags="point", point=(1e-6, 1e-6, 1e-6), seed=1, rand_refine=0.0, rand_coarsen=0.0,
               u0="random"),
    "c3b": dict(dim=3, base=3, maxl=12, lo=0.0, hi=1.0, periodic=(0, 0, 0), cycles=18, p=1, nvars=5,
                flags="point", point=(0.5 - 1e-6, 0.5 - 1e-6, 0.5 - 1e-6), seed=1, rand_refine=0.0,
                rand_coarsen=0.0, u0="random"),
    "c4": dict(dim=3, base=5, maxl=8, lo=-10.0, hi=10.0, periodic=(1, 1, 1), cycles=20, p=2, nvars=5,
               flags="vortex", seed=0, rand_refine=0.0, rand_coarsen=0.0, u0="vortex"),
    "c5": dict(dim=3, base=6, maxl=9, lo=-10.0, hi=10.0, periodic=(1, 1, 1), cycles=10, p=3, nvars=5,
               flags="vortex", seed=2, rand_refine=0.10, rand_coarsen=0.10, u0="vortex"),
    # The paper's own 3-D domain (Table 5): the slab [-12.5, 12.5]^2 x [0, 1.5625], one element
    # thick at D_min = 4 -- a brick of 16 x 16 x 1 root cubes of edge 1.5625 (lt_build_brick), levels counted
    # from the cubes: max level +4 = the paper's D_max 8 (dx_min = 25/256).  Flags: config 4's vortex-tube
    # recipe.  "lo" is per axis, "cube" the edge of a root cube; hi = lo + nroot * cube.
    "slab": dict(dim=3, nroot=(16, 16, 1), base=0, maxl=4, lo=(-12.5, -12.5, 0.0), cube=1.5625, periodic=(1, 1, 1),
                 cycles=20, p=2, nvars=5, flags="vortex", seed=0, rand_refine=0.0, rand_coarsen=0.0, u0="vortex"),
}


def geometry(cfg: dict):
    """(lo[dim], cube edge, nroot[dim]) of a config: a single cube [lo, hi]^dim unless "nroot" is given."""
    dim = cfg["dim"]
    nroot = tuple(cfg.get("nroot", (1,) * dim))
    lo = cfg["lo"]
    lo = tuple(float(v) for v in lo) if isinstance(lo, (tuple, list)) else (float(lo),) * dim
    cube = float(cfg["cube"]) if "cube" in cfg else float(cfg["hi"]) - lo[0]
    return lo, cube, nroot


def domain(cfg: dict):
    """lo_x.., hi_x.. of the whole domain (the `domain` argument of lt_build / lt_build_brick)."""
    lo, cube, nroot = geometry(cfg)
    return list(lo) + [lo[a] + nroot[a] * cube for a in range(cfg["dim"])]

_M64 = (1 << 64) - 1


def _i64(v: int) -> int:
    """Python int -> two's-complement int64 value."""
    v &= _M64
    return v - (1 << 64) if v >= (1 << 63) else v


_C1 = _i64(0xBF58476D1CE4E5B9)
_C2 = _i64(0x94D049BB133111EB)
_GOLD = _i64(0x9E3779B97F4A7C15)


def _lsr(v: torch.Tensor, s: int) -> torch.Tensor:
    """Logical right shift of int64 tensors."""
    return (v >> s) & ((1 << (64 - s)) - 1)


def _mix(v: torch.Tensor) -> torch.Tensor:
    """splitmix64 finaliser on int64 tensors (wrapping arithmetic)."""
    v = (v ^ _lsr(v, 30)) * _C1
    v = (v ^ _lsr(v, 27)) * _C2
    return v ^ _lsr(v, 31)


def counter_uniform(seed: int, stream: int, *ints: torch.Tensor) -> torch.Tensor:
    """Counter-based uniform [0,1) float64 from (seed, stream, integer tensors...).

    Order- and device-independent: the value depends only on the integers."""
    h = None
    for t in ints:
        t = t.to(torch.int64)
        if h is None:
            h = torch.full_like(t, _i64(seed * 0x9E3779B97F4A7C15 + stream * 0xD1B54A32D192ED03 + 0x2545F4914F6CDD1D))
            h = _mix(h)
        h = _mix((h + _GOLD) ^ t)
    return _lsr(h, 11).to(torch.float64) * (1.0 / 9007199254740992.0)


def centres(cfg: dict, level: torch.Tensor, xyz: torch.Tensor) -> torch.Tensor:
    """Leaf centres [M,dim] float64: lo + (x + w/2) (hi-lo)/2^Dmax, w = 2^(Dmax-level)."""
    dim, maxl = cfg["dim"], cfg["maxl"]
    lo, cube, _ = geometry(cfg)
    w = torch.pow(2.0, (maxl - level.to(torch.int64)).to(torch.float64))
    scale = cube / float(1 << maxl)
    lo_t = torch.tensor(lo, dtype=torch.float64, device=level.device)
    return lo_t[None, :] + (xyz[:, :dim].to(torch.float64) + 0.5 * w[:, None]) * scale


def _min_image(d: torch.Tensor, period: float) -> torch.Tensor:
    return d - period * torch.round(d / period)


def _vortex_w(cfg: dict, cycle: int, pos: torch.Tensor) -> torch.Tensor:
    """Relative vorticity magnitude |1 - r^2/2| exp(-r^2/2) of the vortex of Eq. 21
    (tube along z in 3-D) centred at (0.2 c, 0.2 c), minimum-image distance."""
    _, cube, nroot = geometry(cfg)
    dx = pos[:, 0] - 0.2 * cycle
    dy = pos[:, 1] - 0.2 * cycle
    if cfg["periodic"][0]:
        dx = _min_image(dx, nroot[0] * cube)
    if cfg["periodic"][1]:
        dy = _min_image(dy, nroot[1] * cube)
    r2 = dx * dx + dy * dy
    return torch.abs(1.0 - 0.5 * r2) * torch.exp(-0.5 * r2)


def flags(name_or_cfg, cycle: int, level: torch.Tensor, xyz: torch.Tensor) -> torch.Tensor:
    """int8 adaptation flags (-1/0/+1) for one cycle of a config."""
    cfg = CONFIGS[name_or_cfg] if isinstance(name_or_cfg, str) else name_or_cfg
    dim, maxl = cfg["dim"], cfg["maxl"]
    lvl = level.to(torch.int64)
    X = xyz.to(torch.int64)
    M = lvl.shape[0]
    f = torch.zeros(M, dtype=torch.int8, device=lvl.device)
    kind = cfg["flags"]
    if kind == "disc":
        c = centres(cfg, level, xyz)
        d = torch.sqrt((c[:, 0] - (0.5 + 0.05 * cycle)) ** 2 + (c[:, 1] - 0.5) ** 2)
        f[d < 0.15] = 1
        f[d > 0.4] = -1
    elif kind == "vortex":
        w = _vortex_w(cfg, cycle, centres(cfg, level, xyz))
        f[w > 0.05] = 1
        f[w < 0.01] = -1
    elif kind == "point":
        half = cfg["cycles"] // 2
        if cycle < half:  # refine the leaf containing the point
            glo, gcube, _ = geometry(cfg)
            scale = float(1 << maxl) / gcube
            inside = torch.ones(M, dtype=torch.bool, device=lvl.device)
            wd = torch.ones_like(lvl) << (maxl - lvl)
            for a in range(dim):
                pi = int(math.floor((cfg["point"][a] - glo[a]) * scale))
                inside &= (X[:, a] <= pi) & (pi < X[:, a] + wd)
            f[inside] = 1
        else:  # coarsen everything
            f[:] = -1
    else:
        raise ValueError(kind)
    if cfg["rand_refine"] > 0.0:
        u = counter_uniform(cfg["seed"], 2 * cycle, lvl, X[:, 0], X[:, 1], X[:, 2])
        f[u < cfg["rand_refine"]] = 1
    if cfg["rand_coarsen"] > 0.0:
        # one draw per sibling group: identified by the parent's box (level-1, anchor
        # with the bit of the own width cleared).  Result-equivalent to flagging only
        # complete groups, because adapt ignores incomplete / mixed groups.
        wd = torch.ones_like(lvl) << (maxl - lvl)
        par = X & ~(2 * wd[:, None] - 1)
        u = counter_uniform(cfg["seed"], 2 * cycle + 1, lvl - 1, par[:, 0], par[:, 1], par[:, 2])
        f[(u < cfg["rand_coarsen"]) & (f <= 0) & (lvl > 0)] = -1
    return f


def _gl_nodes(p: int) -> np.ndarray:
    return np.polynomial.legendre.leggauss(p + 1)[0]  # library routine; placement only


def initial_solution(name_or_cfg, level: torch.Tensor, xyz: torch.Tensor) -> torch.Tensor:
    """u0[M, nvars, N] float64 on the initial tree (N = (p+1)^dim, x fastest)."""
    cfg = CONFIGS[name_or_cfg] if isinstance(name_or_cfg, str) else name_or_cfg
    dim, maxl, p, nvars = cfg["dim"], cfg["maxl"], cfg["p"], cfg["nvars"]
    P1 = p + 1
    N = P1 ** dim
    lvl = level.to(torch.int64)
    X = xyz.to(torch.int64)
    M = lvl.shape[0]
    dev = lvl.device
    if cfg["u0"] == "random":
        v = torch.arange(nvars, device=dev, dtype=torch.int64)[None, :, None].expand(M, nvars, N)
        n = torch.arange(N, device=dev, dtype=torch.int64)[None, None, :].expand(M, nvars, N)
        e = lambda t: t[:, None, None].expand(M, nvars, N)
        u = counter_uniform(cfg["seed"], 1 << 20, e(lvl), e(X[:, 0]), e(X[:, 1]), e(X[:, 2]), v, n)
        return (2.0 * u - 1.0).contiguous()
    # analytic vortex, conserved variables at the solution points (SURVEY 8(d) relations)
    z = torch.as_tensor(_gl_nodes(p), dtype=torch.float64, device=dev)
    w = torch.pow(2.0, (maxl - lvl).to(torch.float64))
    glo, gcube, _ = geometry(cfg)
    scale = gcube / float(1 << maxl)
    idx = torch.arange(N, device=dev)
    pos = []
    for a in range(dim):
        ia = (idx // (P1 ** a)) % P1
        pos.append(glo[a] + (X[:, a].to(torch.float64)[:, None] + 0.5 * w[:, None] * (1.0 + z[ia][None, :])) * scale)
    alpha, phi, gamma = 5.0, 0.5, 1.4
    dx, dy = pos[0], pos[1]
    r2 = dx * dx + dy * dy
    e1 = torch.exp(phi * (1.0 - r2))
    du = -alpha / (2 * math.pi) * dy * e1
    dv = alpha / (2 * math.pi) * dx * e1
    dT = -(alpha ** 2) * (gamma - 1.0) / (16 * phi * gamma * math.pi ** 2) * e1 * e1
    cinf = math.sqrt(2.0) / 0.5
    pinf = 1.0 * cinf * cinf / gamma
    Tinf = pinf / 1.0
    T = Tinf + dT
    rho = torch.pow(T / Tinf, 1.0 / (gamma - 1.0))
    pr = rho * T
    uu, vv = 1.0 + du, 1.0 + dv
    E = pr / (gamma - 1.0) + 0.5 * rho * (uu * uu + vv * vv)
    comps = [rho, rho * uu, rho * vv]
    if dim == 3:
        comps.append(torch.zeros_like(rho))
    comps.append(E)
    out = torch.stack(comps[:nvars], dim=1)
    return out.contiguous()


# ---------------------------------------------------------------------------------------
# Scattered points for tree construction (Alg. 2).  The paper builds its
# construction / balance benchmark from the Stanford bunny surface, which is
# not available here; these seeded synthetic surfaces stand in for it.
POINT_CLOUDS = {
    # name: dim, base (the paper's D_min = 4), maxl, surface, points
    "pc_tiny": dict(dim=2, base=1, maxl=5, lo=0.0, hi=1.0, periodic=(0, 0), surface="sphere", n=40, seed=3),
    "pc2": dict(dim=2, base=2, maxl=9, lo=0.0, hi=1.0, periodic=(0, 0), surface="sphere", n=4000, seed=4),
    "pc3_small": dict(dim=3, base=2, maxl=6, lo=0.0, hi=1.0, periodic=(0, 0, 0), surface="torus", n=3000, seed=5),
    "pc9": dict(dim=3, base=4, maxl=9, lo=-1.0, hi=1.0, periodic=(0, 0, 0), surface="torus", n=4_000_000, seed=6),
    "pc10": dict(dim=3, base=4, maxl=10, lo=-1.0, hi=1.0, periodic=(0, 0, 0), surface="sphere", n=16_000_000,
                 seed=7),
}


def surface_points(cfg, device="cpu", n=None) -> torch.Tensor:
    """float64 [n, dim] points on a closed surface inside the domain: "sphere" (circle in 2-D)
    of radius 0.35 widths about the centre, or "torus" (major 0.30, minor 0.12 widths, axis z;
    2-D: an annulus boundary pair).  Drawn from the counter generator, so the cloud depends only
    on (seed, index).  Trigonometric results may differ in the last bit between devices: generate
    ONCE and hand the same bytes to both sides."""
    dim, lo, hi = cfg["dim"], cfg["lo"], cfg["hi"]
    n = int(cfg["n"] if n is None else n)
    i = torch.arange(n, dtype=torch.int64, device=device)
    u = counter_uniform(cfg["seed"], 11, i)
    v = counter_uniform(cfg["seed"], 12, i)
    w = hi - lo
    c = 0.5 * (lo + hi)
    two_pi = 2.0 * math.pi
    if dim == 2:
        r = 0.35 * w if cfg["surface"] == "sphere" else torch.where(v < 0.5, 0.18 * w, 0.42 * w)
        return torch.stack([c + r * torch.cos(two_pi * u), c + r * torch.sin(two_pi * u)], dim=1)
    if cfg["surface"] == "sphere":
        z = 2.0 * v - 1.0
        s = torch.sqrt(torch.clamp(1.0 - z * z, min=0.0))
        r = 0.35 * w
        return torch.stack([c + r * s * torch.cos(two_pi * u), c + r * s * torch.sin(two_pi * u), c + r * z], dim=1)
    R, r = 0.30 * w, 0.12 * w
    q = R + r * torch.cos(two_pi * v)
    return torch.stack([c + q * torch.cos(two_pi * u), c + q * torch.sin(two_pi * u),
                        c + r * torch.sin(two_pi * v)], dim=1)
