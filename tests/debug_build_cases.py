"""Run by tests/test_gpu_debug_build.py in a subprocess with LT_DEBUG_LIB=1: small cases of every
kernel family through the checked build (liblt_debug.so), compared with the oracle as usual.  Any
device-side assertion traps the kernel and fails the run."""
import os
import sys

import numpy as np
import torch

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(HERE))
sys.path.insert(0, HERE)

import oracle  # noqa: E402
import parity as P  # noqa: E402
from paper_2306_06744_b200 import lt  # noqa: E402
from paper_2306_06744_b200 import workloads as W  # noqa: E402

assert lt.lib().lt_debug_build() == 1, "the checked build was not loaded"

# whole cycles: config 1, the ripple stress 3b (incl. coarsening back), a small brick
P.run_cycles(W.CONFIGS["c1"], 4)
P.run_cycles(W.CONFIGS["c3b"], 18)
P.run_cycles(dict(W.CONFIGS["slab"], nroot=(4, 3, 1), maxl=3), 6)
# strong balance and the paper's append-sort-linearise adapt
P.run_cycles(W.CONFIGS["c1"], 4, options=[(lt.LT_OPT_ADAPT_SORT, 1)])
cfg = W.CONFIGS["c3b"]
gt, ot = P.new_pair(cfg)
gt.set_option(lt.LT_OPT_BALANCE_CONNECTIVITY, 2)
for c in range(9):
    f = P.host_flags(cfg, c, ot)
    ot.adapt(f); gt.adapt(torch.from_numpy(f).cuda())
    assert gt.balance() == ot.balance(2)
    P.assert_keys_equal(gt, ot, "strong balance")
    ot.drop_snapshot()
# the deferred 10-sweep ripple, full sweeps
gt, ot = P.new_pair(cfg)
for c in range(9):
    f = P.host_flags(cfg, c, ot)
    ot.adapt(f); gt.adapt(torch.from_numpy(f).cuda())
assert gt.balance() == ot.balance() == 10
P.assert_faces_equal(gt.connect(), ot.connect(), "deferred ripple faces")
# the one-synchronisation cycle
cfg = W.CONFIGS["c1"]
gt, ot = P.new_pair(cfg)
gt.reserve(1 << 14)
uo = P.initial_u(cfg, ot)
for c in range(4):
    f = P.host_flags(cfg, c, ot)
    d_un = torch.empty((1 << 14, cfg["nvars"], 9), dtype=torch.float64, device="cuda")
    gt.adapt(torch.from_numpy(f).cuda())
    gt.balance(want_iters=False)
    gt.connect_begin()
    gt.transfer_into(torch.from_numpy(uo).cuda(), d_un, cfg["p"], cfg["nvars"])
    Fg = gt.connect_end()
    ot.adapt(f); ot.balance()
    P.assert_faces_equal(Fg, ot.connect(), "one-sync cycle")
    uo = ot.transfer(uo, cfg["p"], cfg["nvars"])
    gt.sync()
    P.assert_u_close(d_un[:ot.num_leaves()], uo, "one-sync transfer")
# construction from points (radix sort, linearise, completion), balance, faces
for name in ("pc_tiny", "pc3_small"):
    pc = W.POINT_CLOUDS[name]
    dim = pc["dim"]
    dom = [pc["lo"]] * dim + [pc["hi"]] * dim
    pts = W.surface_points(pc).numpy()
    ot = oracle.Tree(dim, pc["base"], pc["maxl"], pc["periodic"], points=pts, domain=dom)
    gt = lt.build_from_points(dim, pc["base"], pc["maxl"], torch.from_numpy(pts).cuda(), dom, pc["periodic"])
    P.assert_keys_equal(gt, ot, name)
    assert gt.balance() == ot.balance()
    P.assert_faces_equal(gt.connect(), ot.connect(), name + " faces")
# the sort on adversarial inputs spanning several tiles and a ragged tail
rng = np.random.default_rng(0)
for keys in (rng.integers(0, 1 << 40, 10000), np.zeros(5000, np.int64), np.arange(9000, 0, -1)):
    k = torch.from_numpy(keys.astype(np.int64)).cuda()
    got = lt.sort_keys(3, 12, k).cpu().numpy()
    assert np.array_equal(got, np.sort(keys.astype(np.int64)))
# mortars + one FR stage on an adapted mesh with hanging faces
from test_gpu_mortar import adapted_pair  # noqa: E402
gt, ot, rng = adapted_pair(3, (1, 1, 1), 5, 2, 4, cycles=2)
gt.connect(); ot.connect()
p, nv = 2, 5
M = ot.num_leaves()
u = np.tile(np.array([1.0, 0.3, -0.2, 0.1, 2.5])[None, :, None], (M, 1, 27)) * (1.0 + 0.05 * rng.uniform(-1, 1, (M, 1, 27)))
uf_o = ot.face_interp(u, p, nv)
fs_o = ot.common_flux(uf_o, ot.mortar_project(uf_o, p, nv), p)
fs_o = np.where(np.isnan(fs_o), ot.mortar_gather(fs_o, p, nv), fs_o)
d_u = torch.from_numpy(u).cuda()
uf = gt.face_interp(d_u, p, nv)
fs = gt.common_flux(uf, gt.mortar_project(uf, p, nv), p)
gt.mortar_gather(fs, p, nv, f_face=fs)
assert float(np.abs(fs.cpu().numpy() - fs_o).max()) < 1e-11
R_o = ot.fr_rhs(u, fs_o, p, [1.0] * 3)
out = gt.fr_stage(1, 1e-3, d_u, d_u, fs, p).cpu().numpy()
assert float(np.abs(out - (u + 1e-3 * R_o)).max()) < 1e-12 * max(1.0, float(np.abs(R_o).max()))
gt.sync()
torch.cuda.synchronize()
print("debug build cases ok")
