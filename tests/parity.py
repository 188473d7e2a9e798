"""Parity driver: runs the CPU oracle and the CUDA library side by side on the same seeded
inputs and compares every output of the cycle.

Flags are computed ONCE per cycle, on the host, from the oracle's leaf boxes and the same
byte array is given to both sides; the GPU's own decoder is
checked against the oracle's boxes separately.  Bit-exact: keys, balance iteration count,
nbr/kind, the three face tables, the Alg. 7 map.  Solution values: per variable
max|u_gpu - u_ref| <= 1e-12 * max(1, max|u_ref|) (BASELINE.json; reading E-8).
"""
import numpy as np
import torch

import oracle
from paper_2306_06744_b200 import lt
from paper_2306_06744_b200 import workloads as W

TOL = 1e-12


def u64(t):
    """int64 CUDA view of uint64 keys -> numpy uint64"""
    return t.cpu().numpy().view(np.uint64)


def assert_keys_equal(gt, ot, what=""):
    gk, ok = u64(gt.keys()), ot.keys()
    assert gk.shape == ok.shape, "%s: leaf count %d vs oracle %d" % (what, gk.size, ok.size)
    assert np.array_equal(gk, ok), "%s: keys differ at %s" % (what, np.nonzero(gk != ok)[0][:5])


def assert_faces_equal(Fg, Fo, what=""):
    for k in ("n_conf", "n_hang", "n_bnd"):
        assert int(Fg[k]) == int(Fo[k]), "%s: %s %d vs oracle %d" % (what, k, Fg[k], Fo[k])
    for k in ("nbr", "kind", "conf", "conf_axis", "hang", "hang_info", "bnd", "bnd_face"):
        a, b = Fg[k].cpu().numpy(), Fo[k]
        assert a.shape == b.shape, "%s: %s shape %s vs %s" % (what, k, a.shape, b.shape)
        assert np.array_equal(a, b), "%s: %s differs at %s" % (what, k, np.argwhere(a != b)[:5].tolist())


def assert_u_close(ug, uo, what=""):
    ug = ug.cpu().numpy()
    assert ug.shape == uo.shape, "%s: u shape %s vs %s" % (what, ug.shape, uo.shape)
    for v in range(uo.shape[1]):
        scale = max(1.0, float(np.max(np.abs(uo[:, v]))) if uo.size else 1.0)
        err = float(np.max(np.abs(ug[:, v] - uo[:, v]))) if uo.size else 0.0
        assert err <= TOL * scale, "%s: var %d error %.3e > %.1e * %.3g" % (what, v, err, TOL, scale)


def host_flags(cfg, cycle, ot):
    lvl, xyz = ot.leaf_boxes()
    return W.flags(cfg, cycle, torch.from_numpy(lvl), torch.from_numpy(xyz.astype(np.int64))).numpy()


def new_pair(cfg):
    """Both sides on the config's domain: one cube, or a brick of root cubes when cfg has "nroot"."""
    nroot = cfg.get("nroot")
    gt = lt.Tree(cfg["dim"], cfg["base"], cfg["maxl"], W.domain(cfg), cfg["periodic"], nroot=nroot)
    ot = oracle.Tree(cfg["dim"], cfg["base"], cfg["maxl"], cfg["periodic"], nroot=nroot)
    return gt, ot


def initial_u(cfg, ot):
    lvl, xyz = ot.leaf_boxes()
    return W.initial_solution(cfg, torch.from_numpy(lvl), torch.from_numpy(xyz.astype(np.int64))).numpy()


def run_cycles(cfg, ncycles, options=(), check_faces=True, check_transfer=True, drift_free=True, log=None,
               record=None):
    """Drive both sides through `ncycles` adaptation cycles of a workload config.
    log (list): one row per cycle (cycle, leaves out, balance sweeps, n_conf, n_hang, n_bnd, leaves in) -- the
    ORACLE's numbers (the GPU's were asserted equal).  record (list): per cycle (flags, oracle keys after
    balance, sweeps), for GPU-only replays with other options."""
    gt, ot = new_pair(cfg)
    for opt, val in options:
        gt.set_option(opt, val)
    assert_keys_equal(gt, ot, "build")
    p, nvars = cfg["p"], cfg["nvars"]
    uo = initial_u(cfg, ot)
    ug = torch.from_numpy(uo).cuda()
    for c in range(ncycles):
        tag = "cycle %d" % c
        # the GPU's own decoder must give the boxes the flags are computed from
        glvl, gxyz = gt.leaf_boxes()
        olvl, oxyz = ot.leaf_boxes()
        assert np.array_equal(glvl.cpu().numpy(), olvl) and np.array_equal(gxyz.cpu().numpy().astype(np.uint32), oxyz)
        f = host_flags(cfg, c, ot)
        n_in = ot.num_leaves()
        ot.adapt(f)
        gt.adapt(torch.from_numpy(f).cuda())
        assert_keys_equal(gt, ot, tag + " adapt")
        assert np.array_equal(u64(gt.old_keys()), ot.old_keys()), tag + " snapshot"
        it_o = ot.balance()
        it_g = gt.balance()
        assert_keys_equal(gt, ot, tag + " balance")
        assert it_g == it_o, "%s: balance iters %d vs oracle %d" % (tag, it_g, it_o)
        counts = (-1, -1, -1)
        if check_faces:
            Fo = ot.connect()
            assert_faces_equal(gt.connect(), Fo, tag + " connect")
            counts = (Fo["n_conf"], Fo["n_hang"], Fo["n_bnd"])
        if record is not None:
            record.append((f, ot.keys(), it_o))
        if check_transfer:
            src_o, kind_o = ot.build_map()
            un_o = ot.transfer_rows(uo, p, nvars, 0, ot.num_leaves())
            ot.drop_snapshot()
            un_g = gt.transfer(ug, p, nvars)
            gt.sync()
            src_g, kind_g = gt.map()
            assert np.array_equal(src_g.cpu().numpy(), src_o), tag + " map src"
            assert np.array_equal(kind_g.cpu().numpy(), kind_o), tag + " map kind"
            assert_u_close(un_g, un_o, tag + " transfer")
            uo = un_o
            # drift_free: feed the GPU the oracle's values next cycle (reading E-8)
            ug = torch.from_numpy(uo).cuda() if drift_free else un_g
        else:
            ot.drop_snapshot()
        if log is not None:
            log.append((c, ot.num_leaves(), it_o) + counts + (n_in,))
    return gt, ot, ug, uo


def replay_gpu(cfg, record, options=()):
    """GPU only: drive a fresh tree through the recorded flags with `options` set and compare keys and
    sweep counts with the recorded (oracle) ones -- options must not change results."""
    gt = lt.Tree(cfg["dim"], cfg["base"], cfg["maxl"], W.domain(cfg), cfg["periodic"], nroot=cfg.get("nroot"))
    for opt, val in options:
        gt.set_option(opt, val)
    for c, (f, keys, iters) in enumerate(record):
        gt.adapt(torch.from_numpy(f).cuda())
        it = gt.balance()
        assert it == iters, "replay cycle %d: balance sweeps %d vs %d" % (c, it, iters)
        gk = u64(gt.keys())
        assert gk.shape == keys.shape and np.array_equal(gk, keys), "replay cycle %d: keys differ" % c
    return gt
