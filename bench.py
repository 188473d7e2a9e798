#!/usr/bin/env python
"""bench.py -- throughput of the h-adaptation cycle (adapt + 2:1 balance + connectivity +
FR transfer) on BASELINE.json's throughput config (configs[4], "c5": 3-D octree, periodic
[-10,10]^3, base 64^3, max level +3, vortex-tube flags + 10 % random refine / group coarsen,
p = 3, 5 fp64 variables).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

A step is one adaptation cycle of the whole hot path through the C ABI (lt_adapt,
lt_balance, lt_connect, lt_transfer).  The tree is first brought, untimed, to the state
after config-5 cycles 0-2 (8.86 M leaves); steps then run cycles 3, 4, 5 (13.5 M, 18.9 M,
26.1 M leaves out), rewinding to the prepared state after cycle 5 because from cycle 7 on
u_old + u_new no longer fit 180 GB.  Prints ONE JSON line.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "leaves/s per full adapt+2:1 balance+connectivity+transfer cycle"
UNIT = "leaves/s"
CONFIG = "c5"             # --config: c5 is the bench line; c1 / c2 / c4 are secondary lines
PREP_CYCLES = 3           # config-5 cycles 0..2 run untimed to develop the tree
OVERLAP = True            # --no-overlap: lt_connect then lt_transfer instead of begin / transfer / end
CONNECTIVITY = 1          # --connectivity: 1 face balance (BASELINE.json), 2 the paper's strong balance
PERIOD = (3, 4, 5)        # config-5 cycles a step runs (--cycles a,b,.. overrides: profiling aid)
FALLBACK_HBM_GBS = 6650.0  # /opt/skills/guides/B200_PROFILING.md fallback

# untimed preparation cycles and the cycles the steps run through, per config: c5 cannot run its 10 stated
# cycles (reading F-2); the small configs run ALL their stated cycles from the uniform tree, one step each
SCHEDULES = {"c5": (3, (3, 4, 5)), "c1": (0, tuple(range(4))), "c2": (0, tuple(range(50))),
             "c4": (0, tuple(range(20))), "slab": (0, tuple(range(20)))}
WORKLOADS = {
    "c5": "c5 (BASELINE.json configs[4]): 3D octree, periodic [-10,10]^3, base 64^3, max level +3, vortex-tube flags + "
          "10% random refine / 10% random group coarsen (seed 2), p=3 (64 solution points), 5 fp64 vars",
    "c1": "c1 (BASELINE.json configs[0]): 2D quadtree, [0,1]^2 non-periodic, base 8^2, max level 8, moving-disc flags + "
          "5% random refine (seed 0), 4 cycles, p=2, 4 fp64 vars",
    "c2": "c2 (BASELINE.json configs[1]): 2D quadtree, periodic [-10,10]^2, base 128^2, max level +4, isentropic-vortex "
          "flags, 50 cycles, p=3, 4 fp64 vars",
    "c4": "c4 (BASELINE.json configs[3]): 3D octree, periodic [-10,10]^3, base 32^3, max level +3, vortex-tube flags, "
          "20 cycles, p=2, 5 fp64 vars",
    "slab": "slab (the paper's own 3-D domain, PAPER.md:410 / Table 5): periodic [-12.5,12.5]^2 x [0,1.5625] as a brick of "
            "16 x 16 x 1 root cubes (lt_build_brick), max level +4 (the paper's D_max 8), config 4's vortex-tube flags, "
            "20 cycles, p=2, 5 fp64 vars",
}


def hbm_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        v = float(json.load(open(p))["hbm_gbs"])
        return v, "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc, self.thr = index, [], None, None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None
            return
        self.thr = threading.Thread(target=self._read, daemon=True)
        self.thr.start()

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx = float(r[1])
            except Exception:
                continue
            for nm, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm)}


def mem_available_bytes():
    try:
        for line in open("/proc/meminfo"):
            if line.startswith("MemAvailable"):
                return int(line.split()[1]) * 1024
    except Exception:
        pass
    return 16 << 30


# --------------------------------------------------------------------------- oracle legs
def cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except Exception:
        pass
    return "unknown"


class PinnedThread:
    """The oracle is sequential: pin this process to ONE of its allowed cores while it is timed."""

    def __enter__(self):
        self.old = None
        try:
            self.old = os.sched_getaffinity(0)
            self.cpu = max(self.old)
            os.sched_setaffinity(0, {self.cpu})
        except Exception:
            self.cpu = None
        return self

    def __exit__(self, *exc):
        if self.old:
            try:
                os.sched_setaffinity(0, self.old)
            except Exception:
                pass


def oracle_cycles(cfg, cycles, transfer_fraction=1.0):
    """The oracle, as it stands, on cycles 0..cycles-1 of a config; only its four calls are timed (flag
    and solution generation are the harness's).  transfer_fraction < 1: the transfer of a cycle is
    timed on evenly spaced slabs covering that fraction of the new elements and scaled (config 5's deep
    cycles: a dense M^-1 S_c per element is minutes of host time); tree, balance, faces and the map are
    always timed in full.  Returns a list of per-cycle dicts."""
    import numpy as np
    import torch
    import oracle
    from paper_2306_06744_b200 import workloads as W
    p, nvars = cfg["p"], cfg["nvars"]
    ot = oracle.Tree(cfg["dim"], cfg["base"], cfg["maxl"], cfg["periodic"], nroot=cfg.get("nroot"))
    lvl, xyz = ot.leaf_boxes()
    L, X = torch.from_numpy(lvl), torch.from_numpy(xyz.astype(np.int64))
    full = transfer_fraction >= 1.0
    uo = W.initial_solution(cfg, L, X).numpy() if full else None
    rows = []
    for c in range(cycles):
        f = W.flags(cfg, c, L, X).numpy()
        m0 = ot.num_leaves()
        t0 = time.perf_counter()
        ot.adapt(f)
        t1 = time.perf_counter()
        it = ot.balance()
        t2 = time.perf_counter()
        F = ot.connect()
        t3 = time.perf_counter()
        m1 = ot.num_leaves()
        scaled = False
        if full:
            uo = ot.transfer(uo, p, nvars)
            t4 = time.perf_counter()
            t_tr = t4 - t3
        else:
            src, kind = ot.build_map()
            t_map = time.perf_counter() - t3
            slab = 4096
            nslab = max(1, int(transfer_fraction * m1 / slab))
            starts = np.linspace(0, max(0, m1 - slab), nslab).astype(np.int64)
            t_rows, n_rows = 0.0, 0
            for j0 in starts:
                j1 = min(m1, int(j0) + slab)
                lo = int(src[j0:j1].min())
                hi = min(m0, int(src[j0:j1].max()) + (1 << cfg["dim"]))
                win = W.initial_solution(cfg, L[lo:hi], X[lo:hi]).numpy()   # analytic old values, untimed
                ta = time.perf_counter()
                ot.transfer_rows(win, p, nvars, int(j0), j1, old_offset=lo)
                t_rows += time.perf_counter() - ta
                n_rows += j1 - int(j0)
            ot.drop_snapshot()
            t_tr = t_map + t_rows * (m1 / max(n_rows, 1))
            scaled = n_rows < m1
        lvl, xyz = ot.leaf_boxes()
        L, X = torch.from_numpy(lvl), torch.from_numpy(xyz.astype(np.int64))
        rows.append(dict(cycle=c, M0=m0, M1=m1, iters=it, faces=F["n_conf"] + F["n_hang"] + F["n_bnd"],
                         adapt=t1 - t0, balance=t2 - t1, connect=t3 - t2, transfer=t_tr,
                         seconds=(t3 - t0) + t_tr, transfer_scaled=scaled))
        del F
    return rows


# default (bounded, 3-30 s of host time) and --oracle-full samples of the cpu_baseline per config
ORACLE_SAMPLES = {"c5": (1, 1.0, 4, 0.02), "c1": (4, 1.0, 4, 1.0), "c2": (12, 1.0, 50, 1.0), "c4": (3, 1.0, 20, 1.0),
                  "slab": (20, 1.0, 20, 1.0)}


def cpu_baseline(name, cfg, full=False):
    cyc, frac, cyc_full, frac_full = ORACLE_SAMPLES[name]
    if full:
        cyc, frac = cyc_full, frac_full
    with PinnedThread() as pin:
        rows = oracle_cycles(cfg, cyc, frac)
    secs = sum(r["seconds"] for r in rows)
    leaves = sum(r["M1"] for r in rows)
    sample = "%s cycle%s 0%s in full (%d -> %d leaves, p=%d, %d vars): adapt+balance+connect+transfer" % (
        name, "s" if cyc > 1 else "", "-%d" % (cyc - 1) if cyc > 1 else "", rows[0]["M0"], rows[-1]["M1"], cfg["p"],
        cfg["nvars"])
    if frac < 1.0:
        sample += "; transfer timed on slabs covering %.0f %% of the new elements and scaled" % (100 * frac)
    return {"value": leaves / secs, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample, "seconds": secs,
            "faces_per_s": sum(r["faces"] for r in rows) / sum(r["connect"] for r in rows),
            "seconds_per_call": {k: sum(r[k] for r in rows) for k in ("adapt", "balance", "connect", "transfer")},
            "pinned_to_cpu": pin.cpu, "cpu_model": cpu_model(), "host_cores_available": os.cpu_count(),
            "which": "oracle-full" if full else "default (bounded)"}


def profile_traffic(kernel):
    """(DRAM bytes per launch under ncu, algorithmic bytes of that launch) of a kernel, from
    profiles/traffic.txt ("<kernel> <dram bytes> <algorithmic bytes>"), or (None, None)."""
    try:
        for line in open(os.path.join(ROOT, "profiles", "traffic.txt")):
            w = line.split()
            if len(w) >= 3 and w[0] == kernel:
                return int(w[1]), int(w[2])
    except Exception:
        pass
    return None, None


def oracle_solver_share(name="slab", prep=8):
    """cpu_baseline of --workload solver: the oracle, as it stands, on the paper's own 3-D domain (the slab
    config: 16 x 16 x 1 root cubes, p = 2): cycles 0..prep-1 replayed untimed, cycle `prep` timed in full
    (adapt, balance, connect, transfer), then ONE SSP-RK3 step (three times Alg. 8 steps 1-4, Eq. 2-5 and
    Eq. 6) timed on the adapted mesh and counted ten times -- the same metric, the adaptation share of
    wall clock at one adaptation per ten steps."""
    import numpy as np
    import torch
    import oracle
    from paper_2306_06744_b200 import workloads as W
    cfg = W.CONFIGS[name]
    p, nvars = cfg["p"], cfg["nvars"]
    lo, cube, nroot = W.geometry(cfg)
    width = [cube * n for n in nroot]
    with PinnedThread() as pin:
        ot = oracle.Tree(cfg["dim"], cfg["base"], cfg["maxl"], cfg["periodic"], nroot=cfg.get("nroot"))
        for c in range(prep + 1):
            lvl, xyz = ot.leaf_boxes()
            L, X = torch.from_numpy(lvl), torch.from_numpy(xyz.astype(np.int64))
            f = W.flags(cfg, c, L, X).numpy()
            if c < prep:
                ot.adapt(f); ot.balance(); ot.drop_snapshot()
                continue
            u = W.initial_solution(cfg, L, X).numpy()
            m0 = ot.num_leaves()
            t0 = time.perf_counter()
            ot.adapt(f); ot.balance(); ot.connect()
            u = ot.transfer(u, p, nvars)
            t_adapt = time.perf_counter() - t0
        m1 = ot.num_leaves()
        dt = 5e-4

        def rhs(x):
            uf = ot.face_interp(x, p, nvars)
            fs = ot.common_flux(uf, ot.mortar_project(uf, p, nvars), p)
            fs = np.where(np.isnan(fs), ot.mortar_gather(fs, p, nvars), fs)
            return ot.fr_rhs(x, fs, p, width)
        t0 = time.perf_counter()
        u1 = oracle.rk3_stage(1, dt, u, u, rhs(u))
        u2 = oracle.rk3_stage(2, dt, u, u1, rhs(u1))
        u3 = oracle.rk3_stage(3, dt, u, u2, rhs(u2))
        t_step = time.perf_counter() - t0
        assert np.isfinite(u3).all()
    return {"value": t_adapt / (t_adapt + 10 * t_step), "unit": "fraction", "cores": 1, "kind": "oracle",
            "sample": "%s cycle %d in full (%d -> %d elements, p=%d) + one SSP-RK3 step timed and counted ten times"
                      % (name, prep, m0, m1, p),
            "seconds": t_adapt + t_step, "seconds_per_call": {"adaptation_cycle": t_adapt, "one_rk3_step": t_step},
            "elements_per_s_rhs": 3 * m1 / t_step, "pinned_to_cpu": pin.cpu, "cpu_model": cpu_model(),
            "host_cores_available": os.cpu_count()}


def run_reference(args):
    """--impl reference: the CPU oracle timed on the box's host cores (tier rule 4), one pinned thread,
    on the sample of --config's workload that cpu_baseline() names; a step = that sample once."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_2306_06744_b200 import workloads as W
    cfg = W.CONFIGS[CONFIG]
    for _ in range(args.warmup):
        cpu_baseline(CONFIG, cfg, args.oracle_full)
    leaves, secs, last = 0, 0.0, None
    for _ in range(args.steps):
        last = cpu_baseline(CONFIG, cfg, args.oracle_full)
        leaves += last["value"] * last["seconds"]
        secs += last["seconds"]
    value = leaves / secs
    out = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * secs / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOADS[CONFIG], "step": last["sample"]},
        "cpu_baseline": dict(last, value=value),
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(out), flush=True)


# --------------------------------------------------------------------------- the CUDA arm
class Runner:
    def __init__(self, cfg, device):
        import torch
        from paper_2306_06744_b200 import lt
        from paper_2306_06744_b200 import workloads as W
        self.torch, self.lt, self.W, self.cfg, self.dev = torch, lt, W, cfg, device
        self.p, self.nvars = cfg["p"], cfg["nvars"]
        self.N = (self.p + 1) ** cfg["dim"]
        self.Bu = 8 * self.nvars * self.N
        self.tree = None

    def flags(self, c):
        lvl, xyz = self.tree.leaf_boxes()
        return self.W.flags(self.cfg, c, lvl, xyz)

    def prepare(self, reserve=None):
        """Uniform base tree, then config-5 cycles 0..PREP_CYCLES-1 (tree only, untimed)."""
        cfg = self.cfg
        if self.tree is not None:
            self.tree.free()
        self.tree = self.lt.Tree(cfg["dim"], cfg["base"], cfg["maxl"], self.W.domain(cfg), cfg["periodic"],
                                 nroot=cfg.get("nroot"))
        if reserve:
            self.tree.reserve(reserve)
        if CONNECTIVITY != 1:
            self.tree.set_option(self.lt.LT_OPT_BALANCE_CONNECTIVITY, CONNECTIVITY)
        for c in range(PREP_CYCLES):
            self.tree.adapt(self.flags(c))
            self.tree.balance()
        return self.tree.num_leaves()

    def analytic_u(self, out):
        """Conserved variables of the analytic vortex at the solution points of the current
        tree, written into out[:M] slab by slab (bounded temporaries)."""
        lvl, xyz = self.tree.leaf_boxes()
        M = lvl.shape[0]
        step = 1 << 20
        for a in range(0, M, step):
            b = min(a + step, M)
            out[a:b] = self.W.initial_solution(self.cfg, lvl[a:b], xyz[a:b])
        return M


def max_over_ranks(ms, world, device):
    """Timing rule for N > 1: the slowest rank's device time (all-reduce MAX)."""
    if world <= 1:
        return float(ms)
    import torch
    import torch.distributed as dist
    tt = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    return float(tt.item())


def whole_job_value(leaves_per_rank, world, ms):
    """Replicas only: every rank runs the same independent workload,
    so the job processed world * leaves in the slowest rank's time."""
    return world * leaves_per_rank / (ms * 1e-3)


def algorithmic_bytes(dim, M0, Ma, M1, n_faces3, Bu, iters=1):
    """SURVEY.md 8(d) minimal bytes of the kernels actually run (path B), per cycle:
    adapt    two passes over key + flag (count, scatter), keys out;
    balance  every splitting sweep reads key + mark of every leaf and writes the new keys (leaf count taken
             as the mean of Ma and M1), the closing sweep only examines the frontier (not counted);
    map      Alg. 7, run in the tail of the balance kernel: old and new keys in, src + kind out;
    connect  keys in, nbr + kind and the three face tables out;
    transfer every old element read once, every new element written once, the map read once."""
    nf = 2 * dim
    n_conf, n_hang, n_bnd = n_faces3
    adapt = 2 * 9 * M0 + 8 * Ma
    balance = iters * (9 + 8) * (Ma + M1) // 2
    connect = 8 * M1 + 5 * nf * M1 + 9 * (n_conf + n_hang) + 5 * n_bnd
    mapk = 8 * (M0 + M1) + 5 * M1
    transfer = Bu * (M0 + M1) + 5 * M1
    return dict(adapt=adapt, balance=balance, connect=connect, map=mapk, transfer=transfer)


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2306_06744_b200 import build as B
    B.build()  # no-op when liblt.so is current; raises if nvcc fails (no fallback)
    from paper_2306_06744_b200 import workloads as W
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product has no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    cfg = W.CONFIGS[CONFIG]
    R = Runner(cfg, dev)
    Bu, p, nvars, N = R.Bu, R.p, R.nvars, R.N
    K, Wm = args.steps, max(args.warmup, 0)

    # ---- dry run (tree only) of one period: buffer sizes, so nothing is allocated in a timed step
    R.prepare()
    sizes = []
    for c in PERIOD:
        m0 = R.tree.num_leaves()
        R.tree.adapt(R.flags(c))
        R.tree.balance()
        sizes.append((m0, R.tree.num_leaves()))
    max_leaves = max(max(s) for s in sizes)
    cap = int(max_leaves * 1.02) + 4096
    # small meshes (the paper's own sizes): reserve the worst case, 2^dim x leaves, so that lt_adapt and
    # lt_balance(iters = NULL) only enqueue and the cycle has ONE host synchronisation (lt_connect_end)
    deferred = (not args.sync_calls) and OVERLAP and (max_leaves << cfg["dim"]) * 160 < (8 << 30)
    if deferred:
        cap = (max_leaves << cfg["dim"]) + 4096
    need = [0, 0]  # step k reads buffer k % 2 and writes the other one
    for k, (m0, m1) in enumerate(sizes):
        need[k % 2] = max(need[k % 2], m0)
        need[(k + 1) % 2] = max(need[(k + 1) % 2], m1)
    ubuf = [torch.empty((need[i] + 1024, nvars, N), dtype=torch.float64, device=dev) for i in range(2)]
    M_prep = R.prepare(reserve=cap)
    R.analytic_u(ubuf[0])
    cur = 0

    stream = torch.cuda.current_stream(dev)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    # timing rule: inputs larger than L2, or L2 flushed between timed iterations
    small = 2 * max_leaves * Bu < (512 << 20)
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev) if small else None

    def one_step(c, overlap=None):
        nonlocal cur
        overlap = OVERLAP if overlap is None else overlap
        t = R.tree
        M0 = t.num_leaves()
        f = R.flags(c)
        u_old = ubuf[cur][:M0]
        if flush is not None:
            flush.fill_(c & 255)
        launches0, syncs0 = t.launch_count(), t.host_syncs()
        torch.cuda.synchronize(dev)
        ev0.record(stream)
        t.adapt(f)
        if deferred and overlap:
            t.balance(want_iters=False)
            t.connect_begin()
            t.transfer_into(u_old, ubuf[cur ^ 1], p, nvars)
            F = t.connect_end()                      # the only host synchronisation of the cycle
            M1 = Ma = int(F["n_leaves"])             # (the count after lt_adapt never reached the host)
            iters = t.last_balance_iters()
        else:
            Ma = t.num_leaves()
            iters = t.balance()
            M1 = t.num_leaves()
            u_new = ubuf[cur ^ 1][:M1]
        if deferred and overlap:
            pass
        elif overlap:
            # the face query (side stream) overlaps the HBM-bound transfer: both depend only on
            # the balanced tree
            t.connect_begin()
            t.transfer(u_old, p, nvars, u_new)
            F = t.connect_end()
        else:
            F = t.connect()
            t.transfer(u_old, p, nvars, u_new)
        ev1.record(stream)
        syncs = t.host_syncs() - syncs0              # before the harness's own waits below
        torch.cuda.synchronize(dev)
        t.sync()
        ms = ev0.elapsed_time(ev1)
        tm = t.timings()
        tm.update({"balance_" + k: v for k, v in t.balance_phases().items()})
        cur ^= 1
        return dict(cycle=c, M0=M0, Ma=Ma, M1=M1, iters=iters, faces=(F["n_conf"], F["n_hang"], F["n_bnd"]),
                    ms=ms, tm=tm, launches=t.launch_count() - launches0, syncs=syncs)

    def rewind():
        nonlocal cur
        R.prepare(reserve=cap)
        R.analytic_u(ubuf[0])
        cur = 0

    seq = 0

    def next_cycle():
        nonlocal seq
        if seq and seq % len(PERIOD) == 0:
            rewind()
        c = PERIOD[seq % len(PERIOD)]
        seq += 1
        return c

    # warm-up: the first step uses the timed code path; the others run lt_connect and lt_transfer back
    # to back, which also gives k_transfer's bandwidth when it has the GPU to itself
    alone = []
    for i in range(Wm):
        r = one_step(next_cycle(), overlap=OVERLAP and i == 0)
        if not (OVERLAP and i == 0):
            alone.append(r)
    if seq % len(PERIOD):   # the timed region always starts at the first cycle of the period
        rewind()
        seq = 0
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize(dev)
    sampler = ClockSampler(local)
    sampler.start()
    t_wall0 = time.perf_counter()
    steps = [one_step(next_cycle()) for _ in range(K)]
    torch.cuda.synchronize(dev)
    if world > 1:
        dist.barrier()
    t_wall = time.perf_counter() - t_wall0
    clocks = sampler.stop()

    tot_ms = max_over_ranks(sum(s["ms"] for s in steps), world, dev)
    leaves = sum(s["M1"] for s in steps)
    faces = sum(sum(s["faces"]) for s in steps)
    value = whole_job_value(leaves, world, tot_ms)

    # ---- roofline of the dominant kernel (k_transfer): algorithmic bytes / measured kernel time
    peak, peak_src = hbm_peak()
    by = [algorithmic_bytes(cfg["dim"], s["M0"], s["Ma"], s["M1"], s["faces"], Bu, s["iters"]) for s in steps]
    tr_bytes = sum(b["transfer"] for b in by)
    tr_ms = sum(s["tm"]["k_transfer"] for s in steps)
    achieved = tr_bytes / (tr_ms * 1e-3) / 1e9
    traffic = traffic_note = None
    if CONFIG == "c5":
        traffic, alg = profile_traffic("k_transfer")
        if traffic is not None:
            traffic_note = ("ncu --set full of the config-5 cycle-3 launch (profiles/, see traffic.txt); "
                            "algorithmic bytes of that launch: %d" % alg)
    alone_GBps = None
    if alone:
        ab = sum(algorithmic_bytes(cfg["dim"], s["M0"], s["Ma"], s["M1"], s["faces"], Bu, s["iters"])["transfer"]
                 for s in alone)
        alone_GBps = ab / (sum(s["tm"]["k_transfer"] for s in alone) * 1e-3) / 1e9
    roofline = {"bound": "hbm", "kernel": "k_transfer<%d,%d>" % (cfg["dim"], p + 1), "achieved": achieved, "peak": peak, "unit": "GB/s",
                "achieved_alone": alone_GBps, "frac_alone": None if alone_GBps is None else alone_GBps / peak,
                "note": "timed steps overlap k_connect (side stream) with k_transfer, so `achieved` is k_transfer's "
                        "bandwidth under that contention; `achieved_alone` is the same kernel in the warm-up steps "
                        "that run lt_connect and lt_transfer back to back" if OVERLAP else "no overlap",
                "frac": achieved / peak, "traffic": traffic, "traffic_note": traffic_note, "peak_source": peak_src,
                "bytes_per_launch": tr_bytes / K, "ms_per_launch": tr_ms / K,
                "share_of_step": tr_ms / sum(s["ms"] for s in steps)}
    cyc_bytes = sum(sum(b.values()) for b in by)
    tree_bytes = sum(b["adapt"] + b["balance"] + b["connect"] + b["map"] for b in by)
    tree_ms = sum(s["ms"] - s["tm"]["k_transfer"] for s in steps)
    own_ms = sum(s["ms"] for s in steps)
    cycle_roofline = {
        "cycle_bytes_per_step": cyc_bytes / K, "cycle_GBps": cyc_bytes / (own_ms * 1e-3) / 1e9,
        "cycle_frac_of_measured_peak": cyc_bytes / (own_ms * 1e-3) / 1e9 / peak,
        "cycle_frac_of_8TBps_nominal": cyc_bytes / (own_ms * 1e-3) / 1e9 / 8000.0,
        "tree_connect_GBps": tree_bytes / (tree_ms * 1e-3) / 1e9,
        "tree_connect_frac_of_measured_peak": tree_bytes / (tree_ms * 1e-3) / 1e9 / peak,
    }
    per_call = {k: sum(s["tm"][k] for s in steps) / K for k in steps[0]["tm"]}
    # overlapped mode: lt_connect as a call has no duration of its own, the kernel's device time is used
    t_conn = sum(s["tm"]["connect"] or s["tm"]["k_connect"] for s in steps)
    faces_per_s = world * faces / (t_conn * 1e-3)
    launches = sum(s["launches"] for s in steps)

    # ---- e2e: the same cycle through the C ABI with HOST buffers (copies inside the timed region)
    e2e = None
    if not args.no_e2e:
        del ubuf
        R.tree.free()
        R.tree = None
        torch.cuda.empty_cache()
        e2e = run_e2e(R, args, world, dev)
        e2e["ms"] = max_over_ranks(e2e["ms"], world, dev)
        e2e["value"] = whole_job_value(e2e["leaves"], world, e2e["ms"])

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = cpu_baseline(CONFIG, cfg, args.oracle_full)

    if rank == 0:
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
            "ms_per_step": tot_ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOADS[CONFIG],
                       "step": ("one adaptation cycle; steps run %s cycles %s after an untimed tree-only replay of "
                                "cycles 0-%d" % (CONFIG, list(PERIOD), PREP_CYCLES - 1)) if PREP_CYCLES else
                               ("one adaptation cycle; steps run %s cycles %d..%d from the uniform base tree"
                                % (CONFIG, PERIOD[0], PERIOD[-1])),
                       "leaves_out_per_step": [s["M1"] for s in steps], "leaves_in_per_step": [s["M0"] for s in steps],
                       "balance_iters": [s["iters"] for s in steps], "balance_connectivity": CONNECTIVITY,
                       "connect_transfer_overlap": OVERLAP,
                       "host_synchronisations": "one per cycle (lt_connect_end): buffers reserved for 2^dim x leaves, "
                                                "lt_adapt and lt_balance(iters=NULL) only enqueue" if deferred else
                                                "three per cycle (lt_adapt sizes its buffers, lt_balance returns the "
                                                "sweep count, lt_connect_end the face counts)",
                       "l2": "L2 flushed between timed steps (a 512 MB fill; the inputs are smaller than L2)" if small
                             else "inputs larger than L2 (u_old + u_new are %.0f-%.0f GB per step)" % (
                                 min(sum(x) for x in sizes) * Bu / 1e9, max(sum(x) for x in sizes) * Bu / 1e9),
                       "parallelism": "replicas only (one independent tree per GPU)" if world > 1 else "single GPU",
                       "timing": "CUDA events on the tree's stream around lt_adapt..lt_transfer of each step; "
                                 "flag generation between steps is excluded"},
            "roofline": roofline, "cycle_roofline": cycle_roofline, "ms_per_call": per_call,
            "ms_per_cycle": [round(s["ms"], 4) for s in steps] if len(steps) <= 64 else None,
            "launches_per_cycle": launches / K, "host_syncs_per_cycle": sum(s["syncs"] for s in steps) / K,
            "faces_per_s": faces_per_s, "cpu_baseline": cpu, "clocks": clocks, "gpu_launches": launches,
            "wall_s_timed_region": t_wall,
            "e2e": None if e2e is None else {"value": e2e["value"], "unit": UNIT,
                                             "h2d_bytes_per_step": e2e["h2d"], "d2h_bytes_per_step": e2e["d2h"],
                                             "ms_per_step": e2e["ms"], "ms_each": e2e["ms_each"], "runs": e2e["runs"],
                                             "cycle": e2e["cycle"], "note": e2e["note"]},
        }
        print(json.dumps(out), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_e2e(R, args, world, dev):
    """One adaptation cycle with HOST inputs and outputs: flags and u_old start in pinned host memory;
    u_new, the keys, nbr / kind and the three face tables end in pinned host memory; every copy is inside
    the timed region.  Runs the largest cycle <= PERIOD[-1] (config 5: <= PERIOD[0]) whose host buffers fit
    the budget: one untimed warm-up run (staging ring, pools), then three timed runs from the same state."""
    torch = R.torch
    cfg, Bu, p, nvars, N = R.cfg, R.Bu, R.p, R.nvars, R.N
    nf = 2 * cfg["dim"]
    budget = min(64 << 30, int(0.4 * mem_available_bytes() / max(world, 1)))
    last = PERIOD[0] if CONFIG == "c5" else PERIOD[-1]
    dom = R.W.domain(cfg)

    def fresh(upto):
        if R.tree is not None:
            R.tree.free()
        t = R.lt.Tree(cfg["dim"], cfg["base"], cfg["maxl"], dom, cfg["periodic"], nroot=cfg.get("nroot"))
        if CONNECTIVITY != 1:
            t.set_option(R.lt.LT_OPT_BALANCE_CONNECTIVITY, CONNECTIVITY)
        R.tree = t
        counts = []
        for c in range(upto):
            m0 = t.num_leaves()
            t.adapt(R.flags(c))
            t.balance()
            counts.append((m0, t.num_leaves()))
        return t, counts

    _, counts = fresh(last + 1)
    pick = 0
    for c, (m0, m1) in enumerate(counts):
        if (m0 + m1) * (Bu + 160) <= budget:
            pick = c
    M0, M1 = counts[pick]
    h_old = torch.empty((M0, nvars, N), dtype=torch.float64, pin_memory=True)
    h_new = torch.empty((M1, nvars, N), dtype=torch.float64, pin_memory=True)
    # host copies of the tree-side results: keys, the paper's face array (nbr + kind), the face tables
    h_keys = torch.empty(M1, dtype=torch.int64, pin_memory=True)
    h_nbr = torch.empty(M1 * nf, dtype=torch.int32, pin_memory=True)
    h_kind = torch.empty(M1 * nf, dtype=torch.uint8, pin_memory=True)
    h_rows = torch.empty(M1 * (4 * cfg["dim"] + nf), dtype=torch.int32, pin_memory=True)
    h_bytes = torch.empty(M1 * (2 * cfg["dim"] + nf), dtype=torch.uint8, pin_memory=True)
    t, _ = fresh(pick)
    tmp = torch.empty((M0, nvars, N), dtype=torch.float64, device=dev)
    R.analytic_u(tmp)
    h_old.copy_(tmp)
    del tmp
    torch.cuda.empty_cache()
    h_flags = R.flags(pick).cpu().pin_memory()
    d_flags = torch.empty(M0, dtype=torch.int8, device=dev)
    stream = torch.cuda.current_stream(dev)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ms_each, d2h = [], 0
    for run in range(4):   # run 0 is the warm-up
        if run:
            t, _ = fresh(pick)
        t.reserve(int(M1 * 1.02) + 4096)
        torch.cuda.synchronize(dev)
        ev0.record(stream)
        d_flags.copy_(h_flags, non_blocking=True)
        t.adapt(d_flags)
        t.balance()
        F = t.connect()
        assert F["n_leaves"] == M1
        d2h, ro, bo = 0, 0, 0
        h_keys.copy_(t.keys(), non_blocking=True)
        h_nbr.copy_(F["nbr"], non_blocking=True)
        h_kind.copy_(F["kind"], non_blocking=True)
        d2h += 8 * M1 + 5 * nf * M1
        for rows_k, bytes_k in (("conf", "conf_axis"), ("hang", "hang_info"), ("bnd", "bnd_face")):
            a, bb = F[rows_k].reshape(-1), F[bytes_k]
            h_rows[ro:ro + a.numel()].copy_(a, non_blocking=True)
            h_bytes[bo:bo + bb.numel()].copy_(bb, non_blocking=True)
            ro, bo = ro + a.numel(), bo + bb.numel()
            d2h += 4 * a.numel() + bb.numel()
        t.transfer_host(h_old, h_new, p, nvars)
        ev1.record(stream)
        torch.cuda.synchronize(dev)
        if run:
            ms_each.append(ev0.elapsed_time(ev1))
        d2h += M1 * Bu + 64
    ms = sum(ms_each) / len(ms_each)
    return {"ms": ms, "ms_each": ms_each, "runs": len(ms_each), "leaves": M1, "h2d": M0 * Bu + M0, "d2h": d2h,
            "cycle": pick,
            "note": "%s cycle %d (%d -> %d leaves), mean of %d runs after one warm-up run; down: u_new, keys, nbr/kind "
                    "and the three face tables; host budget %.0f GB; lt_transfer_host pipelines upload / kernel / "
                    "download in slabs (three streams, 3-slab staging ring)"
                    % (CONFIG, pick, M0, M1, len(ms_each), budget / 2 ** 30)}


# --------------------------------------------------------------------------- construction leg
CONSTRUCT_METRIC = "leaves/s per tree construction from a point cloud (Alg. 2) + full-depth 2:1 balance + connectivity"


def oracle_construct(pc, pts_host):
    """The oracle on the same points: Alg. 2 + balance + connect.  Returns (leaves, seconds)."""
    import oracle
    dim = pc["dim"]
    dom = [pc["lo"]] * dim + [pc["hi"]] * dim
    t0 = time.perf_counter()
    ot = oracle.Tree(dim, pc["base"], pc["maxl"], pc["periodic"], points=pts_host, domain=dom)
    ot.balance()
    ot.connect()
    return ot.num_leaves(), time.perf_counter() - t0


def run_construct(args):
    """--workload construct: SURVEY.md 8(f)-1.  A step = lt_build_from_points (encode, radix sort,
    linearise, completion) + lt_balance + lt_connect on the seeded surface cloud `pc10`
    (16 M points, D_min 4, D_max 10: the stand-in for the paper's bunny run)."""
    import torch
    from paper_2306_06744_b200 import build as B
    B.build()
    from paper_2306_06744_b200 import lt
    from paper_2306_06744_b200 import workloads as W
    if int(os.environ.get("RANK", "0")) != 0:
        return
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product has no CPU fallback)")
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    name = args.cloud
    pc = W.POINT_CLOUDS[name]
    dim = pc["dim"]
    dom = [pc["lo"]] * dim + [pc["hi"]] * dim
    pts = W.surface_points(pc, device=dev)
    h_pts = pts.cpu().pin_memory()
    d_in = torch.empty_like(pts)                                           # e2e: upload target
    h_out = torch.empty(max(pts.shape[0], 1 << 22), dtype=torch.int64).pin_memory()  # e2e: keys back
    stream = torch.cuda.current_stream(dev)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)]

    def step(from_host=False):
        torch.cuda.synchronize(dev)
        ev[0].record(stream)
        if from_host:
            d_in.copy_(h_pts, non_blocking=True)
        x = d_in if from_host else pts
        t = lt.build_from_points(dim, pc["base"], pc["maxl"], x, dom, pc["periodic"])
        ev[1].record(stream)
        n0 = t.num_leaves()
        it = t.balance()
        ev[2].record(stream)
        F = t.connect()
        h_keys = None
        if from_host:
            k = t.keys()
            if k.numel() > h_out.numel():
                raise SystemExit("bench.py: the e2e key buffer is smaller than the tree (sparse cloud)")
            h_keys = h_out[:k.numel()]
            h_keys.copy_(k, non_blocking=True)
        ev[3].record(stream)
        torch.cuda.synchronize(dev)
        r = dict(n0=n0, n1=t.num_leaves(), iters=it, faces=int(F["n_conf"] + F["n_hang"] + F["n_bnd"]),
                 ms=ev[0].elapsed_time(ev[3]), build=ev[0].elapsed_time(ev[1]), balance=ev[1].elapsed_time(ev[2]),
                 connect=ev[2].elapsed_time(ev[3]), launches=t.launch_count(),
                 d2h=0 if h_keys is None else h_keys.numel() * 8)
        t.free()
        return r

    for _ in range(max(args.warmup, 0)):
        step()
    sampler = ClockSampler(0)
    sampler.start()
    steps = [step() for _ in range(args.steps)]
    clocks = sampler.stop()
    tot = sum(s["ms"] for s in steps)
    leaves = sum(s["n1"] for s in steps)
    e = [step(from_host=True) for _ in range(max(1, min(args.steps, 3)))]
    e_ms = sum(s["ms"] for s in e)
    cpu = None
    if not args.no_cpu_baseline:
        small = W.POINT_CLOUDS["pc9"]
        hp = W.surface_points(small).numpy()
        n, dt = oracle_construct(small, hp)
        cpu = {"value": n / dt, "unit": UNIT, "cores": 1, "kind": "oracle", "seconds": dt,
               "sample": "cloud pc9 in full (4 M points, D_min 4, D_max 9 -> %d leaves): Alg. 2 + balance + connect" % n}
    peak, peak_src = hbm_peak()
    s0 = steps[0]
    out = {
        "metric": CONSTRUCT_METRIC, "value": leaves / (tot * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": tot / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "int64", "data": "synthetic",
        "config": {"workload": "construct/%s: %d seeded points on a %s surface, %d-D, D_min %d, D_max %d -> %d leaves "
                               "after completion, %d after balance (%d sweeps), %d faces"
                               % (name, pts.shape[0], pc["surface"], dim, pc["base"], pc["maxl"], s0["n0"], s0["n1"],
                                  s0["iters"], s0["faces"]),
                   "l2": "each step builds a new tree from the 384 MB point array (larger than L2)",
                   "timing": "CUDA events around lt_build_from_points + lt_balance + lt_connect; includes the "
                             "library's own device allocations"},
        "ms_per_call": {k: sum(s[k] for s in steps) / args.steps for k in ("build", "balance", "connect")},
        "points_per_s": pts.shape[0] * args.steps / (sum(s["build"] for s in steps) * 1e-3),
        "roofline": {"bound": "hbm", "kernel": "whole construction call (launch- and allocation-bound, see profiles/r2_construct.md)",
                     "achieved": (24 * pts.shape[0] + 8 * s0["n0"]) * args.steps / (sum(s["build"] for s in steps) * 1e-3) / 1e9,
                     "peak": peak, "unit": "GB/s", "peak_source": peak_src, "traffic": None,
                     "frac": (24 * pts.shape[0] + 8 * s0["n0"]) * args.steps / (sum(s["build"] for s in steps) * 1e-3) / 1e9 / peak},
        "cpu_baseline": cpu, "clocks": clocks, "gpu_launches": sum(s["launches"] for s in steps),
        "e2e": {"value": sum(s["n1"] for s in e) / (e_ms * 1e-3), "unit": UNIT,
                "h2d_bytes_per_step": h_pts.numel() * 8, "d2h_bytes_per_step": e[0]["d2h"], "ms_per_step": e_ms / len(e)},
    }
    print(json.dumps(out), flush=True)


# --------------------------------------------------------------------------- mortar leg
def run_mortar(args):
    """--workload mortar: SURVEY.md 8(f)-2.  A step = lt_mortar_project + lt_mortar_gather over
    the face arrays [M][6][5][16] (p = 3, 5 fp64 variables) of the config-5 mesh after cycles
    0-2 (8.86 M leaves, 34 GB per face array)."""
    import torch
    from paper_2306_06744_b200 import build as B
    B.build()
    from paper_2306_06744_b200 import workloads as W
    if int(os.environ.get("RANK", "0")) != 0:
        return
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product has no CPU fallback)")
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    cfg = W.CONFIGS["c5"]
    R = Runner(cfg, dev)
    M = R.prepare()
    t = R.tree
    F = t.connect()
    kind = F["kind"] & 15
    n1, n2, n3 = int((kind == 1).sum()), int((kind == 2).sum()), int((kind == 3).sum())
    p, nvars, nf = cfg["p"], cfg["nvars"], 6
    Nf = (p + 1) ** 2
    Bf = 8 * nvars * Nf
    uf = torch.empty((M, nf, nvars, Nf), dtype=torch.float64, device=dev)
    step = 1 << 19
    for a in range(0, M, step):  # seeded face data, slab by slab
        b = min(a + step, M)
        i = torch.arange(a * nf * nvars * Nf, b * nf * nvars * Nf, dtype=torch.int64, device=dev)
        uf[a:b] = (2.0 * W.counter_uniform(5, 21, i) - 1.0).view(b - a, nf, nvars, Nf)
        del i
    out = torch.empty_like(uf)
    N = (p + 1) ** 3
    u = torch.empty((M, nvars, N), dtype=torch.float64, device=dev)  # Alg. 8 step 1 input
    R.analytic_u(u)
    stream = torch.cuda.current_stream(dev)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
    ms_i_all = []

    def step_once():
        torch.cuda.synchronize(dev)
        ev[3].record(stream)
        t.face_interp(u, p, nvars, u_face=out)
        ev[0].record(stream)
        t.mortar_project(uf, p, nvars, u_nb=out)
        ev[1].record(stream)
        t.mortar_gather(uf, p, nvars, f_face=out)
        ev[2].record(stream)
        torch.cuda.synchronize(dev)
        t.sync()
        ms_i_all.append(ev[3].elapsed_time(ev[0]))
        return ev[0].elapsed_time(ev[1]), ev[1].elapsed_time(ev[2])

    for _ in range(max(args.warmup, 0)):
        step_once()
    sampler = ClockSampler(0)
    sampler.start()
    del ms_i_all[:]
    times = [step_once() for _ in range(args.steps)]
    clocks = sampler.stop()
    ms_i = sum(ms_i_all) / args.steps
    bytes_i = (8 * nvars * N + nf * Bf) * M
    ms_p = sum(a for a, _ in times) / args.steps
    ms_g = sum(b for _, b in times) / args.steps
    bytes_p = 2 * Bf * (n1 + n2) + 5 * nf * M
    bytes_g = Bf * (n2 + n3) + (nf + 8) * M
    peak, peak_src = hbm_peak()
    ach = bytes_p / (ms_p * 1e-3) / 1e9
    cpu = None
    if not args.no_cpu_baseline:
        import numpy as np
        import oracle
        ot = oracle.Tree(cfg["dim"], cfg["base"], cfg["maxl"], cfg["periodic"])
        lvl, xyz = ot.leaf_boxes()
        ot.adapt(W.flags(cfg, 0, torch.from_numpy(lvl), torch.from_numpy(xyz.astype(np.int64))).numpy())
        ot.balance()
        ot.connect()
        h = np.random.default_rng(0).uniform(-1, 1, (ot.num_leaves(), nf, nvars, Nf))
        t0 = time.perf_counter()
        ot.mortar_project(h, p, nvars)
        ot.mortar_gather(h, p, nvars)
        dt = time.perf_counter() - t0
        cpu = {"value": ot.num_leaves() * nf / dt, "unit": "face slots/s", "cores": 1, "kind": "oracle", "seconds": dt,
               "sample": "config-5 mesh after cycle 0 (%d leaves): project + gather" % ot.num_leaves()}
    e2e = None
    if not args.no_e2e:   # the same step with the face array coming from, and the result going to, pinned host memory
        h_in = torch.empty(uf.shape, dtype=torch.float64, pin_memory=True)
        h_out = torch.empty(uf.shape, dtype=torch.float64, pin_memory=True)
        h_in.copy_(uf)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ms_e = []
        for _ in range(2):  # (the first run is the warm-up)
            torch.cuda.synchronize(dev)
            e0.record(stream)
            uf.copy_(h_in, non_blocking=True)
            t.mortar_project(uf, p, nvars, u_nb=out)
            t.mortar_gather(uf, p, nvars, f_face=out)
            h_out.copy_(out, non_blocking=True)
            e1.record(stream)
            torch.cuda.synchronize(dev)
            ms_e.append(e0.elapsed_time(e1))
        e2e = {"value": M * nf / (ms_e[-1] * 1e-3), "unit": "face slots/s", "h2d_bytes_per_step": uf.numel() * 8,
               "d2h_bytes_per_step": out.numel() * 8, "ms_per_step": ms_e[-1],
               "note": "face array uploaded from, result downloaded to pinned host memory inside the timed step"}
        del h_in, h_out
    traffic, traffic_alg = profile_traffic("k_mortar_project")
    print(json.dumps({
        "metric": "face slots/s through lt_mortar_project + lt_mortar_gather (Alg. 8 steps 2 and 4)",
        "value": M * nf / ((ms_p + ms_g) * 1e-3), "unit": "face slots/s", "n_gpus": 1, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_p + ms_g, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "mortar: config-5 mesh after cycles 0-2 (%d leaves; %d conforming, %d fine-side and %d "
                               "coarse-side hanging face slots), p=3, 5 fp64 vars, face arrays [M][6][5][16]"
                               % (M, n1, n2, n3),
                   "l2": "face arrays of %.1f GB each, larger than L2" % (uf.numel() * 8 / 1e9)},
        "ms_per_call": {"face_interp": ms_i, "mortar_project": ms_p, "mortar_gather": ms_g},
        "face_interp": {"GBps": bytes_i / (ms_i * 1e-3) / 1e9, "bytes_per_launch": bytes_i,
                        "frac": bytes_i / (ms_i * 1e-3) / 1e9 / peak,
                        "note": "Alg. 8 step 1, timed before the mortar step; not part of `value`"},
        "roofline": {"bound": "hbm", "kernel": "k_mortar_project<3>", "achieved": ach, "peak": peak, "unit": "GB/s",
                     "frac": ach / peak, "traffic": traffic, "traffic_note": None if traffic is None else
                     "ncu --set full of one launch on the same mesh (profiles/r1f_mortar_full.md, traffic.txt); "
                     "algorithmic bytes of that launch: %d" % traffic_alg,
                     "peak_source": peak_src, "bytes_per_launch": bytes_p,
                     "gather_GBps": bytes_g / (ms_g * 1e-3) / 1e9, "gather_bytes_per_launch": bytes_g},
        "cpu_baseline": cpu, "clocks": clocks, "gpu_launches": 4 * args.steps,
        "e2e": e2e}), flush=True)


# --------------------------------------------------------------------------- solver leg
def run_solver(args):
    """--workload solver: SURVEY.md 8(f)-4, the paper's headline (adaptation below
    2 % of wall clock in 3-D with one adaptation every 10 steps of the 3-stage RK scheme).
    Config-5 mesh: one adaptation cycle (cycle 2: 1.9 M -> 8.86 M leaves, with the solution transfer),
    then 10 SSP-RK3 steps (30 right-hand sides = Alg. 8 steps 1-4 + Eq. 2-5 + Eq. 6) on the adapted mesh."""
    import torch
    from paper_2306_06744_b200 import build as B
    B.build()
    from paper_2306_06744_b200 import workloads as W
    if int(os.environ.get("RANK", "0")) != 0:
        return
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product has no CPU fallback)")
    global PREP_CYCLES
    # c5: cycle 2 (1.9 M -> 8.86 M leaves); slab (the paper's own 3-D domain and mesh sizes): cycle 8;
    # c4: cycle 5 (1.14 M leaves, p = 2: the generic right-hand-side kernel on arrays larger than L2)
    name = CONFIG if CONFIG in ("c5", "slab", "c4") else "c5"
    PREP_CYCLES = {"c5": 2, "slab": 8, "c4": 5}[name]
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    cfg = W.CONFIGS[name]
    R = Runner(cfg, dev)
    p, nvars, nf = cfg["p"], cfg["nvars"], 6
    N, Nf = (p + 1) ** 3, (p + 1) ** 2
    stream = torch.cuda.current_stream(dev)

    def timed(fn):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize(dev)
        e0.record(stream)
        out = fn()
        e1.record(stream)
        torch.cuda.synchronize(dev)
        return e0.elapsed_time(e1), out

    def adapt_cycle(host_u_old=None):
        """untimed set-up of the pre-adaptation state, then the timed cycle 2; host_u_old: (e2e) the old
        solution starts in pinned host memory and its upload is part of the timed cycle (None on the
        first call of that mode, which creates the pinned copy untimed and returns it)"""
        M0 = R.prepare()
        t = R.tree
        u_old = torch.empty((M0, nvars, N), dtype=torch.float64, device=dev)
        if host_u_old is None or host_u_old is True:
            R.analytic_u(u_old)
        if host_u_old is True:
            host_u_old = torch.empty(u_old.shape, dtype=torch.float64, pin_memory=True)
            host_u_old.copy_(u_old)
            u_old.zero_()
        f = R.flags(PREP_CYCLES)
        # a small mesh (the paper's sizes): buffers for the worst case, so that the cycle has one host wait
        small = (M0 << 3) * (160 + 8 * nvars * N) < (8 << 30)
        buf = None
        if small:
            t.reserve((M0 << 3) + 4096)
            buf = torch.empty(((M0 << 3) + 4096, nvars, N), dtype=torch.float64, device=dev)

        def cyc():
            if host_u_old is not None:
                u_old.copy_(host_u_old, non_blocking=True)
            t.adapt(f)
            if small:
                t.balance(want_iters=False)
                t.connect_begin()
                t.transfer_into(u_old, buf, p, nvars)
                F = t.connect_end()
                return buf[:int(F["n_leaves"])], F
            t.balance()
            M1 = t.num_leaves()
            u_new = torch.empty((M1, nvars, N), dtype=torch.float64, device=dev)
            t.connect_begin()
            t.transfer(u_old, p, nvars, u_new)
            F = t.connect_end()
            return u_new, F
        ms, (u_new, F) = timed(cyc)
        t.sync()
        return ms, M0, u_new.contiguous(), F

    adapt_cycle()                                  # warm-up (allocations, operators)
    ms_adapt_e2e = h2d = None
    if not args.no_e2e:                            # the same cycle with u_old coming from pinned host memory
        ms_adapt_e2e, M0e, ue, _ = adapt_cycle(host_u_old=True)
        h2d = M0e * 8 * nvars * N
        del ue
    ms_adapt, M0, u, F = adapt_cycle()
    t = R.tree
    M = t.num_leaves()
    uf = torch.empty((M, nf, nvars, Nf), dtype=torch.float64, device=dev)
    fs = torch.empty_like(uf)
    rhs, us = torch.empty_like(u), torch.empty_like(u)
    # finest cell 20 / 512 (c5, p = 3) or 25 / 256 (slab, p = 2), |v| + c about 4.2: well inside the RK3 limit
    dt = 5e-4 if name == "slab" else 2e-4

    def fluxes_of(x):
        t.face_interp(x, p, nvars, u_face=uf)
        t.mortar_project(uf, p, nvars, u_nb=fs)
        t.common_flux(uf, fs, p, f_star=fs)        # in place over the neighbour traces
        t.mortar_gather(fs, p, nvars, f_face=fs)

    def rhs_of(x):
        fluxes_of(x)
        t.fr_rhs(x, fs, p, rhs=rhs)

    fused = not args.unfused

    def rk3_step():
        if not fused:                              # round-1 chain: five passes per stage
            fluxes_of(u)
            t.fr_stage(1, dt, u, u, fs, p, out=us)
            fluxes_of(us)
            t.fr_stage(2, dt, u, us, fs, p, out=us)
            fluxes_of(us)
            t.fr_stage(3, dt, u, us, fs, p, out=u)
            return
        # three passes per stage: lt_face_flux (Alg. 8 steps 2 + 3, neighbour traces never stored),
        # lt_mortar_gather, lt_fr_stage_faces (Eq. 2-6 + the traces of the result for the next stage);
        # uf holds the traces of u on entry and on exit
        for stage, (src, dst) in enumerate(((u, us), (us, us), (us, u)), start=1):
            t.face_flux(uf, p, f_star=fs)
            t.mortar_gather(fs, p, nvars, f_face=fs)
            t.fr_stage_faces(stage, dt, u, src, fs, p, out=dst, u_face_out=uf)

    t.face_interp(u, p, nvars, u_face=uf)
    rk3_step()                                     # warm-up
    ms_solve, _ = timed(lambda: [rk3_step() for _ in range(10)])
    ms_rhs, _ = timed(lambda: rhs_of(u))
    sampler = ClockSampler(0)
    sampler.start()
    ms_solve2, _ = timed(lambda: [rk3_step() for _ in range(10)])
    clocks = sampler.stop()
    ms_solve = min(ms_solve, ms_solve2)
    assert bool(torch.isfinite(u).all()), "the solution blew up"
    e2e = None
    if ms_adapt_e2e is not None:                   # ten steps and the result back in pinned host memory
        h_u = torch.empty(u.shape, dtype=torch.float64, pin_memory=True)
        ms_solve_e2e, _ = timed(lambda: ([rk3_step() for _ in range(10)], h_u.copy_(u, non_blocking=True)))
        e2e = {"value": ms_adapt_e2e / (ms_adapt_e2e + ms_solve_e2e), "unit": "fraction",
               "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": u.numel() * 8,
               "ms_per_step": ms_adapt_e2e + ms_solve_e2e, "ms_adaptation_cycle": ms_adapt_e2e,
               "ms_ten_rk3_steps": ms_solve_e2e,
               "note": "u_old uploaded from pinned host memory inside the timed cycle; the solution after the ten "
                       "steps downloaded to pinned host memory inside the timed solve"}
        del h_u
    cpu = None if args.no_cpu_baseline else oracle_solver_share()
    traffic, traffic_alg = profile_traffic("rk_stage") if (name == "c5" and fused) else (None, None)
    frac = ms_adapt / (ms_adapt + ms_solve)
    Bu, Bf = 8 * nvars * N, 8 * nvars * Nf
    # algorithmic bytes of one RK stage: face_interp (Bu + 6 Bf) + project (~2 * 6 Bf) + common flux (3 * 6 Bf)
    # + fused right-hand side and update (read u_stage, u_n and 6 Bf, write u_out: 3 Bu + 6 Bf)
    bytes_stage = M * (3 * Bu + 24 * Bf) if fused else M * (4 * Bu + 6 * Bf * 7)
    peak, peak_src = hbm_peak()
    print(json.dumps({
        "metric": "adaptation share of wall clock, one adaptation cycle per 10 SSP-RK3 steps (PAPER.md:449)",
        "value": frac, "unit": "fraction", "n_gpus": 1, "steps": 1, "warmup": 1,
        "ms_per_step": ms_adapt + ms_solve, "higher_is_better": False, "scaling": "weak", "vs_baseline": frac / 0.0194,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": "solver: %s cycle %d (%d -> %d leaves, p=%d, 5 fp64 vars, Euler) + 10 RK3 steps "
                               "(30 right-hand sides) on the adapted mesh" % (name, PREP_CYCLES, M0, M, p),
                   "baseline": "paper Table 5, p2 D_max 8, RTX 2060: 81.39 s / 4193.54 s = 1.94 % (160 k elements)",
                   "l2": "arrays of %.2f-%.2f GB%s" % (M * Bu / 1e9, M * 6 * Bf / 1e9,
                                                        ", larger than L2" if M * Bu > (256 << 20) else
                                                        " (smaller than L2: the paper's own mesh size, launch-bound)")},
        "ms_per_call": {"adaptation_cycle": ms_adapt, "ten_rk3_steps": ms_solve, "one_rhs_chain": ms_rhs},
        "roofline": {"bound": "hbm", "kernel": "RK stage (face_flux, mortar_gather, fr_stage_faces)" if fused else
                     "RK stage (face_interp, mortar_project, common_flux, mortar_gather, fr_stage)", "achieved": bytes_stage * 30 / (ms_solve * 1e-3) / 1e9,
                     "peak": peak, "unit": "GB/s", "frac": bytes_stage * 30 / (ms_solve * 1e-3) / 1e9 / peak,
                     "traffic": traffic, "traffic_note": None if traffic is None else
                     "stage 1 of the fused chain under ncu --set full (profiles/r2_solver.md, traffic.txt); "
                     "algorithmic bytes of that stage: %d" % traffic_alg,
                     "peak_source": peak_src, "bytes_per_launch": bytes_stage},
        "elements_per_s_rhs": M * 30 / (ms_solve * 1e-3),
        "cpu_baseline": cpu, "clocks": clocks, "gpu_launches": (30 * 4 if fused else 30 * 6) + 6, "e2e": e2e}),
        flush=True)

def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None,
                    help="timed steps (default: 3 for c5, one pass over all cycles for --config c1 / c2 / c4)")
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="c5", choices=sorted(SCHEDULES),
                    help="c5 (default): the config BASELINE.json's metric is quoted on; c1 / c2 / c4: secondary lines "
                         "in the same schema (one step = one adaptation cycle, all stated cycles from the uniform tree)")
    ap.add_argument("--oracle-full", action="store_true",
                    help="cpu_baseline / --impl reference on the config's full sample (c1-c4: every cycle; c5: cycles "
                         "0-3 with the transfer timed on slabs) instead of the bounded default")
    ap.add_argument("--unfused", action="store_true",
                    help="--workload solver: the round-1 chain of five passes per RK stage instead of the three fused ones")
    ap.add_argument("--sync-calls", action="store_true",
                    help="small configs: keep the synchronising lt_adapt / lt_balance (the before of the "
                         "one-synchronisation cycle)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--workload", default="cycle", choices=["cycle", "construct", "mortar", "solver"],
                    help="cycle (default): the adaptation cycle BASELINE.json's metric is quoted on; construct: "
                         "tree construction from a point cloud (SURVEY.md 8(f)-1)")
    ap.add_argument("--cloud", default="pc10", help="point cloud of --workload construct (workloads.POINT_CLOUDS)")
    ap.add_argument("--no-overlap", action="store_true",
                    help="run lt_connect and lt_transfer back to back instead of overlapping them "
                         "(lt_connect_begin / lt_transfer / lt_connect_end)")
    ap.add_argument("--connectivity", type=int, default=1,
                    help="2:1 balance across faces (1, default = BASELINE.json's contract), faces + edges (2, the "
                         "paper's strong balance, PAPER.md:132) or faces + edges + corners (3)")
    ap.add_argument("--cycles", default=None,
                    help="consecutive config-5 cycles a step cycles through (default 3,4,5 = the bench "
                         "workload; smaller ones, e.g. 2, keep an ncu --set full capture short)")
    args = ap.parse_args()
    global CONNECTIVITY, OVERLAP, CONFIG, PERIOD, PREP_CYCLES
    CONNECTIVITY = args.connectivity
    OVERLAP = not args.no_overlap
    CONFIG = args.config
    PREP_CYCLES, PERIOD = SCHEDULES[CONFIG]
    if args.cycles:
        PERIOD = tuple(int(c) for c in args.cycles.split(","))
        assert all(b == a + 1 for a, b in zip(PERIOD, PERIOD[1:])), "--cycles must be consecutive"
        PREP_CYCLES = PERIOD[0]
    if args.steps is None:
        args.steps = 3 if CONFIG == "c5" or args.impl == "reference" else len(PERIOD)
    if args.steps < 1:
        args.steps = 1
    if args.workload == "construct" and args.impl == "ours":
        run_construct(args)
    elif args.workload == "mortar" and args.impl == "ours":
        run_mortar(args)
    elif args.workload == "solver" and args.impl == "ours":
        run_solver(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
