"""GPU parity tests: the CUDA library (through the C ABI binding) against the CPU oracle,
element by element on the same seeded inputs.  Run on the B200 box: pytest -m gpu."""
import numpy as np
import pytest
import torch

import oracle
import parity as P
from paper_2306_06744_b200 import lt
from paper_2306_06744_b200 import workloads as W

pytestmark = pytest.mark.gpu


# ---------------------------------------------------------------- a-1 keys
@pytest.mark.parametrize("dim,maxl", [(2, 8), (2, 29), (3, 9), (3, 19)])
def test_encode_decode_matches_oracle(dim, maxl):
    rng = np.random.default_rng(7 + dim * 100 + maxl)
    n = 3000
    lvl = rng.integers(0, maxl + 1, n).astype(np.int32)
    xyz = np.zeros((n, 3), np.int64)
    for a in range(dim):
        xyz[:, a] = rng.integers(0, 1 << maxl, n)
    xyz = (xyz >> (maxl - lvl)[:, None]) << (maxl - lvl)[:, None]  # aligned anchors
    keys = lt.encode(dim, maxl, torch.from_numpy(xyz.astype(np.int32)).cuda(), torch.from_numpy(lvl).cuda())
    ref = np.array([oracle.encode(dim, maxl, int(lvl[i]), xyz[i].astype(np.uint32)) for i in range(n)], np.uint64)
    assert np.array_equal(P.u64(keys), ref)
    l2, x2 = lt.decode(dim, maxl, keys)
    assert np.array_equal(l2.cpu().numpy(), lvl)
    assert np.array_equal(x2.cpu().numpy().astype(np.int64), xyz)
    # unaligned coordinates are truncated to the cell anchor (Alg. 1 step 2)
    xyz_u = xyz + rng.integers(0, 1 << 20, (n, 3)) % np.maximum(1, (1 << (maxl - lvl)))[:, None]
    xyz_u[:, dim:] = 0
    keys_u = lt.encode(dim, maxl, torch.from_numpy(xyz_u.astype(np.int32)).cuda(), torch.from_numpy(lvl).cuda())
    assert np.array_equal(P.u64(keys_u), ref)


@pytest.mark.parametrize("dim,base,maxl,per", [(2, 0, 3, (0, 0)), (2, 3, 8, (0, 0)), (2, 7, 11, (1, 1)),
                                               (3, 0, 2, (1, 1, 1)), (3, 3, 12, (0, 0, 0)), (3, 5, 8, (1, 1, 1))])
def test_build_uniform(dim, base, maxl, per):
    gt = lt.Tree(dim, base, maxl, None, per)
    ot = oracle.Tree(dim, base, maxl, per)
    P.assert_keys_equal(gt, ot, "uniform build")
    P.assert_faces_equal(gt.connect(), ot.connect(), "uniform connect")
    assert gt.balance() == 0


# ---------------------------------------------------------------- whole cycles, BASELINE.json configs
def test_config1_full():
    cfg = W.CONFIGS["c1"]
    P.run_cycles(cfg, cfg["cycles"])


def test_config1_free_running():
    cfg = W.CONFIGS["c1"]
    P.run_cycles(cfg, cfg["cycles"], drift_free=False)


def test_config3_full():
    cfg = W.CONFIGS["c3"]
    log = []
    gt, ot, ug, uo = P.run_cycles(cfg, cfg["cycles"], log=log)
    assert [r[2] for r in log] == [0] * 18  # a domain-corner leaf has no cascade
    assert log[8][1] == 575 and log[-1][1] == 512
    # coarsen-everything restores the original tree and u to round-off
    P.assert_keys_equal(gt, oracle.Tree(cfg["dim"], cfg["base"], cfg["maxl"], cfg["periodic"]), "restored")


def test_config3b_ripple():
    cfg = W.CONFIGS["c3b"]
    log = []
    P.run_cycles(cfg, cfg["cycles"], log=log)
    assert [r[1] for r in log[:9]] == [519, 547, 596, 652, 708, 764, 820, 876, 932]
    assert [r[2] for r in log[:9]] == [0, 1, 2, 3, 3, 3, 3, 3, 3]


def test_config3b_deferred_balance_and_mapping_error():
    """Nine adapts then ONE balance: a 10-sweep ripple; the map from
    the last snapshot then spans more than one level -> LT_ERR_MAPPING."""
    cfg = W.CONFIGS["c3b"]
    gt, ot = P.new_pair(cfg)
    for c in range(9):
        f = P.host_flags(cfg, c, ot)
        ot.adapt(f)
        gt.adapt(torch.from_numpy(f).cuda())
        P.assert_keys_equal(gt, ot, "adapt %d" % c)
    with pytest.raises(lt.LtError) as ei:
        gt.connect()
    assert ei.value.status == lt.LT_ERR_UNBALANCED
    it_o = ot.balance()
    it_g = gt.balance()
    assert it_g == it_o == 10
    P.assert_keys_equal(gt, ot, "deferred balance")
    assert gt.num_leaves() == 932
    P.assert_faces_equal(gt.connect(), ot.connect(), "deferred connect")
    with pytest.raises(oracle.OracleError):
        ot.build_map()
    u = torch.zeros((gt.num_old_leaves(), 5, 8), dtype=torch.float64, device="cuda")
    gt.transfer(u, 1, 5)
    with pytest.raises(lt.LtError) as ei:
        gt.sync()
    assert ei.value.status == lt.LT_ERR_MAPPING


def test_config2_first_cycles():
    cfg = W.CONFIGS["c2"]
    log = []
    P.run_cycles(cfg, 6, log=log)
    assert [r[1] for r in log] == [19312, 30115, 68131, 199249, 255919, 276682]  # SURVEY 8d census
    assert [r[2] for r in log] == [0, 1, 2, 2, 2, 2]


def test_config4_first_cycles():
    cfg = W.CONFIGS["c4"]
    log = []
    P.run_cycles(cfg, 3, log=log)
    assert [r[1] for r in log] == [48000, 157984, 926752]
    assert [r[2] for r in log] == [0, 1, 2]


def test_config5_recipe_small():
    """Config 5's recipe (vortex tube + 10 % random refine / group coarsen, p = 3) on a
    16^3 base so that the oracle finishes in seconds."""
    cfg = dict(W.CONFIGS["c5"], base=4, maxl=7)
    P.run_cycles(cfg, 4)


# ---------------------------------------------------------------- options must not change results
def test_adapt_path_a_equals_path_b():
    """Alg. 6 as printed (append, radix sort, linearise) == ordered expansion (reading B-5)."""
    for name, nc in (("c1", 4), ("c3b", 12), ("c2", 4)):
        cfg = W.CONFIGS[name]
        P.run_cycles(cfg, nc, options=[(lt.LT_OPT_ADAPT_SORT, 1)], check_transfer=(name != "c2"))


def test_balance_full_sweeps_equal_frontier():
    cfg = W.CONFIGS["c3b"]
    P.run_cycles(cfg, 12, options=[(lt.LT_OPT_BALANCE_FULL_SWEEPS, 1)], check_transfer=False)
    cfg = W.CONFIGS["c2"]
    P.run_cycles(cfg, 4, options=[(lt.LT_OPT_BALANCE_FULL_SWEEPS, 1)], check_transfer=False, check_faces=False)


# ---------------------------------------------------------------- random trees, all p
@pytest.mark.parametrize("dim,p,nvars", [(2, 0, 1), (2, 1, 3), (2, 2, 4), (2, 3, 4), (2, 4, 2), (2, 7, 1),
                                         (3, 0, 2), (3, 1, 5), (3, 2, 5), (3, 3, 5), (3, 4, 1), (3, 5, 2)])
def test_random_trees_transfer(dim, p, nvars):
    """Random refine/coarsen flags on a periodic-x tree; every transfer case and every p."""
    base, maxl = (2, 6) if dim == 2 else (1, 4)
    per = (1, 0, 1)[:dim]
    gt = lt.Tree(dim, base, maxl, None, per)
    ot = oracle.Tree(dim, base, maxl, per)
    rng = np.random.default_rng(1000 * dim + 10 * p + nvars)
    N = (p + 1) ** dim
    uo = rng.uniform(-1, 1, (ot.num_leaves(), nvars, N))
    for c in range(6):
        M = ot.num_leaves()
        f = rng.choice(np.array([-1, 0, 1], np.int8), M, p=[0.45, 0.3, 0.25] if c % 2 else [0.2, 0.4, 0.4])
        ot.adapt(f)
        gt.adapt(torch.from_numpy(f).cuda())
        P.assert_keys_equal(gt, ot, "adapt")
        assert gt.balance() == ot.balance()
        P.assert_keys_equal(gt, ot, "balance")
        P.assert_faces_equal(gt.connect(), ot.connect(), "connect")
        src_o, kind_o = ot.build_map()
        un_o = ot.transfer_rows(uo, p, nvars, 0, ot.num_leaves())
        ot.drop_snapshot()
        un_g = gt.transfer(torch.from_numpy(uo).cuda(), p, nvars)
        gt.sync()
        src_g, kind_g = gt.map()
        assert np.array_equal(src_g.cpu().numpy(), src_o) and np.array_equal(kind_g.cpu().numpy(), kind_o)
        P.assert_u_close(un_g, un_o, "transfer dim %d p %d cycle %d" % (dim, p, c))
        assert set(np.unique(kind_o & 15).tolist()) <= {0, 1, 2}
        uo = un_o


def test_transfer_host_buffers():
    cfg = W.CONFIGS["c1"]
    gt, ot = P.new_pair(cfg)
    uo = P.initial_u(cfg, ot)
    f = P.host_flags(cfg, 0, ot)
    ot.adapt(f); ot.balance()
    gt.adapt(torch.from_numpy(f).cuda()); gt.balance()
    un_o = ot.transfer(uo, cfg["p"], cfg["nvars"])
    h_old = torch.from_numpy(uo).pin_memory()
    h_new = torch.empty((gt.num_leaves(), cfg["nvars"], 9), dtype=torch.float64).pin_memory()
    gt.transfer_host(h_old, h_new, cfg["p"], cfg["nvars"])
    P.assert_u_close(h_new, un_o, "host transfer")


@pytest.mark.parametrize("slab,pinned", [(1, True), (37, True), (37, False), (1000, True), (0, True)])
def test_transfer_host_pipelined_slabs(slab, pinned):
    # many slabs through the 3-deep staging ring, with refined groups and coarsened groups
    # crossing the candidate slab boundaries; 3-D, copy + interpolate + project in one cycle
    cfg = dict(W.CONFIGS["c4"], base=3, maxl=5)
    gt, ot = P.new_pair(cfg)
    rng = np.random.default_rng(5)
    for c in range(2):
        f = rng.integers(0, 2, ot.num_leaves()).astype(np.int8)
        ot.adapt(f); ot.balance(); ot.drop_snapshot()
        gt.adapt(torch.from_numpy(f).cuda()); gt.balance()
    p, nvars = 2, 3
    uo = rng.uniform(-1, 1, (ot.num_leaves(), nvars, 27))
    f = rng.integers(-1, 2, ot.num_leaves()).astype(np.int8)
    ot.adapt(f); ot.balance()
    gt.adapt(torch.from_numpy(f).cuda()); gt.balance()
    un_o = ot.transfer(uo, p, nvars)
    h_old = torch.from_numpy(uo.copy())
    h_new = torch.full((gt.num_leaves(), nvars, 27), float("nan"), dtype=torch.float64)
    if pinned:
        h_old, h_new = h_old.pin_memory(), h_new.pin_memory()
    gt.set_option(4, slab)
    gt.transfer_host(h_old, h_new, p, nvars)
    assert not torch.isnan(h_new).any()
    P.assert_u_close(h_new, un_o, "pipelined host transfer, slab %d" % slab)
    src, kind = gt.map()
    assert len(set((kind.cpu().numpy() & 15).tolist())) == 3  # copy, refine and coarsen all present
    # the tree stays usable: a second cycle through the device path
    f = rng.integers(-1, 2, ot.num_leaves()).astype(np.int8)
    ot.adapt(f); ot.balance()
    gt.adapt(torch.from_numpy(f).cuda()); gt.balance()
    un_g = gt.transfer(torch.from_numpy(un_o).cuda(), p, nvars)
    P.assert_u_close(un_g, ot.transfer(un_o, p, nvars), "device transfer after host transfer")


def test_transfer_without_snapshot_is_copy():
    gt = lt.Tree(2, 3, 5)
    u = torch.rand((64, 2, 9), dtype=torch.float64, device="cuda")
    v = gt.transfer(u, 2, 2)
    assert torch.equal(u, v)
    src, kind = gt.map()
    assert torch.equal(src.cpu(), torch.arange(64, dtype=torch.int32)) and int(kind.max()) == 0


# ---------------------------------------------------------------- edge cases of adapt
def test_adapt_limits_and_mixed_groups():
    # refine flags at max level and coarsen flags at base level are ignored (reading B-2)
    gt = lt.Tree(2, 2, 2)
    k0 = gt.keys().clone()
    gt.adapt(torch.ones(16, dtype=torch.int8, device="cuda"))
    assert torch.equal(gt.keys(), k0)
    gt.adapt(-torch.ones(16, dtype=torch.int8, device="cuda"))
    assert torch.equal(gt.keys(), k0)
    # a sibling group with mixed flags is not coarsened; its refine flag is honoured (B-3)
    gt, ot = lt.Tree(2, 1, 4), oracle.Tree(2, 1, 4)
    f = np.ones(4, np.int8)
    ot.adapt(f); gt.adapt(torch.from_numpy(f).cuda())
    f = -np.ones(16, np.int8)
    f[5] = 1   # group 1 mixed
    f[8] = 0   # group 2 incomplete flags
    ot.adapt(f); gt.adapt(torch.from_numpy(f).cuda())
    P.assert_keys_equal(gt, ot, "mixed groups")
    assert gt.num_leaves() == 16 - 2 * 3 + 3
    # all-zero flags: nothing changes, snapshot equals the tree
    k = gt.keys().clone()
    gt.adapt(torch.zeros(gt.num_leaves(), dtype=torch.int8, device="cuda"))
    assert torch.equal(gt.keys(), k) and torch.equal(gt.old_keys(), k)


def test_refine_all_then_coarsen_all_restores():
    for dim, base, maxl in ((2, 3, 6), (3, 2, 4)):
        gt = lt.Tree(dim, base, maxl, None, (1,) * dim)
        k0 = gt.keys().clone()
        for _ in range(maxl - base):
            gt.adapt(torch.ones(gt.num_leaves(), dtype=torch.int8, device="cuda"))
        assert gt.num_leaves() == 1 << (dim * maxl)
        assert gt.balance() == 0
        for _ in range(maxl - base + 1):
            gt.adapt(-torch.ones(gt.num_leaves(), dtype=torch.int8, device="cuda"))
        assert torch.equal(gt.keys(), k0)


def test_periodic_one_and_two_cells_wide():
    """Reading D-6: a periodic axis one cell wide makes a leaf its own neighbour."""
    for base in (0, 1):
        for dim in (2, 3):
            gt = lt.Tree(dim, base, 3, None, (1,) * dim)
            ot = oracle.Tree(dim, base, 3, (1,) * dim)
            P.assert_faces_equal(gt.connect(), ot.connect(), "periodic base %d" % base)


def test_bad_arguments():
    import ctypes as C
    L = lt.lib()
    h = C.c_void_p()
    assert L.lt_build(4, 1, 2, None, None, None, C.byref(h)) == lt.LT_ERR_ARG
    assert L.lt_build(3, 3, 2, None, None, None, C.byref(h)) == lt.LT_ERR_ARG
    assert L.lt_build(3, 1, 20, None, None, None, C.byref(h)) == lt.LT_ERR_ARG
    assert L.lt_build(2, 1, 30, None, None, None, C.byref(h)) == lt.LT_ERR_ARG
    gt = lt.Tree(2, 1, 3)
    assert L.lt_adapt(gt._h, None) == lt.LT_ERR_ARG
    assert L.lt_transfer(gt._h, None, None, 2, 4) == lt.LT_ERR_ARG
    u = torch.zeros(4 * 9, dtype=torch.float64, device="cuda")
    assert L.lt_transfer(gt._h, C.c_void_p(u.data_ptr()), C.c_void_p(u.data_ptr()), 8, 1) == lt.LT_ERR_ARG
    assert L.lt_connect(gt._h, None) == lt.LT_ERR_ARG


def test_capacity_growth():
    """Buffers grow on demand (adapt) and the balance retries after LT_ERR_CAPACITY."""
    cfg = W.CONFIGS["c3b"]
    gt, ot = P.new_pair(cfg)
    for c in range(9):
        f = P.host_flags(cfg, c, ot)
        ot.adapt(f)
        gt.adapt(torch.from_numpy(f).cuda())
    gt.set_option(lt.LT_OPT_DEBUG_BALANCE_SLACK, 16)  # forces several capacity retries
    it_g, it_o = gt.balance(), ot.balance()
    assert it_g >= it_o  # a retry restarts with a full sweep; the tree must still be the same
    P.assert_keys_equal(gt, ot, "after growth")
    # adapt grows buffers on demand
    g2 = lt.Tree(2, 2, 9)
    for _ in range(5):
        g2.adapt(torch.ones(g2.num_leaves(), dtype=torch.int8, device="cuda"))
    assert g2.num_leaves() == 16 * 4 ** 5
    P.assert_keys_equal(g2, oracle.Tree(2, 7, 9), "grown uniform")
    gt.reserve(100000)
    P.assert_keys_equal(gt, ot, "after reserve")
    P.assert_faces_equal(gt.connect(), ot.connect(), "after reserve")


def test_connect_begin_end_overlaps_transfer():
    # lt_connect_begin / lt_transfer / lt_connect_end: the face query runs on the tree's side stream
    # beside the transfer; faces, map and solution must equal the oracle's, cycle after cycle
    cfg = dict(W.CONFIGS["c4"], base=3, maxl=6)
    gt, ot = P.new_pair(cfg)
    p, nvars = cfg["p"], cfg["nvars"]
    uo = P.initial_u(cfg, ot)
    with pytest.raises(lt.LtError):
        gt.connect_end()  # nothing pending
    for c in range(4):
        f = P.host_flags(cfg, c, ot)
        ot.adapt(f); ot.balance()
        gt.adapt(torch.from_numpy(f).cuda()); gt.balance()
        gt.connect_begin()
        un_g = gt.transfer(torch.from_numpy(uo).cuda(), p, nvars)
        Fg = gt.connect_end()
        P.assert_faces_equal(Fg, ot.connect(), "cycle %d faces (async)" % c)
        un_o = ot.transfer(uo, p, nvars)
        gt.sync()
        P.assert_u_close(un_g, un_o, "cycle %d transfer beside the face query" % c)
        uo = un_o
    # a pending query is joined by the next mutating call; the mortar calls refuse stale faces
    gt.connect_begin()
    with pytest.raises(lt.LtError):
        gt.mortar_project(torch.zeros((gt.num_leaves(), 6, 1, 4), dtype=torch.float64, device="cuda"), 1, 1)
    f = P.host_flags(cfg, 4, ot)
    ot.adapt(f); ot.balance()
    gt.adapt(torch.from_numpy(f).cuda()); gt.balance()
    P.assert_keys_equal(gt, ot, "adapt after an uncollected connect_begin")
    P.assert_faces_equal(gt.connect(), ot.connect(), "sync connect afterwards")


@pytest.mark.parametrize("dim,base,maxl,periodic", [(2, 2, 7, (1, 0)), (3, 1, 5, (1, 1, 1)), (3, 2, 5, (0, 0, 0))])
def test_balance_after_adapt_uses_the_adapt_frontier(dim, base, maxl, periodic):
    # lt_balance's first sweep looks only at the leaves lt_adapt created (children examined as fine
    # leaves, merged parents checked from their own side); with coarsening-heavy random flags the
    # result, the sweep count and the split count must still be the oracle's -- and the same as with
    # full sweeps
    rng = np.random.default_rng(dim * 100 + maxl)
    dom = [0.0] * dim + [1.0] * dim
    gt, gf = lt.Tree(dim, base, maxl, dom, periodic), lt.Tree(dim, base, maxl, dom, periodic)
    gf.set_option(lt.LT_OPT_BALANCE_FULL_SWEEPS, 1)
    ot = oracle.Tree(dim, base, maxl, periodic)
    for c in range(10):
        pr = [0.45, 0.25, 0.30] if c % 2 else [0.15, 0.25, 0.60]   # coarsen-heavy / refine-heavy
        f = rng.choice(np.array([-1, 0, 1], np.int8), size=ot.num_leaves(), p=pr)
        ot.adapt(f); it_o = ot.balance(); ot.drop_snapshot()
        for g in (gt, gf):
            g.adapt(torch.from_numpy(f).cuda())
            assert g.balance() == it_o, "cycle %d" % c
            P.assert_keys_equal(g, ot, "cycle %d" % c)
        if c == 4:  # two adapts without a balance in between: the second one has no valid frontier
            f2 = rng.choice(np.array([-1, 0, 1], np.int8), size=ot.num_leaves(), p=[0.2, 0.5, 0.3])
            ot.adapt(f2); ot.drop_snapshot()
            gt.adapt(torch.from_numpy(f2).cuda()); gf.adapt(torch.from_numpy(f2).cuda())


# ---------------------------------------------------------------- the one-synchronisation cycle
@pytest.mark.parametrize("name,ncyc", [("c1", 4), ("c2", 9), ("c3b", 12), ("c4", 3), ("slab", 8)])
def test_cycle_with_one_host_synchronisation(name, ncyc):
    """With buffers reserved for the worst case (2^dim * leaves) lt_adapt and lt_balance(iters = NULL)
    only enqueue: the leaf count and the buffer the balanced tree ends in stay on the device,
    lt_connect_begin / lt_transfer read them there, and lt_connect_end is the only call that makes the
    host wait.  Same results as the synchronous calls, bit for bit, against the oracle."""
    cfg = W.CONFIGS[name]
    gt, ot = P.new_pair(cfg)
    p, nvars = cfg["p"], cfg["nvars"]
    N = (p + 1) ** cfg["dim"]
    uo = P.initial_u(cfg, ot)
    cap = 1 << 14
    for c in range(ncyc):
        while cap < (8 << cfg["dim"]) * ot.num_leaves():
            cap *= 4
        gt.reserve(cap)
        f = P.host_flags(cfg, c, ot)
        d_f = torch.from_numpy(f).cuda()
        d_uo = torch.from_numpy(uo).cuda()
        d_un = torch.empty((cap, nvars, N), dtype=torch.float64, device="cuda")
        torch.cuda.synchronize()
        s0 = gt.host_syncs()
        gt.adapt(d_f)
        gt.balance(want_iters=False)
        gt.connect_begin()
        gt.transfer_into(d_uo, d_un, p, nvars)
        Fg = gt.connect_end()
        assert gt.host_syncs() - s0 == 1, "cycle %d: %d host synchronisations" % (c, gt.host_syncs() - s0)
        ot.adapt(f)
        it_o = ot.balance()
        assert gt.last_balance_iters() == it_o
        P.assert_keys_equal(gt, ot, "cycle %d" % c)
        P.assert_faces_equal(Fg, ot.connect(), "cycle %d faces" % c)
        src_o, kind_o = ot.build_map()
        un_o = ot.transfer_rows(uo, p, nvars, 0, ot.num_leaves())
        ot.drop_snapshot()
        gt.sync()
        src_g, kind_g = gt.map()
        assert np.array_equal(src_g.cpu().numpy(), src_o) and np.array_equal(kind_g.cpu().numpy(), kind_o)
        P.assert_u_close(d_un[:ot.num_leaves()], un_o, "cycle %d transfer" % c)
        uo = un_o


def test_deferred_balance_reports_a_mapping_error_through_the_status():
    """Two adapts, then a balance that does not wait: the Alg. 7 tail finds leaves two levels from the
    snapshot; lt_transfer moves nothing and lt_sync returns LT_ERR_MAPPING."""
    cfg = W.CONFIGS["c3b"]
    gt, ot = P.new_pair(cfg)
    gt.reserve(1 << 16)
    for c in range(9):
        f = P.host_flags(cfg, c, ot)
        ot.adapt(f)
        gt.adapt(torch.from_numpy(f).cuda())
    # (the tree entering the last lt_adapt was not balanced, so this lt_balance takes the waiting path;
    # its tail still leaves the map to lt_transfer's checked k_map)
    gt.balance(want_iters=False)
    u = torch.zeros((gt.num_old_leaves(), 5, 8), dtype=torch.float64, device="cuda")
    gt.transfer(u, 1, 5)
    with pytest.raises(lt.LtError) as ei:
        gt.sync()
    assert ei.value.status == lt.LT_ERR_MAPPING
    assert gt.num_leaves() == 932


@pytest.mark.parametrize("base,maxl,p,nvars,recipes", [
    (2, 5, 1, 2, ["refine"] * 3 + ["coarsen", "mixed", "coarsen_half", "mixed"]),
    (4, 7, 0, 1, ["refine"] * 3 + ["coarsen", "mixed"]),
])
def test_map_from_the_window_and_from_the_per_leaf_search(base, maxl, p, nvars, recipes):
    """Alg. 7 in the tail of lt_balance locates a tile of 1024 new leaves in a shared-memory window of
    2048 old keys and falls back to the per-leaf bucketed search when the tile's old range does not fit (a
    tile of merged parents spans 2^dim old leaves per new one).  The small case stays inside the window;
    coarsen-everything on a uniform 128^3 tree (262 144 parents of 2 097 152 leaves: 512 parents per block
    chunk, 4096 old keys per tile) takes the fallback in every tile, the mixed cycle after it both.  Map,
    keys and the transferred solution must be the oracle's either way."""
    dim = 3
    gt = lt.Tree(dim, base, maxl, None, (1, 0, 1))
    ot = oracle.Tree(dim, base, maxl, (1, 0, 1))
    rng = np.random.default_rng(7)
    uo = rng.uniform(-1, 1, (ot.num_leaves(), nvars, (p + 1) ** dim))
    for c, what in enumerate(recipes):
        n = ot.num_leaves()
        lvl, xyz = ot.leaf_boxes()
        if what == "refine":
            f = np.ones(n, np.int8)
        elif what == "coarsen":
            f = -np.ones(n, np.int8)
        elif what == "coarsen_half":
            f = np.where(xyz[:, 0] < (1 << (maxl - 1)), -1, 0).astype(np.int8)
        else:
            f = rng.choice(np.array([-1, 0, 1], np.int8), size=n, p=[0.5, 0.3, 0.2])
        ot.adapt(f)
        gt.adapt(torch.from_numpy(f).cuda())
        assert gt.balance() == ot.balance(), "cycle %d" % c
        P.assert_keys_equal(gt, ot, "cycle %d (%s)" % (c, what))
        src_o, kind_o = ot.build_map()
        un_o = ot.transfer_rows(uo, p, nvars, 0, ot.num_leaves())
        ot.drop_snapshot()
        un_g = gt.transfer(torch.from_numpy(uo).cuda(), p, nvars)
        gt.sync()
        src_g, kind_g = gt.map()
        assert np.array_equal(src_g.cpu().numpy(), src_o), "cycle %d (%s): map src" % (c, what)
        assert np.array_equal(kind_g.cpu().numpy(), kind_o), "cycle %d (%s): map kind" % (c, what)
        P.assert_u_close(un_g, un_o, "cycle %d (%s)" % (c, what))
        uo = un_o
