"""-m gpu: the CUDA path (through the C ABI, via the ctypes binding) against the CPU oracle,
element by element, bit-exact (every output is integer / index work), on the same seeded inputs.
Sizes span several sort tiles (2048), scan chunks and ragged tails."""
import numpy as np
import pytest
import torch

import oracle
from harness import workloads as W

pytestmark = pytest.mark.gpu

DEV = "cuda:0"


def _b():
    from paper_2607_02525_b200 import binding
    return binding


def _dev(a, dtype=None):
    t = torch.from_numpy(np.ascontiguousarray(a))
    if dtype is not None:
        t = t.view(dtype)
    return t.to(DEV)


def _np(t, dtype=None):
    a = t.cpu()
    if a.dtype == torch.uint64:
        return a.view(torch.int64).numpy().view(np.uint64)
    return a.numpy()


def _radix_dev(r):
    b = _b()
    return b.Radix(_dev(r.c_tokens), _dev(r.n_tok_off), _dev(r.n_tok_len), _dev(r.n_child_off),
                   _dev(r.e_first_tok), _dev(r.e_child))


def _orc_radix(r):
    return oracle.Radix(r.c_tokens, r.n_tok_off, r.n_tok_len, r.n_child_off, r.e_first_tok, r.e_child)


def run_pipeline(toks, off, radix, t_keys, arrival, check_tree_free=True):
    """GPU pipeline vs oracle on CSR tokens (numpy).  radix: workloads.RadixArrays or None."""
    b = _b()
    N = off.shape[0] - 1
    o_bo, o_h = oracle.block_hash(toks, off, 16, 0)
    NB = int(o_bo[-1])
    d_tok = _dev(toks) if toks.shape[0] else torch.zeros(0, dtype=torch.int32, device=DEV)
    d_off = _dev(off)
    g_bo, g_h = b.peek_block_hash(d_tok, d_off, NB)
    assert np.array_equal(_np(g_bo), o_bo)
    assert np.array_equal(_np(g_h), o_h)

    ot = oracle.pending_tree(o_h, o_bo)
    gt = b.peek_pending_tree(g_h, g_bo)
    assert np.array_equal(_np(gt.order), ot.order)
    assert np.array_equal(_np(gt.lcp), ot.lcp)
    assert np.array_equal(_np(gt.group_id), ot.group_id)
    assert np.array_equal(_np(gt.group_size), ot.group_size)
    assert int(gt.n_groups.item()) == ot.n_groups
    assert np.array_equal(_np(gt.cluster_depth), ot.cluster_depth)
    assert np.array_equal(_np(gt.cluster_size), ot.cluster_size)
    assert np.array_equal(_np(gt.cluster_id), ot.cluster_id)

    d_keys = _dev(t_keys.view(np.int64), torch.uint64) if t_keys is not None else None
    d_radix = _radix_dev(radix) if radix is not None else None
    o_hr = oracle.lpm_radix(toks, off, _orc_radix(radix)) if radix is not None else None
    o_hh = oracle.lpm_hash(o_h, o_bo, t_keys) if t_keys is not None else None
    # every co-descent strategy (dual-walk at several window sizes, speculative + scan) and the
    # naive per-request walk (no tree view) must all equal the oracle
    variants = [(gt, b.LPM_DUAL_WALK, 0), (gt, b.LPM_DUAL_WALK, 1), (gt, b.LPM_DUAL_WALK, 5),
                (gt, b.LPM_DUAL_WALK, 32), (gt, b.LPM_DUAL_WALK, 64), (gt, b.LPM_SPECULATIVE, 0),
                (gt, b.LPM_AUTO, 0)]
    if check_tree_free:
        variants.append((None, b.LPM_AUTO, 0))
    try:
        for tree, strategy, window in variants:
            b.set_option(b.OPT_LPM_STRATEGY, strategy)
            b.set_option(b.OPT_LPM_WINDOW, window)
            g_hr, g_hh = b.peek_lpm(d_tok, d_off, g_h, g_bo, radix=d_radix, t_keys=d_keys, tree=tree)
            what = "tree=%s strategy=%d window=%d" % (tree is not None, strategy, window)
            if radix is not None:
                assert np.array_equal(_np(g_hr), o_hr), "hit_radix " + what
            if t_keys is not None:
                assert np.array_equal(_np(g_hh), o_hh), "hit_hash " + what
    finally:
        b.set_option(b.OPT_LPM_STRATEGY, b.LPM_AUTO)
        b.set_option(b.OPT_LPM_WINDOW, 0)

    if radix is not None:  # per-radix-node demand from the (verified) radix hits
        g_nd = b.peek_radix_demand(d_tok, d_off, d_radix, _dev(o_hr))
        assert np.array_equal(_np(g_nd), oracle.radix_demand(toks, off, _orc_radix(radix))), "node_demand"

    hit_np = o_hr if o_hr is not None else o_hh
    d_hit = _dev(hit_np)
    d_arr = _dev(arrival) if arrival is not None else None
    g_dem, g_ord = b.peek_demand_rank(g_h, g_bo, tree=gt, t_keys=d_keys, hit=d_hit,
                                      cluster_size=gt.cluster_size, arrival=d_arr)
    if t_keys is not None:
        assert np.array_equal(_np(g_dem), oracle.demand(o_h, o_bo, t_keys))
    assert np.array_equal(_np(g_ord), oracle.clpm_order(hit_np, ot.cluster_size, arrival))
    check_next_rows(b, g_h, g_bo, gt, o_h, o_bo, ot, hit_np, arrival, t_keys, d_keys)
    torch.cuda.synchronize()
    return dict(N=N, NB=NB)


def check_next_rows(b, g_h, g_bo, gt, o_h, o_bo, ot, hit_np, arrival, t_keys, d_keys):
    """peek_clpm_signals / peek_clpm_order_full against the oracle."""
    d_hit = _dev(hit_np)
    d_arr = _dev(arrival) if arrival is not None else None
    o_score = oracle.score(o_h, o_bo, 16)
    taus = [0, int(np.median(hit_np))] if hit_np.shape[0] else [0]
    for tau in taus:
        g_sec, g_score, g_ev = b.peek_clpm_signals(g_h, g_bo, gt, hit=d_hit, tau=tau, arrival=d_arr, t_keys=d_keys)
        o_sec = oracle.sections(o_h, o_bo, hit_np, tau, arrival)
        assert np.array_equal(_np(g_sec), o_sec), "section tau=%d" % tau
        assert np.array_equal(_np(g_score), o_score), "score"
        if t_keys is not None:
            assert np.array_equal(_np(g_ev), oracle.evict_score(o_h, o_bo, t_keys, 16)), "evict_score"
        # every oracle input below is the oracle's own (never a CUDA output)
        o_full = oracle.clpm_order_full(o_sec, hit_np, o_score, ot.cluster_size, arrival)
        o_lb = oracle.lane_b(o_sec, hit_np, arrival)
        g_full = b.peek_clpm_order_full(g_sec, d_hit, g_score, gt.cluster_size, d_arr)
        assert np.array_equal(_np(g_full), o_full), "full cLPM order tau=%d" % tau
        g_lb = b.peek_clpm_lane_b(g_sec, d_hit, d_arr)
        assert np.array_equal(_np(g_lb), o_lb), "lane B order"
        for alpha in (0.7, 0.4):
            g_adm = b.peek_stride_interleave(g_full, g_lb, alpha)
            assert np.array_equal(_np(g_adm), oracle.stride_interleave(o_full, o_lb, alpha)), "interleave"
        g_gm = b.peek_clpm_group_major(g_full, gt.cluster_id)
        assert np.array_equal(_np(g_gm), oracle.group_major(o_full, ot.cluster_id)), "group-major order"
    for age, prev in ((0.0, 0.15), (0.37, 0.3), (1.0, 0.6)):
        g_dl = b.peek_dynamic_lane(gt.cluster_size, age, prev).cpu().numpy()
        assert g_dl.tolist() == list(oracle.dynamic_lane(ot.cluster_size, age, prev)), "dynamic lane"
    for depth in (8, 3):
        g_off, g_guards = b.peek_offline_phase1(g_h, g_bo, depth)
        o_off, o_guards = oracle.offline_phase1(o_h, o_bo, depth)
        assert np.array_equal(_np(g_off), o_off), "offline phase 1 order depth=%d" % depth
        assert np.array_equal(g_guards.cpu().numpy(), o_guards), "offline guards depth=%d" % depth


@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5])
@pytest.mark.parametrize("seed", [42, 142])
def test_small_configs(cfg, seed):
    wl = W.make(cfg, seed=seed, small=True)
    toks, off = wl.queue.materialize_np()
    cache = W.build_cache(wl, lambda t, o: oracle.block_hash(t, o, 16, 0))
    run_pipeline(toks, off, cache.radix, cache.t_keys, wl.arrival)


def _csr(seqs):
    off = np.zeros(len(seqs) + 1, dtype=np.int64)
    off[1:] = np.cumsum([len(s) for s in seqs])
    toks = np.concatenate([np.asarray(s, dtype=np.int32) for s in seqs]) if off[-1] else np.zeros(0, np.int32)
    return toks.astype(np.int32), off


def _cache_from(seqs, slots):
    toks, off = _csr(seqs)
    n = len(seqs)
    pcs = W.Pieces(toks, off[:-1].copy(), np.diff(off), np.arange(n + 1, dtype=np.int64))
    radix, _ = W.build_radix(pcs, 16, 0)
    _, keys = oracle.block_hash(toks, off, 16, 0)
    return radix, W.build_table(keys, slots)


def test_edge_cases_tiny_vocab():
    """Tiny vocab so prefixes collide at every depth; empty, sub-block, duplicate and
    prefix-of-another requests; arrival = NULL."""
    rng = np.random.default_rng(5)
    stems = [rng.integers(0, 3, size=int(rng.integers(1, 200))).astype(np.int32) for _ in range(6)]
    reqs = [np.zeros(0, np.int32), np.zeros(5, np.int32), np.zeros(16, np.int32), np.zeros(16, np.int32)]
    for _ in range(700):
        s = stems[int(rng.integers(0, 6))]
        cut = int(rng.integers(0, len(s) + 1))
        tail = rng.integers(0, 3, size=int(rng.integers(0, 60))).astype(np.int32)
        reqs.append(np.concatenate([s[:cut], tail]))
    reqs += [reqs[10].copy(), reqs[10][: len(reqs[10]) // 2].copy(), reqs[11].copy()]
    toks, off = _csr(reqs)
    radix, t_keys = _cache_from([s for s in stems] + [reqs[20], reqs[21]], 1 << 10)
    run_pipeline(toks, off, radix, t_keys, None)


def test_empty_cache_and_self_cache():
    rng = np.random.default_rng(9)
    reqs = [rng.integers(0, 1000, size=int(rng.integers(0, 300))).astype(np.int32) for _ in range(300)]
    toks, off = _csr(reqs)
    # empty cache: V = 1, all-EMPTY table
    radix, _ = W.build_radix(None, 16, 0)
    t_keys = np.full(64, W.EMPTY, dtype=np.uint64)
    run_pipeline(toks, off, radix, t_keys, None)
    # the cache is the requests themselves: hit_radix = len, hit_hash = 16 * nb
    radix, t_keys = _cache_from([r for r in reqs if len(r)], 1 << 14)
    run_pipeline(toks, off, radix, t_keys, rng.permutation(len(reqs)).astype(np.int32))


def test_single_and_identical():
    one = [np.arange(100, dtype=np.int32)]
    toks, off = _csr(one)
    radix, t_keys = _cache_from(one, 64)
    run_pipeline(toks, off, radix, t_keys, None)
    same = [np.arange(64, dtype=np.int32)] * 2500
    toks, off = _csr(same)
    run_pipeline(toks, off, radix, t_keys, None)


def test_wide_root_fanout_and_long_edges():
    """Root with thousands of children (32-ary child search) and a 40k-token edge."""
    rng = np.random.default_rng(11)
    cached = [np.concatenate([[i * 7], rng.integers(0, 128256, size=30)]).astype(np.int32) for i in range(5000)]
    long = rng.integers(0, 128256, size=40000).astype(np.int32)
    cached.append(long)
    reqs = [c[: int(rng.integers(1, 32))] for c in cached[:800]]
    reqs += [np.concatenate([long[: int(rng.integers(1, 40000))], rng.integers(0, 9, size=40)]).astype(np.int32)
             for _ in range(40)]
    reqs += [rng.integers(-5, 128256, size=50).astype(np.int32) for _ in range(100)]
    toks, off = _csr(reqs)
    radix, t_keys = _cache_from(cached, 1 << 18)
    run_pipeline(toks, off, radix, t_keys, rng.permutation(len(reqs)).astype(np.int32))


def test_arg_errors():
    b = _b()
    L = b.lib()
    assert L.peek_block_hash(None, None, -1, 16, 0, None, None, 0, None, 0, None) == -1
    assert L.peek_block_hash(None, None, 4, 8, 0, None, None, 0, None, 0, None) == -5
    assert L.peek_block_hash(None, None, 0, 16, 0, None, None, 0, None, 0, None) == 0
    assert L.peek_pending_tree(None, None, 0, None, None, None, None, None, None, None, None, None, 0, None) == 0
    off = torch.zeros(5, dtype=torch.int64, device=DEV)
    with pytest.raises(b.PeekError):
        b.peek_lpm(None, off, None, off, radix=None, t_keys=torch.zeros(6, dtype=torch.uint64, device=DEV))


def test_errors_leave_outputs_untouched():
    """include/peek.h: argument and workspace errors are detected before anything is enqueued."""
    b = _b()
    L = b.lib()
    rng = np.random.default_rng(4)
    reqs = [rng.integers(0, 50, size=64).astype(np.int32) for _ in range(40)]
    toks, off = _csr(reqs)
    o_bo, o_h = oracle.block_hash(toks, off, 16, 0)
    d_h, d_bo = _dev(o_h.view(np.int64), torch.uint64), _dev(o_bo)
    tree = b.peek_pending_tree(d_h, d_bo)
    keys = torch.full((64,), -1, dtype=torch.int64, device=DEV).view(torch.uint64)
    demand = torch.full((64,), 7, dtype=torch.int32, device=DEV)
    evict = torch.full((64,), 7, dtype=torch.int64, device=DEV)
    tbl = b._Table(b._ptr(keys), 64)
    import ctypes
    small = torch.zeros(256, dtype=torch.uint8, device=DEV)
    p = b._ptr
    st = L.peek_demand_rank(p(d_h), p(d_bo), 40, p(tree.order), p(tree.lcp), ctypes.byref(tbl), None, None, None,
                            p(demand), None, p(small), 256, None)
    assert st == -3  # PEEK_ERR_WORKSPACE
    st2 = L.peek_clpm_signals(p(d_h), p(d_bo), 40, p(tree.order), p(tree.lcp), None, 0, None, ctypes.byref(tbl),
                              None, None, p(evict), p(small), 256, None)
    assert st2 == -3
    st3 = L.peek_clpm_signals(None, p(d_bo), 40, p(tree.order), p(tree.lcp), None, 0, None, ctypes.byref(tbl),
                              None, None, p(evict), p(small), 256, None)
    assert st3 == -1  # PEEK_ERR_INVALID_ARG: evict_score needs hashes
    torch.cuda.synchronize()
    assert bool((demand == 7).all()) and bool((evict == 7).all())
    assert L.peek_pending_tree(None, p(d_bo), 40, p(tree.order), p(tree.lcp), None, None, None, None, None, None,
                               p(small), 256, None) == -1
    assert L.peek_offline_phase1(None, p(d_bo), 40, 8, p(tree.order), p(evict), p(small), 256, None) == -1


def _nested_queue(rng, n, vocab=4):
    """Short requests over a tiny vocabulary: deep nesting, duplicates, prefix-of relations."""
    stems = [rng.integers(0, vocab, size=int(rng.integers(16, 400))).astype(np.int32) for _ in range(40)]
    reqs = []
    for _ in range(n):
        s = stems[int(rng.integers(0, len(stems)))]
        cut = int(rng.integers(0, len(s) + 1))
        tail = rng.integers(0, vocab, size=int(rng.integers(0, 48))).astype(np.int32)
        reqs.append(np.concatenate([s[:cut], tail]))
    return reqs, stems


@pytest.mark.parametrize("grid_limit", [1, 3, 0])
def test_persistent_kernels_multi_tile(grid_limit):
    """peek_pending_tree / peek_demand_rank with the cooperative grid capped (PEEK_OPT_GRID_LIMIT):
    with 1 or 3 CTAs every CTA owns several 8192-position tiles, so the tile loops, the carries
    across tiles and CTAs and the multi-tile sort passes all run; results never depend on it."""
    b = _b()
    rng = np.random.default_rng(77)
    reqs, stems = _nested_queue(rng, 30011)
    toks, off = _csr(reqs)
    radix, t_keys = _cache_from(stems[:20], 1 << 13)
    b.set_option(b.OPT_GRID_LIMIT, grid_limit)
    try:
        run_pipeline(toks, off, radix, t_keys, rng.permutation(len(reqs)).astype(np.int32),
                     check_tree_free=False)
    finally:
        b.set_option(b.OPT_GRID_LIMIT, 0)


def _tree_only(b, reqs):
    """peek_pending_tree alone against the oracle, every output."""
    toks, off = _csr(reqs)
    o_bo, o_h = oracle.block_hash(toks, off, 16, 0)
    d_h = _dev(o_h.view(np.int64), torch.uint64) if o_h.shape[0] else torch.zeros(0, dtype=torch.uint64, device=DEV)
    gt = b.peek_pending_tree(d_h, _dev(o_bo))
    ot = oracle.pending_tree(o_h, o_bo)
    for name in ("order", "lcp", "group_id", "group_size", "cluster_depth", "cluster_size", "cluster_id"):
        assert np.array_equal(_np(getattr(gt, name)), getattr(ot, name)), name
    assert int(gt.n_groups.item()) == ot.n_groups


@pytest.mark.parametrize("local_cap", [128, 700, 4096, 0])
@pytest.mark.parametrize("grid_limit", [2, 0])
def test_pending_tree_local_stage(local_cap, grid_limit):
    """peek_pending_tree's two stages with the local capacity lowered (PEEK_OPT_TREE_LOCAL_CAP): segments
    above the capacity go through more grid-wide rounds, those above the quantum are work items of
    their own, the rest is taken a quantum of positions at a time - deeply nested queues (tiny
    vocabulary), flat ones (big vocabulary), many duplicates, and sizes around the capacities."""
    b = _b()
    rng = np.random.default_rng(1234 + local_cap)
    b.set_option(b.OPT_TREE_LOCAL_CAP, local_cap)
    b.set_option(b.OPT_GRID_LIMIT, grid_limit)
    try:
        for n in (127, 129, 1500, 12288, 12289, 30011):
            reqs, _ = _nested_queue(rng, n)
            _tree_only(b, reqs)
        flat = [rng.integers(0, 128256, size=int(rng.integers(0, 200))).astype(np.int32) for _ in range(20000)]
        _tree_only(b, flat)
        base = rng.integers(0, 9, size=4000).astype(np.int32)
        nested = [base[: int(rng.integers(0, 4000))] for _ in range(9000)]  # every request a prefix of one chain
        _tree_only(b, nested)
        dup = [flat[int(rng.integers(0, 50))] for _ in range(14000)]        # 50 distinct chains
        _tree_only(b, dup)
        shared = [np.concatenate([base[:1600], rng.integers(0, 3, size=int(rng.integers(0, 90)))]).astype(np.int32)
                  for _ in range(15000)]                                    # one long shared prefix
        _tree_only(b, shared)
    finally:
        b.set_option(b.OPT_TREE_LOCAL_CAP, 0)
        b.set_option(b.OPT_GRID_LIMIT, 0)


def test_lpm_work_counters():
    """The amortisation claim (Fig. 6(a); SURVEY.md section 4 "work-counter tests"):
    five requests under a shared system prefix, clusters A x3 and B x2, the cache holds sys and
    sys+A.  Stock LPM (no tree view) walks from the root once per request and compares every
    request's whole cached prefix; the dual walk starts ONE walk at the root, compares every cached
    token once, and reaches the other requests by child lookups below the shared prefixes."""
    b = _b()
    rng = np.random.default_rng(66)
    tok = lambda n: rng.integers(0, 128256, size=n).astype(np.int32)
    sys_p, a_p, b_p = tok(160), tok(96), tok(64)
    reqs = [np.concatenate([sys_p, a_p, tok(40)]) for _ in range(3)] + [np.concatenate([sys_p, b_p, tok(40)]) for _ in range(2)]
    toks, off = _csr(reqs)
    radix, t_keys = _cache_from([sys_p, np.concatenate([sys_p, a_p])], 256)
    o_bo, o_h = oracle.block_hash(toks, off, 16, 0)
    o_hr = oracle.lpm_radix(toks, off, _orc_radix(radix))
    d_tok, d_off, d_h, d_bo = _dev(toks), _dev(off), _dev(o_h.view(np.int64), torch.uint64), _dev(o_bo)
    d_radix, d_keys = _radix_dev(radix), _dev(t_keys.view(np.int64), torch.uint64)
    tree = b.peek_pending_tree(d_h, d_bo)
    cnt = torch.zeros(4, dtype=torch.uint64, device=DEV)
    read = lambda: cnt.cpu().view(torch.int64).tolist()
    b.lpm_counters(cnt)
    try:
        b.set_option(b.OPT_LPM_STRATEGY, b.LPM_DUAL_WALK)
        b.set_option(b.OPT_LPM_WINDOW, 8)
        hr, hh = b.peek_lpm(d_tok, d_off, d_h, d_bo, radix=d_radix, t_keys=d_keys, tree=tree)
        torch.cuda.synchronize()
        dual = read()
        cnt.zero_()
        b.set_option(b.OPT_LPM_STRATEGY, b.LPM_AUTO)
        hr0, hh0 = b.peek_lpm(d_tok, d_off, d_h, d_bo, radix=d_radix, t_keys=d_keys, tree=None)
        torch.cuda.synchronize()
        naive = read()
    finally:
        b.lpm_counters(None)
        b.set_option(b.OPT_LPM_STRATEGY, b.LPM_AUTO)
        b.set_option(b.OPT_LPM_WINDOW, 0)
    assert np.array_equal(_np(hr), o_hr) and np.array_equal(_np(hr0), o_hr)
    assert o_hr.tolist() == [256, 256, 256, 160, 160]
    # stock LPM: 5 walks from the root in each mode, every request's cached prefix compared in full
    assert naive[0] == 10
    assert naive[2] == int(o_hr.sum())               # every walk ends at a node boundary: matched tokens only
    assert naive[3] == int(np.diff(o_bo).sum())      # a warp probes 32 blocks of a request at once: all of them here
    # dual walk: one walk from the root per mode; sys and A compared once, B's first token once
    assert dual[0] == 2
    assert dual[2] == 160 + 96
    assert dual[2] * 3 < naive[2] and dual[3] * 2 < naive[3]


def test_lpm_both_modes_side_stream():
    """peek_lpm with both modes and a tree view runs the hash probes on the library's side stream
    next to the radix walk (fork/join around the caller's stream).  Same hits as the oracle on the
    default stream, on a user stream, back to back, and under CUDA-graph capture (where the call must
    stay on the capturing stream)."""
    b = _b()
    wl = W.make(5, seed=77, small=True)
    toks, off = wl.queue.materialize_np()
    cache = W.build_cache(wl, lambda t, o: oracle.block_hash(t, o, 16, 0))
    o_bo, o_h = oracle.block_hash(toks, off, 16, 0)
    o_hr = oracle.lpm_radix(toks, off, _orc_radix(cache.radix))
    o_hh = oracle.lpm_hash(o_h, o_bo, cache.t_keys)
    d_tok, d_off, d_h, d_bo = _dev(toks), _dev(off), _dev(o_h.view(np.int64), torch.uint64), _dev(o_bo)
    d_radix, d_keys = _radix_dev(cache.radix), _dev(cache.t_keys.view(np.int64), torch.uint64)
    tree = b.peek_pending_tree(d_h, d_bo)
    call = lambda: b.peek_lpm(d_tok, d_off, d_h, d_bo, radix=d_radix, t_keys=d_keys, tree=tree)
    b.set_option(b.OPT_LPM_STRATEGY, b.LPM_DUAL_WALK)  # the small case would take the one-launch path
    try:
        for _ in range(3):
            hr, hh = call()
            assert np.array_equal(_np(hr), o_hr) and np.array_equal(_np(hh), o_hh)
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):
            outs = [call() for _ in range(4)]
        side.synchronize()
        for hr, hh in outs:
            assert np.array_equal(_np(hr), o_hr) and np.array_equal(_np(hh), o_hh)
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph):
            ghr, ghh = call()
        ghr.zero_(); ghh.zero_()
        graph.replay()
        torch.cuda.synchronize()
        assert np.array_equal(_np(ghr), o_hr) and np.array_equal(_np(ghh), o_hh)
    finally:
        b.set_option(b.OPT_LPM_STRATEGY, b.LPM_AUTO)


def test_lpm_side_stream_two_host_threads():
    """Two host threads, each on its own stream with its own outputs and workspace, call peek_lpm (both
    modes, dual walk) at the same time: they share the library's side stream and its events, which a
    mutex keeps consistent between fork and join.  Every result equals the oracle."""
    import threading
    b = _b()
    wl = W.make(2, seed=91, small=True)
    toks, off = wl.queue.materialize_np()
    cache = W.build_cache(wl, lambda t, o: oracle.block_hash(t, o, 16, 0))
    o_bo, o_h = oracle.block_hash(toks, off, 16, 0)
    o_hr = oracle.lpm_radix(toks, off, _orc_radix(cache.radix))
    o_hh = oracle.lpm_hash(o_h, o_bo, cache.t_keys)
    d_tok, d_off, d_h, d_bo = _dev(toks), _dev(off), _dev(o_h.view(np.int64), torch.uint64), _dev(o_bo)
    d_radix, d_keys = _radix_dev(cache.radix), _dev(cache.t_keys.view(np.int64), torch.uint64)
    tree = b.peek_pending_tree(d_h, d_bo)
    torch.cuda.synchronize()
    b.set_option(b.OPT_LPM_STRATEGY, b.LPM_DUAL_WALK)
    errors = []

    def worker(tid):
        try:
            st = torch.cuda.Stream()
            with torch.cuda.stream(st):
                for it in range(25):
                    hr, hh = b.peek_lpm(d_tok, d_off, d_h, d_bo, radix=d_radix, t_keys=d_keys, tree=tree)
                    if it % 6 == 0:
                        st.synchronize()
                        if not (np.array_equal(_np(hr), o_hr) and np.array_equal(_np(hh), o_hh)):
                            errors.append("thread %d call %d differs" % (tid, it))
                st.synchronize()
                if not (np.array_equal(_np(hr), o_hr) and np.array_equal(_np(hh), o_hh)):
                    errors.append("thread %d last call differs" % tid)
        except Exception as e:  # noqa: BLE001 - reported below
            errors.append("thread %d: %r" % (tid, e))

    try:
        ts = [threading.Thread(target=worker, args=(i,)) for i in range(2)]
        for t in ts:
            t.start()
        for t in ts:
            t.join(timeout=120)
        assert not any(t.is_alive() for t in ts), "a thread hangs"
    finally:
        b.set_option(b.OPT_LPM_STRATEGY, b.LPM_AUTO)
    assert not errors, errors


@pytest.mark.parametrize("cfg,G", [(2, 2), (5, 3), (4, 4)])
def test_sharded_queue_emulated(cfg, G):
    """SURVEY.md section 8(e) through the CUDA calls: the G shards of one queue (by first-block hash) run
    one after the other on this GPU, demand summed, cLPM keys merged - equal to the oracle on the
    whole queue (the collectives themselves are covered by tests/test_sharded_gloo.py)."""
    b = _b()
    from paper_2607_02525_b200 import sharded
    wl = W.make(cfg, seed=42, small=True)
    toks, off = wl.queue.materialize_np()
    cache = W.build_cache(wl, lambda t, o: oracle.block_hash(t, o, 16, 0))
    d_keys = _dev(cache.t_keys.view(np.int64), torch.uint64)
    d_radix = _radix_dev(cache.radix) if cache.radix is not None else None
    res = sharded.sharded_step_emulated(b, _dev(toks), _dev(off), _dev(wl.arrival), d_radix, d_keys,
                                        int(d_keys.shape[0]), G)
    o_bo, o_h = oracle.block_hash(toks, off, 16, 0)
    ot = oracle.pending_tree(o_h, o_bo)
    o_hit = oracle.lpm_radix(toks, off, _orc_radix(cache.radix)) if cache.radix is not None else \
        oracle.lpm_hash(o_h, o_bo, cache.t_keys)
    assert np.array_equal(_np(res.hit), o_hit)
    assert np.array_equal(_np(res.cluster_size), ot.cluster_size)
    assert np.array_equal(_np(res.demand), oracle.demand(o_h, o_bo, cache.t_keys))
    assert np.array_equal(_np(res.clpm_order), oracle.clpm_order(o_hit, ot.cluster_size, wl.arrival))
    assert len(np.unique(_np(res.owner))) > 1 or cfg == 3


def test_pending_tree_scale_shapes():
    """peek_pending_tree at the sizes where its launch plan changes (one CTA up to 2048 requests, item
    capacity and quantum growing with the queue, full capacity from ~90 000 on) and on shapes that
    stress each stage: deep tries (several grid-wide rounds), a few giant clusters (segments far above
    the local capacity), 250 000 requests over 200 distinct chains (huge resolved segments), and a
    multi-turn queue (conversations whose turns are prefixes of one another under shared prompts)."""
    b = _b()
    rng = np.random.default_rng(7)
    for n in (2048, 2049, 11265, 90113):
        reqs, _ = _nested_queue(rng, n)
        _tree_only(b, reqs)
    bases = [rng.integers(0, 50000, size=int(rng.integers(200, 3000))).astype(np.int32) for _ in range(5)]
    reqs = []
    for _ in range(70000):
        k = int(rng.integers(0, 8))
        if k < 5:
            bse = bases[k]
            reqs.append(np.concatenate([bse[: int(rng.integers(len(bse) // 2, len(bse) + 1))],
                                        rng.integers(0, 50000, size=int(rng.integers(0, 100))).astype(np.int32)]))
        else:
            reqs.append(rng.integers(0, 50000, size=int(rng.integers(0, 300))).astype(np.int32))
    _tree_only(b, reqs)
    pool = [rng.integers(0, 1000, size=int(rng.integers(0, 400))).astype(np.int32) for _ in range(200)]
    _tree_only(b, [pool[int(i)] for i in rng.integers(0, 200, size=250000)])
    prompts = [rng.integers(0, 128256, size=1024).astype(np.int32) for _ in range(12)]
    reqs = []
    for c in range(3000):
        ctx = prompts[int(rng.integers(0, 12))]
        for t in range(int(rng.integers(1, 24))):
            ctx = np.concatenate([ctx, rng.integers(0, 128256, size=int(rng.integers(64, 512))).astype(np.int32)])
            reqs.append(ctx)
    perm = rng.permutation(len(reqs))
    _tree_only(b, [reqs[i] for i in perm])


def test_rank_two_phase_wide_keys():
    """cLPM keys too wide for one 64-bit packed key (full-range hit, cluster size and arrival):
    the arrival sort followed by the stable (hit, cluster size) sort."""
    b = _b()
    rng = np.random.default_rng(3)
    n = 20000
    hit = rng.integers(-2**31, 2**31 - 1, size=n, dtype=np.int64).astype(np.int32)
    hit[::3] = hit[0]  # ties on the leading key
    cs = rng.integers(-2**31, 2**31 - 1, size=n, dtype=np.int64).astype(np.int32)
    cs[::2] = 7
    arr = rng.integers(-2**31, 2**31 - 1, size=n, dtype=np.int64).astype(np.int32)
    arr[::5] = arr[1]  # duplicate arrivals: the request index decides
    for a in (arr, None):
        _, g_ord = b.peek_demand_rank(None, None, tree=None, t_keys=None, hit=_dev(hit),
                                      cluster_size=_dev(cs), arrival=_dev(a) if a is not None else None)
        assert np.array_equal(_np(g_ord), oracle.clpm_order(hit, cs, a))


def test_demand_tagged_probe_dense_table():
    """Tables of 65 536 slots and more are probed through one-byte tags, eight at a time
    (`k_demand<true>`).  A 93 %-full table makes long probe runs that wrap around the end; filler keys
    share the tag (top byte) and the home slot of pending hashes, so tag matches with a different key,
    runs that cross tag words and absent keys behind a matching tag all occur.  demand against the oracle."""
    b = _b()
    rng = np.random.default_rng(4242)
    base = rng.integers(0, 1000, size=16 * 40).astype(np.int32)
    reqs = [np.concatenate([base[:16 * int(rng.integers(1, 40))], rng.integers(0, 1000, size=int(rng.integers(0, 400))).astype(np.int32)])
            for _ in range(3000)]
    toks, off = _csr(reqs)
    o_bo, o_h = oracle.block_hash(toks, off, 16, 0)
    S = 1 << 16
    mask = np.uint64(S - 1)
    uniq = np.unique(o_h)
    cached = uniq[rng.random(uniq.shape[0]) < 0.5]                    # half of the pending blocks are cached
    absent = uniq[~np.isin(uniq, cached)]
    # fillers: same top byte and same home slot as an absent pending hash, different middle bits
    pick = absent[rng.integers(0, absent.shape[0], size=20000)]
    mid = rng.integers(1, 1 << 30, size=pick.shape[0], dtype=np.uint64) << np.uint64(20)
    fill_same = (pick ^ mid) & ~np.uint64(0)
    fill_same = fill_same[~np.isin(fill_same, uniq)]
    # fillers that pile up in the last slots of the table (runs wrap around to slot 0)
    tail = (rng.integers(0, 1 << 40, size=3000, dtype=np.uint64) << np.uint64(16)) | (np.uint64(S - 1) - rng.integers(0, 8, size=3000, dtype=np.uint64))
    rest = rng.integers(0, 2**63, size=S, dtype=np.uint64)
    keys = np.concatenate([cached, fill_same, tail, rest])
    keys = keys[keys != np.uint64(0xFFFFFFFFFFFFFFFF)]
    t_keys = W.build_table(keys, S, max_keys=int(0.93 * S))
    assert (t_keys != np.uint64(0xFFFFFFFFFFFFFFFF)).sum() >= int(0.9 * S)
    d_h, d_bo = _dev(o_h.view(np.int64), torch.uint64), _dev(o_bo)
    tree = b.peek_pending_tree(d_h, d_bo)
    g_dem, _ = b.peek_demand_rank(d_h, d_bo, tree=tree, t_keys=_dev(t_keys.view(np.int64), torch.uint64))
    want = oracle.demand(o_h, o_bo, t_keys)
    assert want.sum() > 0
    assert np.array_equal(_np(g_dem), want)


@pytest.mark.parametrize("n", [1, 2, 31, 200, 511, 512, 513])
def test_rank_small_queue_path(n):
    """Queues of at most 512 requests rank by counting (one CTA, `k_clpm_rank_small`); 513 takes the sort.
    Extreme and heavily tied keys, with and without arrival; the grid-limit test hook must give the
    same order through the general path."""
    b = _b()
    rng = np.random.default_rng(900 + n)
    hit = rng.choice(np.array([-2**31, -1, 0, 16, 160, 2**31 - 1], dtype=np.int64), size=n).astype(np.int32)
    cs = rng.integers(1, 4, size=n).astype(np.int32)
    arr = rng.integers(-5, 5, size=n).astype(np.int32)
    for a in (arr, None):
        want = oracle.clpm_order(hit, cs, a)
        for limit in (0, 1):
            b.set_option(b.OPT_GRID_LIMIT, limit)
            try:
                _, g_ord = b.peek_demand_rank(None, None, tree=None, t_keys=None, hit=_dev(hit),
                                              cluster_size=_dev(cs), arrival=_dev(a) if a is not None else None)
            finally:
                b.set_option(b.OPT_GRID_LIMIT, 0)
            assert np.array_equal(_np(g_ord), want)


@pytest.mark.parametrize("cfg,seed", [(2, 42), (2, 142), (3, 42), (3, 242), (4, 42), (4, 142), (5, 42)])
def test_full_size_configs(cfg, seed):
    """BASELINE.json configs[1..4] at FULL size in the launch configuration bench.py times (config 5:
    N = 1 048 576, 4.28e9 tokens, one CTA per SM): every output of every call against the oracle,
    element by element.  For config 5 the oracle needs the 17 GB of tokens on the host and about
    half a minute."""
    b = _b()
    wl = W.make(cfg, seed=seed)
    d_tok, d_off = wl.queue.materialize(DEV)
    toks = d_tok.cpu().numpy()
    off = d_off.cpu().numpy()
    cache = W.build_cache(wl, lambda t, o: oracle.block_hash(t, o, 16, 0))
    o_bo, o_h = oracle.block_hash(toks, off, 16, 0)
    NB = int(o_bo[-1])
    g_bo, g_h = b.peek_block_hash(d_tok, d_off, NB)
    assert np.array_equal(_np(g_bo), o_bo)
    assert np.array_equal(_np(g_h), o_h)

    gt = b.peek_pending_tree(g_h, g_bo)
    ot = oracle.pending_tree(o_h, o_bo)
    for name in ("order", "lcp", "group_id", "group_size", "cluster_depth", "cluster_size", "cluster_id"):
        assert np.array_equal(_np(getattr(gt, name)), getattr(ot, name)), name
    assert int(gt.n_groups.item()) == ot.n_groups

    d_keys = _dev(cache.t_keys.view(np.int64), torch.uint64)
    d_radix = _radix_dev(cache.radix) if cache.radix is not None else None
    g_hr, g_hh = b.peek_lpm(d_tok, d_off, g_h, g_bo, radix=d_radix, t_keys=d_keys, tree=gt)
    o_hh = oracle.lpm_hash(o_h, o_bo, cache.t_keys)
    assert np.array_equal(_np(g_hh), o_hh)
    o_hit = o_hh
    if cache.radix is not None:
        o_hr = oracle.lpm_radix(toks, off, _orc_radix(cache.radix))
        assert np.array_equal(_np(g_hr), o_hr)
        # mirrored, prefix-closed table: the two modes agree up to block rounding
        assert np.array_equal(o_hh, 16 * (o_hr // 16))
        o_hit = o_hr
        g_nd = b.peek_radix_demand(d_tok, d_off, d_radix, g_hr)
        assert np.array_equal(_np(g_nd), oracle.radix_demand(toks, off, _orc_radix(cache.radix))), "node_demand"

    g_dem, g_ord = b.peek_demand_rank(g_h, g_bo, tree=gt, t_keys=d_keys, hit=_dev(o_hit),
                                      cluster_size=_dev(ot.cluster_size), arrival=_dev(wl.arrival))
    assert np.array_equal(_np(g_dem), oracle.demand(o_h, o_bo, cache.t_keys))
    assert np.array_equal(_np(g_ord), oracle.clpm_order(o_hit, ot.cluster_size, wl.arrival))
    check_next_rows(b, g_h, g_bo, gt, o_h, o_bo, ot, o_hit, wl.arrival, cache.t_keys, d_keys)


def test_block_hash_ragged_queue():
    """peek_block_hash on a ragged queue: every start alignment, empty and sub-block requests, a
    request ending at the very end of the token pool, lengths around the 32-block chunk; two seeds."""
    b = _b()
    rng = np.random.default_rng(21)
    lens = list(range(0, 200)) + [16 * n + d for n in (4, 5, 8, 31, 32, 33, 64, 65, 100) for d in (0, 1, 15)]
    lens += [int(x) for x in rng.integers(0, 5000, size=3000)]
    rng.shuffle(lens)
    lens.append(16 * 7)  # the last request ends exactly at the pool end, on a block boundary
    reqs = [rng.integers(-3, 128256, size=n).astype(np.int32) for n in lens]
    toks, off = _csr(reqs)
    o_bo, o_h = oracle.block_hash(toks, off, 16, 0)
    o_bo2, o_h2 = oracle.block_hash(toks, off, 16, 0x9E3779B97F4A7C15)
    d_tok, d_off = _dev(toks), _dev(off)
    g_bo, g_h = b.peek_block_hash(d_tok, d_off, int(o_bo[-1]))
    assert np.array_equal(_np(g_bo), o_bo)
    assert np.array_equal(_np(g_h), o_h)
    g_bo, g_h = b.peek_block_hash(d_tok, d_off, int(o_bo[-1]), seed=0x9E3779B97F4A7C15)
    assert np.array_equal(_np(g_h), o_h2)


def _update_case(b, old_reqs, keep_mask, arrivals):
    """old queue -> (remove ~keep_mask, append arrivals) -> peek_pending_tree_update must equal the
    oracle's rebuild on the new queue, every output."""
    toks, off = _csr(old_reqs)
    o_bo, o_h = oracle.block_hash(toks, off, 16, 0)
    d_h = _dev(o_h.view(np.int64), torch.uint64) if o_h.shape[0] else torch.zeros(0, dtype=torch.uint64, device=DEV)
    old = b.peek_pending_tree(d_h, _dev(o_bo)) if len(old_reqs) else b.PendingTree(
        *[torch.zeros(0, dtype=torch.int32, device=DEV)] * 6, torch.zeros(0, dtype=torch.int64, device=DEV),
        torch.zeros(1, dtype=torch.int32, device=DEV))
    survivors = [r for r, k in zip(old_reqs, keep_mask) if k]
    remap = np.full(len(old_reqs), -1, dtype=np.int32)
    remap[np.nonzero(keep_mask)[0]] = np.arange(len(survivors), dtype=np.int32)
    new_reqs = survivors + arrivals
    ntoks, noff = _csr(new_reqs)
    n_bo, n_h = oracle.block_hash(ntoks, noff, 16, 0)
    want = oracle.pending_tree(n_h, n_bo)
    dn_h = _dev(n_h.view(np.int64), torch.uint64) if n_h.shape[0] else torch.zeros(0, dtype=torch.uint64, device=DEV)
    d_remap = _dev(remap) if len(old_reqs) else torch.zeros(0, dtype=torch.int32, device=DEV)
    got = b.peek_pending_tree_update(dn_h, _dev(n_bo), len(arrivals), old, d_remap)
    for name in ("order", "lcp", "group_id", "group_size", "cluster_depth", "cluster_size", "cluster_id"):
        assert np.array_equal(_np(getattr(got, name)), getattr(want, name)), name
    assert int(got.n_groups.item()) == want.n_groups
    return got


def test_pending_tree_update_matches_rebuild():
    """removals (scattered, in long runs, all, none) and arrivals (new chains,
    copies of surviving and of removed chains, prefixes and extensions of survivors, empty and
    sub-block prompts), chained over several cycles."""
    b = _b()
    rng = np.random.default_rng(31)
    reqs, stems = _nested_queue(rng, 6000)
    N = len(reqs)

    def arrivals(n, pool):
        out = []
        for _ in range(n):
            kind = int(rng.integers(0, 6))
            base = pool[int(rng.integers(0, len(pool)))]
            if kind == 0:
                out.append(base.copy())
            elif kind == 1:
                out.append(base[: int(rng.integers(0, len(base) + 1))].copy())
            elif kind == 2:
                out.append(np.concatenate([base, rng.integers(0, 4, size=int(rng.integers(1, 60)))]).astype(np.int32))
            elif kind == 3:
                out.append(rng.integers(0, 4, size=int(rng.integers(0, 300))).astype(np.int32))
            elif kind == 4:
                out.append(np.zeros(int(rng.integers(0, 20)), np.int32))
            else:
                s = stems[int(rng.integers(0, len(stems)))]
                out.append(np.concatenate([s[: int(rng.integers(0, len(s) + 1))], rng.integers(0, 4, size=8)]).astype(np.int32))
        return out

    keep = rng.random(N) > 0.02
    _update_case(b, reqs, keep, arrivals(100, reqs))                      # small delta
    keep = rng.random(N) > 0.5
    keep[1000:3000] = False                                               # a long run removed
    _update_case(b, reqs, keep, arrivals(2500, reqs))                     # large delta
    _update_case(b, reqs, np.zeros(N, bool), arrivals(300, reqs))         # everything removed
    _update_case(b, reqs, np.ones(N, bool), [])                           # nothing changes
    _update_case(b, reqs, np.ones(N, bool), arrivals(1, reqs))
    _update_case(b, [], np.zeros(0, bool), arrivals(500, reqs))           # empty old queue
    keep = rng.random(N) > 0.3
    keep[0] = keep[-1] = False
    _update_case(b, reqs, keep, [])                                       # removals only
    # several cycles on top of each other, each from the previous UPDATE result
    cur = reqs
    toks, off = _csr(cur)
    bo, h = oracle.block_hash(toks, off, 16, 0)
    tree = b.peek_pending_tree(_dev(h.view(np.int64), torch.uint64), _dev(bo))
    for cycle in range(4):
        keep = rng.random(len(cur)) > 0.1
        arr = arrivals(400, cur)
        survivors = [r for r, k in zip(cur, keep) if k]
        remap = np.full(len(cur), -1, dtype=np.int32)
        remap[np.nonzero(keep)[0]] = np.arange(len(survivors), dtype=np.int32)
        cur = survivors + arr
        toks, off = _csr(cur)
        bo, h = oracle.block_hash(toks, off, 16, 0)
        tree = b.peek_pending_tree_update(_dev(h.view(np.int64), torch.uint64), _dev(bo), len(arr), tree, _dev(remap))
        want = oracle.pending_tree(h, bo)
        assert np.array_equal(_np(tree.order), want.order) and np.array_equal(_np(tree.lcp), want.lcp), cycle
        assert np.array_equal(_np(tree.cluster_size), want.cluster_size), cycle


def _random_case(seed):
    """A random prefix forest of token segments and a queue drawn from it: exact nodes, prefixes of
    nodes, nodes with random tails; vocab 2 .. 128256 (tiny vocab = collisions at every depth),
    queue sizes around the one-CTA limit (1024) and the tile size (8192), a cache of random nodes
    and requests (possibly empty), arrival a permutation or NULL."""
    rng = np.random.default_rng(seed)
    vocab = int(rng.choice([2, 3, 5, 50, 128256]))
    n = int(rng.choice([1, 2, 7, 33, 200, 1023, 1024, 1025, 3000, 8191, 8193, 20000]))
    levels, fan = int(rng.integers(1, 6)), int(rng.integers(1, 9))
    seg = int(rng.choice([1, 5, 16, 17, 40, 200]))
    nodes, frontier = [np.zeros(0, np.int32)], [0]
    for _ in range(levels):
        nxt = []
        for p in frontier:
            for _ in range(int(rng.integers(1, fan + 1))):
                s = rng.integers(0, vocab, size=int(rng.integers(1, seg + 1))).astype(np.int32)
                nodes.append(np.concatenate([nodes[p], s]))
                nxt.append(len(nodes) - 1)
        frontier = nxt[:4000]
    reqs = []
    for _ in range(n):
        base = nodes[int(rng.integers(0, len(nodes)))]
        mode = int(rng.integers(0, 4))
        if mode == 0:
            r = base
        elif mode == 1:
            r = base[: int(rng.integers(0, len(base) + 1))]
        else:
            r = np.concatenate([base, rng.integers(0, vocab, size=int(rng.integers(0, 3 * seg))).astype(np.int32)])
        reqs.append(r.astype(np.int32))
    toks, off = _csr(reqs)
    ncache = int(rng.integers(0, min(len(nodes), 300) + 1))
    cached = [nodes[int(i)] for i in rng.integers(0, len(nodes), size=ncache) if len(nodes[int(i)])]
    cached += [reqs[int(i)] for i in rng.integers(0, n, size=int(rng.integers(0, 20))) if len(reqs[int(i)])]
    if cached:
        nblk = sum(len(c) // 16 for c in cached) + 8
        radix, t_keys = _cache_from(cached, 1 << int(np.ceil(np.log2(2 * nblk + 2))))
    else:
        radix, _ = W.build_radix(None, 16, 0)
        t_keys = np.full(64, W.EMPTY, dtype=np.uint64)
    arrival = rng.permutation(n).astype(np.int32) if rng.integers(0, 2) else None
    return toks, off, radix, t_keys, arrival


@pytest.mark.parametrize("seed0", [0, 40, 80])
def test_random_forests(seed0):
    """40 random cases per parameter through the whole pipeline (every call, every LPM strategy),
    bit-exact against the oracle.  Seeds 1 and 34 are queues without a single full block / without a
    single token (NB = 0, T = 0: empty hash and token arrays)."""
    for seed in range(seed0, seed0 + 40):
        run_pipeline(*_random_case(seed))


def test_random_forest_updates():
    """peek_pending_tree_update on 60 random forests: a random share of the queue removed (none,
    2 %, half, 98 %, all) and 0 .. N + 3 arrivals (copies, prefixes, extensions, unrelated chains)."""
    b = _b()
    for seed in range(60):
        rng = np.random.default_rng(10_000 + seed)
        toks, off, _, _, _ = _random_case(seed)
        reqs = [toks[off[i]:off[i + 1]].copy() for i in range(len(off) - 1)]
        n = len(reqs)
        keep = rng.random(n) >= float(rng.choice([0.0, 0.02, 0.5, 0.98, 1.0]))
        m = min(int(rng.choice([0, 1, 5, 100, max(1, n // 2), n + 3])), 6000)
        arr = []
        for _ in range(m):
            base = reqs[int(rng.integers(0, n))]
            kind = int(rng.integers(0, 4))
            if kind == 0:
                arr.append(base.copy())
            elif kind == 1:
                arr.append(base[: int(rng.integers(0, len(base) + 1))].copy())
            elif kind == 2:
                arr.append(np.concatenate([base, rng.integers(0, 3, size=int(rng.integers(1, 40)))]).astype(np.int32))
            else:
                arr.append(rng.integers(0, 3, size=int(rng.integers(0, 100))).astype(np.int32))
        _update_case(b, reqs, keep, arr)


def test_stride_interleave_cases():
    """Identical lanes (every candidate clashes), reversed lanes, locally shuffled lanes (clashes in
    most steps, resolved in time order), alpha 0, 1 and next to 1, a queue shorter than one step,
    and sizes around the 1024-slot step and the 2048-entry window."""
    b = _b()
    rng = np.random.default_rng(8)
    for n in (1, 5, 31, 32, 33, 1000, 1023, 1024, 1025, 2047, 2049, 4096, 5000, 50000):
        a = rng.permutation(n).astype(np.int32)
        near = a[np.argsort(np.arange(n) + rng.uniform(0, 300, n), kind="stable")].copy()
        for lane_b in (a.copy(), a[::-1].copy(), near, rng.permutation(n).astype(np.int32)):
            for alpha in (0.0, 0.3, 0.5, 0.7, 0.999, 1.0 - 2.0 ** -40, 1.0):
                got = b.peek_stride_interleave(_dev(a), _dev(lane_b), alpha)
                assert np.array_equal(_np(got), oracle.stride_interleave(a, lane_b, alpha)), (n, alpha)
    n = 1_700_000  # the admitted-bitmap no longer fits shared memory: global-memory bitmap
    a, lane_b = rng.permutation(n).astype(np.int32), rng.permutation(n).astype(np.int32)
    got = b.peek_stride_interleave(_dev(a), _dev(lane_b), 0.7)
    assert np.array_equal(_np(got), oracle.stride_interleave(a, lane_b, 0.7))
