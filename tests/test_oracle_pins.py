"""Pins for the CPU oracle (-m "not gpu").  Every check is against something other than
the oracle itself: values fixed by the paper / the survey's big-int vectors, the plain
definitions in tests/bruteforce.py, closed forms, invariants and textbook reductions
(SURVEY.md section 8(c) P0-P8)."""
import os

import numpy as np
import pytest

import oracle
from harness import workloads as W
from tests import bruteforce as bf

GOLD = os.path.join(os.path.dirname(__file__), "golden", "hash_vectors.txt")


def _orc_radix(r):
    return oracle.Radix(r.c_tokens, r.n_tok_off, r.n_tok_len, r.n_child_off, r.e_first_tok, r.e_child)


def _csr(seqs):
    off = np.zeros(len(seqs) + 1, dtype=np.int64)
    for i, s in enumerate(seqs):
        off[i + 1] = off[i] + len(s)
    toks = np.zeros(max(int(off[-1]), 1), dtype=np.int32)
    for i, s in enumerate(seqs):
        toks[off[i]:off[i + 1]] = s
    return toks[:int(off[-1])], off


def _pieces(seqs):
    toks, off = _csr(seqs)
    n = len(seqs)
    return W.Pieces(np.ascontiguousarray(toks), off[:-1].copy(), np.diff(off), np.arange(n + 1, dtype=np.int64))


def _chains(seqs, B, seed=0):
    toks, off = _csr(seqs)
    bo, h = oracle.block_hash(toks, off, B, seed)
    return bo, h, [list(map(int, h[bo[i]:bo[i + 1]])) for i in range(len(seqs))]


# ---------------------------------------------------------------- P0: hash vectors
def _gold():
    out = []
    for line in open(GOLD):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        lhs, rhs = line.split("->")
        out.append((lhs.split(), [int(x, 16) for x in rhs.split()]))
    return out


def _tokens_of(spec):
    name, arg = spec.split("=")[1].split("(")
    arg = arg.rstrip(")")
    if name == "range":
        a, b = arg.split(",")
        return list(range(int(a), int(b)))
    if name == "zeros":
        return [0] * int(arg)
    if name == "minus_ones":
        return [-1] * int(arg)
    raise ValueError(spec)


def test_golden_hash_vectors():
    seen = set()
    for lhs, vals in _gold():
        kind = lhs[0]
        seen.add(kind)
        if kind == "splitmix64_stream":
            s = 0
            for v in vals:
                s = (s + 0x9E3779B97F4A7C15) & bf.MASK
                assert oracle.mix64(s) == v
                assert bf.mix64(s) == v
        elif kind == "mix64":
            assert oracle.mix64(int(lhs[1])) == vals[0]
        elif kind == "multipliers":
            for j, v in enumerate(vals):
                assert oracle.position_multiplier(j) == v
        elif kind == "multiplier_sum":
            n = int(lhs[1])
            assert sum(oracle.position_multiplier(j) for j in range(n)) & bf.MASK == vals[0]
        elif kind == "chain":
            seed = int(lhs[1].split("=")[1], 16)
            toks = _tokens_of(lhs[2])
            t = np.asarray(toks, dtype=np.int32)
            bo, h = oracle.block_hash(t, np.asarray([0, len(toks)], dtype=np.int64), 16, seed)
            assert [int(x) for x in h] == vals
            assert int(bo[1]) == len(vals) == len(toks) // 16
            assert bf.chain(toks, 16, seed) == vals
    assert seen == {"splitmix64_stream", "mix64", "multipliers", "multiplier_sum", "chain"}


def test_hash_structure():
    """Chaining: equal prefixes <=> equal leading hashes; a change in block i
    changes k_i and everything after; position matters inside a block; trailing partial
    block ignored; EMPTY never produced."""
    rng = np.random.default_rng(7)
    a = rng.integers(0, 50, size=100).astype(np.int32)
    b = a.copy()
    b[37] += 1  # block 2 differs
    _, _, ch = _chains([a, b, a[:64], a[:70]], 16)
    assert ch[0][:2] == ch[1][:2] and all(x != y for x, y in zip(ch[0][2:], ch[1][2:]))
    assert ch[2] == ch[0][:4] and ch[3] == ch[0][:4]
    c = a.copy()
    c[[0, 1]] = c[[1, 0]]
    if a[0] != a[1]:
        assert _chains([c], 16)[2][0][0] != ch[0][0]
    assert all(k != bf.EMPTY for x in ch for k in x)
    # different seed, different chain
    assert _chains([a], 16, seed=5)[2][0][0] != ch[0][0]


# ---------------------------------------------------------------- P1: brute force on tiny inputs
def _tiny(rng, vocab, n, maxlen):
    # a few stems so prefixes collide often
    stems = [rng.integers(0, vocab, size=rng.integers(0, maxlen)).tolist() for _ in range(4)]
    seqs = []
    for _ in range(n):
        st = stems[rng.integers(0, 4)]
        cut = rng.integers(0, len(st) + 1)
        tail = rng.integers(0, vocab, size=rng.integers(0, 12)).tolist()
        s = (st[:cut] + tail)[:maxlen]
        seqs.append(s)
    return seqs


@pytest.mark.parametrize("seed", range(8))
@pytest.mark.parametrize("B", [2, 4, 16])
def test_bruteforce_tiny(seed, B):
    rng = np.random.default_rng([seed, B])
    vocab = int(rng.integers(2, 5))
    reqs = _tiny(rng, vocab, int(rng.integers(1, 48)), 80)
    cached = _tiny(rng, vocab, int(rng.integers(0, 10)), 80)
    toks, off = _csr(reqs)
    bo, h, ch = _chains(reqs, B)
    # block hash against the big-int restatement
    for r, s in enumerate(reqs):
        assert ch[r] == bf.chain(s, B, 0)
    # radix hit = max LCP over cached sequences
    radix, accepted = W.build_radix(_pieces(cached) if cached else None, B, 0)
    hr = oracle.lpm_radix(toks, off, _orc_radix(radix))
    assert hr.tolist() == [bf.hit_radix(s, cached) for s in reqs]
    # hash hit against a python set; table built from the cached chains
    ckeys = [k for s in cached for k in bf.chain(s, B, 0)]
    S = 64
    while S < 2 * max(len(set(ckeys)), 1):
        S *= 2
    t = W.build_table(np.asarray(ckeys, dtype=np.uint64), S)
    assert sorted(int(x) for x in t if x != W.EMPTY) == sorted(set(ckeys))
    hh = oracle.lpm_hash(h, bo, t, B)
    assert hh.tolist() == [bf.hit_hash(c, set(ckeys), B) for c in ch]
    # mirror identity P5 (table == full blocks of the radix cache's sequences)
    assert hh.tolist() == [B * (x // B) for x in hr.tolist()]
    # pending tree
    tr = oracle.pending_tree(h, bo)
    o, L, gid, gsz, cd, cs, ng = bf.pending_tree(ch)
    assert tr.order.tolist() == o and tr.lcp.tolist() == L
    assert tr.group_id.tolist() == gid and tr.group_size.tolist() == gsz and tr.n_groups == ng
    assert tr.cluster_depth.tolist() == cd and tr.cluster_size.tolist() == cs
    # cluster ids: equal id <=> same (depth, shared prefix) for non-singletons
    for a in range(len(reqs)):
        for b in range(len(reqs)):
            same = cd[a] == cd[b] and cd[a] > 0 and ch[a][:cd[a]] == ch[b][:cd[b]]
            if cd[a] > 0 and cd[b] > 0:
                assert (tr.cluster_id[a] == tr.cluster_id[b]) == same
    assert len(set(tr.cluster_id[[r for r in range(len(reqs)) if cd[r] == 0]].tolist())) == cd.count(0)
    assert tr.has_sharing == (max(gsz) >= 2)
    # demand by nested loops
    dm = oracle.demand(h, bo, t)
    assert dm.tolist() == bf.demand(ch, [int(x) for x in t])
    # cLPM order with duplicate arrivals to exercise the index tie-break
    arr = rng.integers(0, 5, size=len(reqs)).astype(np.int32)
    co = oracle.clpm_order(hr, tr.cluster_size, arr)
    assert co.tolist() == bf.clpm_order(hr.tolist(), cs, arr.tolist())
    co2 = oracle.clpm_order(hh, tr.cluster_size, None)
    assert co2.tolist() == bf.clpm_order(hh.tolist(), cs, None)


# ---------------------------------------------------------------- P2: the paper's worked example
def test_paper_worked_example():
    """8 cold requests A1,B1,C1,A2,B2,C2,A3,B3; cluster sizes 3/3/2; all h=0."""
    rng = np.random.default_rng(1)
    pre = {t: rng.integers(0, 1000, size=2048).tolist() for t in "ABC"}
    names = ["A1", "B1", "C1", "A2", "B2", "C2", "A3", "B3"]
    reqs = [pre[n[0]] + rng.integers(0, 1000, size=40).tolist() for n in names]
    toks, off = _csr(reqs)
    bo, h = oracle.block_hash(toks, off)
    tr = oracle.pending_tree(h, bo)
    assert tr.n_groups == 3
    assert tr.cluster_size.tolist() == [3, 3, 2, 3, 3, 2, 3, 3]
    assert tr.cluster_depth.tolist() == [128] * 8           # 2048 tokens = 128 blocks
    assert tr.has_sharing
    radix, _ = W.build_radix(None, 16, 0)                    # cold cache
    hr = oracle.lpm_radix(toks, off, _orc_radix(radix))
    assert hr.tolist() == [0] * 8
    co = oracle.clpm_order(hr, tr.cluster_size, np.arange(8, dtype=np.int32))
    # 3-part key: ties on h, size 3 before 2, then arrival (hand-derived)
    assert [names[i] for i in co] == ["A1", "B1", "A2", "B2", "A3", "B3", "C1", "C2"]


# ---------------------------------------------------------------- P3: Figure 6(a)
def test_figure_6a():
    """5 requests under a shared system prefix, {A x3, B x2}; cache holds sys
    and sys+A; 'PEEK: 2 queries' = 2 non-singleton clusters below the system node."""
    rng = np.random.default_rng(2)
    sys_ = rng.integers(0, 1000, size=64).tolist()
    A = rng.integers(0, 1000, size=48).tolist()
    Bp = rng.integers(0, 1000, size=48).tolist()
    reqs = [sys_ + A + rng.integers(0, 1000, size=20).tolist() for _ in range(3)]
    reqs += [sys_ + Bp + rng.integers(0, 1000, size=20).tolist() for _ in range(2)]
    toks, off = _csr(reqs)
    radix, _ = W.build_radix(_pieces([sys_, sys_ + A]), 16, 0)
    hr = oracle.lpm_radix(toks, off, _orc_radix(radix))
    assert hr.tolist()[:3] == [112] * 3
    assert all(64 <= x < 64 + 16 for x in hr.tolist()[3:])   # sys matched, B prefix not cached
    bo, h = oracle.block_hash(toks, off)
    tr = oracle.pending_tree(h, bo)
    assert tr.n_groups == 1 and tr.group_size.tolist() == [5] * 5
    assert sorted(tr.cluster_size.tolist()) == [2, 2, 3, 3, 3]
    assert len(set(tr.cluster_id.tolist())) == 2
    assert tr.cluster_depth.tolist() == [7] * 5              # (64+48)/16 blocks


# ---------------------------------------------------------------- P4/P5/P6: configs, invariants
@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5])
@pytest.mark.parametrize("seed", [42, 142])
def test_config_invariants(cfg, seed):
    wl = W.make(cfg, seed=seed, small=True)
    B = wl.block_size
    toks, off = wl.queue.materialize_np()
    lens = np.diff(off)
    N = wl.N
    ci = W.build_cache(wl, lambda a, b: oracle.block_hash(a, b, B, 0))
    bo, h = oracle.block_hash(toks, off, B, 0)
    nb = np.diff(bo)
    assert np.array_equal(nb, lens // B)
    hh = oracle.lpm_hash(h, bo, ci.t_keys, B)
    assert (hh % B == 0).all() and (hh <= B * nb).all() and (hh >= 0).all()
    tr = oracle.pending_tree(h, bo)
    assert sorted(tr.order.tolist()) == list(range(N))
    assert tr.lcp[0] == 0
    pair_min = np.minimum(nb[tr.order[1:]], nb[tr.order[:-1]])
    assert (tr.lcp[1:] <= pair_min).all()
    # group sizes over distinct groups sum to N (north_star "cluster sizes summing to N", R-S11)
    gs = {}
    for r in range(N):
        gs[int(tr.group_id[r])] = int(tr.group_size[r])
    assert sum(gs.values()) == N and len(gs) == tr.n_groups
    assert ((tr.cluster_size >= 2) == (tr.cluster_depth >= 1)).all()
    nz = tr.cluster_depth >= 1
    assert (tr.cluster_size[nz] <= tr.group_size[nz]).all()
    dm = oracle.demand(h, bo, ci.t_keys)
    assert dm.sum() <= bo[-1] and dm.max(initial=0) <= N
    assert (dm[ci.t_keys == W.EMPTY] == 0).all()
    if wl.has_radix:
        hr = oracle.lpm_radix(toks, off, _orc_radix(ci.radix))
        assert (hr >= 0).all() and (hr <= lens).all()
        # P5 mirror identity
        assert np.array_equal(hh, B * (hr // B))
        # siblings agree up to their LCP: sorted-adjacent pairs and a random sample
        rng = np.random.default_rng(seed)
        pairs = [(int(tr.order[j - 1]), int(tr.order[j])) for j in range(1, N)]
        pairs += [tuple(map(int, rng.integers(0, N, size=2))) for _ in range(2000)]
        for a, b in pairs:
            sa, sb = toks[off[a]:off[a + 1]], toks[off[b]:off[b + 1]]
            m = min(len(sa), len(sb))
            neq = np.nonzero(sa[:m] != sb[:m])[0]
            l = int(neq[0]) if neq.size else m
            assert min(hr[a], l) == min(hr[b], l)
        hit = hr
    else:
        hit = hh
    co = oracle.clpm_order(hit, tr.cluster_size, wl.arrival)
    assert sorted(co.tolist()) == list(range(N))
    keys = [(-int(hit[r]), -int(tr.cluster_size[r]), int(wl.arrival[r]), int(r)) for r in co]
    assert keys == sorted(keys)
    # the cache holds exactly X distinct full blocks (radix configs) at load 0.5
    if wl.has_radix:
        assert ci.radix.blocks == wl.cache_blocks and ci.n_keys == wl.cache_blocks


def test_config1_planted_structure():
    """P6: members of a cached cluster hit exactly the 512-token prefix; recovered group
    sizes equal the planted Zipf sizes [102,48,31,22,17,14,12,10]."""
    wl = W.make(1, seed=42)
    toks, off = wl.queue.materialize_np()
    ci = W.build_cache(wl, lambda a, b: oracle.block_hash(a, b))
    bo, h = oracle.block_hash(toks, off)
    hr = oracle.lpm_radix(toks, off, _orc_radix(ci.radix))
    hh = oracle.lpm_hash(h, bo, ci.t_keys)
    cl = wl.planted["cluster_of"]
    cached = np.isin(cl, wl.planted["cached_clusters"])
    assert (hr[cached] == 512).all() and (hh[cached] == 512).all()
    assert (hh[~cached] == 0).all() and (hr[~cached] < 16).all()
    tr = oracle.pending_tree(h, bo)
    sizes = sorted({int(g): int(s) for g, s in zip(tr.group_id, tr.group_size)}.values(), reverse=True)
    assert sizes == [102, 48, 31, 22, 17, 14, 12, 10]
    assert sizes == sorted(wl.planted["cluster_sizes"].tolist(), reverse=True)
    assert (tr.cluster_size == tr.group_size).all() and (tr.cluster_depth == 32).all()
    # planted clusters recovered exactly
    for g in set(tr.group_id.tolist()):
        assert len(set(cl[tr.group_id == g].tolist())) == 1
    # demand: each cached prefix block is wanted by every member of its cluster
    dm = oracle.demand(h, bo, ci.t_keys)
    want = sorted(int(wl.planted["cluster_sizes"][c]) for c in wl.planted["cached_clusters"] for _ in range(32))
    assert sorted(dm[dm > 0].tolist()) == want


def test_root_block_demand_is_N():
    """north_star invariant / R-S19: block 0 shared by every request and cached => demand N."""
    wl = W.make(3, seed=42, small=True)
    toks, off = wl.queue.materialize_np()
    ci = W.build_cache(wl, lambda a, b: oracle.block_hash(a, b))
    bo, h = oracle.block_hash(toks, off)
    dm = oracle.demand(h, bo, ci.t_keys)
    k0 = h[bo[0]]
    assert (h[bo[:-1]] == k0).all()
    slot = int(np.nonzero(ci.t_keys == k0)[0][0])
    assert dm[slot] == wl.N


# ---------------------------------------------------------------- P7: special cases
def test_special_cases():
    rng = np.random.default_rng(3)
    B = 16
    reqs = [rng.integers(0, 9, size=n).tolist() for n in (0, 5, 15, 16, 17, 40, 100)]
    toks, off = _csr(reqs)
    bo, h = oracle.block_hash(toks, off)
    assert np.diff(bo).tolist() == [0, 0, 0, 1, 1, 2, 6]
    # empty cache
    radix, _ = W.build_radix(None, B, 0)
    assert radix.V == 1 and radix.E == 0
    assert oracle.lpm_radix(toks, off, _orc_radix(radix)).tolist() == [0] * 7
    t = np.full(8, W.EMPTY, dtype=np.uint64)
    assert oracle.lpm_hash(h, bo, t).tolist() == [0] * 7
    assert oracle.demand(h, bo, t).tolist() == [0] * 8
    # cache = the requests themselves
    radix, _ = W.build_radix(_pieces(reqs), B, 0)
    assert oracle.lpm_radix(toks, off, _orc_radix(radix)).tolist() == [len(s) for s in reqs]
    t = W.build_table(h, 64)
    assert oracle.lpm_hash(h, bo, t).tolist() == [B * (len(s) // B) for s in reqs]
    # nb = 0 requests: own groups, sort first by index
    tr = oracle.pending_tree(h, bo)
    assert tr.order.tolist()[:3] == [0, 1, 2] and tr.lcp.tolist()[:4] == [0, 0, 0, 0]
    assert tr.cluster_size.tolist()[:3] == [1, 1, 1]
    # all identical
    same = [reqs[6]] * 5
    toks, off = _csr(same)
    bo, h = oracle.block_hash(toks, off)
    tr = oracle.pending_tree(h, bo)
    assert tr.order.tolist() == [0, 1, 2, 3, 4] and tr.lcp.tolist() == [0, 6, 6, 6, 6]
    assert tr.n_groups == 1 and tr.cluster_size.tolist() == [5] * 5 and tr.cluster_depth.tolist() == [6] * 5
    # N = 1
    toks, off = _csr([reqs[5]])
    bo, h = oracle.block_hash(toks, off)
    tr = oracle.pending_tree(h, bo)
    assert tr.order.tolist() == [0] and tr.cluster_size.tolist() == [1] and not tr.has_sharing
    # strict prefix sorts first and clusters at its own depth (R8)
    long_ = rng.integers(0, 9, size=64).tolist()
    toks, off = _csr([long_, long_[:32]])
    bo, h = oracle.block_hash(toks, off)
    tr = oracle.pending_tree(h, bo)
    assert tr.order.tolist() == [1, 0] and tr.lcp.tolist() == [0, 2]
    assert tr.cluster_depth.tolist() == [2, 2] and tr.cluster_size.tolist() == [2, 2]
    # first-miss semantics in hash mode (R12): a later present block does not count
    toks, off = _csr([long_])
    bo, h = oracle.block_hash(toks, off)
    t = W.build_table(h[[0, 2, 3]], 16)
    assert oracle.lpm_hash(h, bo, t).tolist() == [16]


# ---------------------------------------------------------------- P8: textbook reductions
def test_single_sequence_cache_is_plain_lcp():
    rng = np.random.default_rng(4)
    s = rng.integers(0, 3, size=300)
    reqs = []
    for _ in range(40):
        r = s[:rng.integers(0, 301)].copy()
        if r.size and rng.random() < 0.7:
            r[rng.integers(0, r.size)] = 7
        reqs.append(np.concatenate([r, rng.integers(0, 3, size=rng.integers(0, 9))]).tolist())
    toks, off = _csr(reqs)
    radix, _ = W.build_radix(_pieces([s.tolist()]), 16, 0)
    hr = oracle.lpm_radix(toks, off, _orc_radix(radix))
    for r, q in enumerate(reqs):
        m = min(len(q), 300)
        neq = np.nonzero(np.asarray(q[:m]) != s[:m])[0]
        assert hr[r] == (int(neq[0]) if neq.size else m)


def test_cluster_size_is_nearest_smaller_value_interval():
    """(order, lcp) is an (SA, LCP) pair: cluster interval = maximal run around j whose
    internal lcps are >= cd, found here with a monotone stack instead of outward scans."""
    wl = W.make(5, seed=142, small=True)
    toks, off = wl.queue.materialize_np()
    bo, h = oracle.block_hash(toks, off)
    tr = oracle.pending_tree(h, bo)
    N = wl.N
    L = tr.lcp.tolist() + [0]
    # for each position: left boundary a(v) / right boundary b(v) for threshold v via stacks
    for j in range(0, N, 7):
        cd = max(L[j], L[j + 1])
        r = int(tr.order[j])
        if cd == 0:
            assert tr.cluster_size[r] == 1
            continue
        a = j
        while L[a] >= cd:
            a -= 1
        b = j
        while L[b + 1] >= cd:
            b += 1
        assert tr.cluster_size[r] == b - a + 1 and tr.cluster_depth[r] == cd
        assert int(tr.cluster_id[r]) == (a << 32) | cd


def test_radix_builder_valid():
    """The engine stand-in produces a well-formed flattened radix cache."""
    wl = W.make(2, seed=42, small=True)
    radix, acc = W.build_radix(wl.cache_candidates, 16, wl.cache_blocks)
    V = radix.V
    assert radix.n_tok_len[0] == 0 and radix.n_child_off[0] == 0 and radix.n_child_off[V] == radix.E
    for v in range(V):
        ft = radix.e_first_tok[radix.n_child_off[v]:radix.n_child_off[v + 1]]
        assert (np.diff(ft) > 0).all()
        for e in range(radix.n_child_off[v], radix.n_child_off[v + 1]):
            u = radix.e_child[e]
            assert u > v and radix.c_tokens[radix.n_tok_off[u]] == radix.e_first_tok[e]
    assert sorted(radix.e_child.tolist()) == list(range(1, V))
    toks, off = acc.materialize_np()
    hr = oracle.lpm_radix(toks, off, _orc_radix(radix))
    assert np.array_equal(hr, np.diff(off))
