"""Pins of the NEXT-1 oracle functions (ancestor score, Eq. 2 eviction score,
sections, the full Eq. 1 key) against definitions written at TOKEN level in pure Python -
tuples of tokens, no hashes - plus closed forms and the paper's worked example."""
import numpy as np
import pytest

import oracle
from harness import workloads as W

B = 16


def _csr(seqs):
    off = np.zeros(len(seqs) + 1, dtype=np.int64)
    for i, s in enumerate(seqs):
        off[i + 1] = off[i] + len(s)
    toks = np.zeros(max(int(off[-1]), 1), dtype=np.int32)
    for i, s in enumerate(seqs):
        toks[off[i]:off[i + 1]] = s
    return toks[:int(off[-1])], off


def _hashes(seqs):
    toks, off = _csr(seqs)
    return oracle.block_hash(toks, off, B, 0)


def _path_count(seqs, prefix):
    """pending_count of the trie node spelled by `prefix` (a whole number of blocks): the pending
    requests passing through or ending at it."""
    n = len(prefix)
    return sum(1 for s in seqs if len(s) >= n and tuple(s[:n]) == prefix)


def bf_score(seqs):
    """PAPER.md:102 score(r) = sum over r's path of pending_count(v) * |edge(v)|, one B-token edge
    per block."""
    out = []
    for s in seqs:
        nb = len(s) // B
        out.append(sum(_path_count(seqs, tuple(s[:B * (i + 1)])) * B for i in range(nb)))
    return out


def bf_evict(seqs, prefix):
    """Eq. 2 for the cached block spelled by `prefix`: max over its ancestors (itself included) of
    pending_count * depth in tokens; 0 when no pending request passes through the block."""
    if _path_count(seqs, prefix) == 0:
        return 0
    return max(_path_count(seqs, prefix[:B * (j + 1)]) * B * (j + 1) for j in range(len(prefix) // B))


def bf_sections(seqs, hit, tau, arrival):
    """Alg. 2 lines 3-13 as printed: arrival order, a `seen` set of the first
    theta = 32 tokens - here the first two full blocks (one if there is only one; a request with no
    full block is never seen: DESIGN.md R22)."""
    order = sorted(range(len(seqs)), key=lambda r: (arrival[r], r))
    seen = set()
    sec = [None] * len(seqs)
    for r in order:
        if hit[r] > tau:
            sec[r] = 0
            continue
        nb = len(seqs[r]) // B
        if nb == 0:
            sec[r] = 1
            continue
        p = tuple(seqs[r][:B * min(nb, 2)])
        if p in seen:
            sec[r] = 2
        else:
            sec[r] = 1
            seen.add(p)
    return sec


def _tiny(rng, n, vocab=3):
    stems = [rng.integers(0, vocab, size=int(rng.integers(0, 120))).tolist() for _ in range(5)]
    seqs = []
    for _ in range(n):
        st = stems[int(rng.integers(0, 5))]
        cut = int(rng.integers(0, len(st) + 1))
        seqs.append(st[:cut] + rng.integers(0, vocab, size=int(rng.integers(0, 40))).tolist())
    seqs += [list(seqs[0]), list(seqs[1][: len(seqs[1]) // 2]), [], [1] * 5, [1] * 16, [1] * 16, [1] * 17]
    return seqs


@pytest.mark.parametrize("seed", range(6))
def test_bruteforce_next_rows(seed):
    rng = np.random.default_rng(100 + seed)
    seqs = _tiny(rng, 60)
    N = len(seqs)
    bo, h = _hashes(seqs)
    # O6 score
    assert oracle.score(h, bo, B).tolist() == bf_score(seqs)
    # O7 evict score: a table over the blocks of some cached sequences (half of them pending)
    cached = [seqs[i] for i in range(0, N, 3)] + [rng.integers(0, 3, size=64).tolist() for _ in range(5)]
    cbo, ch = _hashes(cached)
    keys = np.unique(ch)
    t_keys = W.build_table(keys, 1 << 11)
    prefix_of = {}
    for ci, s in enumerate(cached):
        for i in range(len(s) // B):
            prefix_of[int(ch[cbo[ci] + i])] = tuple(s[:B * (i + 1)])
    ev = oracle.evict_score(h, bo, t_keys, B)
    for p in range(t_keys.shape[0]):
        k = int(t_keys[p])
        want = 0 if k == 0xFFFFFFFFFFFFFFFF else bf_evict(seqs, prefix_of[k])
        assert int(ev[p]) == want, (p, want)
    # every pending cached block scores at least its own pending_count * depth (the j = i term)
    dem = oracle.demand(h, bo, t_keys)
    assert np.all((ev > 0) == (dem > 0))
    # O8 sections, with hits from an arbitrary (random) hit vector and two thresholds
    hit = rng.integers(0, 40, size=N).astype(np.int32)
    arrival = rng.permutation(N).astype(np.int32)
    arrival[::7] = arrival[0]  # duplicate arrivals: the request index decides
    for tau in (0, 20):
        assert oracle.sections(h, bo, hit, tau, arrival).tolist() == bf_sections(seqs, hit, tau, arrival)
    assert oracle.sections(h, bo, hit, 0, None).tolist() == bf_sections(seqs, hit, 0, list(range(N)))
    # O9 full key
    sec = oracle.sections(h, bo, hit, 0, arrival)
    sc = oracle.score(h, bo, B)
    cs = oracle.pending_tree(h, bo).cluster_size
    want = sorted(range(N), key=lambda r: (int(sec[r]), -int(hit[r]), -int(sc[r]), -int(cs[r]), int(arrival[r]), r))
    assert oracle.clpm_order_full(sec, hit, sc, cs, arrival).tolist() == want


def test_closed_forms():
    """N identical requests of nb blocks: every node on the path has pending_count N, so
    score = B * N * nb and a cached block at depth i scores N * B * (i + 1); a cold queue of
    identical prompts has one pioneer (the earliest arrival) and N - 1 siblings."""
    N, nb = 37, 9
    base = np.arange(B * nb).tolist()
    seqs = [list(base) for _ in range(N)]
    bo, h = _hashes(seqs)
    assert oracle.score(h, bo, B).tolist() == [B * N * nb] * N
    t_keys = W.build_table(np.unique(h), 64)
    ev = oracle.evict_score(h, bo, t_keys, B)
    chain = [int(x) for x in h[:nb]]
    for i, k in enumerate(chain):
        p = int(np.nonzero(t_keys == np.uint64(k))[0][0])
        assert int(ev[p]) == N * B * (i + 1)
    arrival = np.arange(N, dtype=np.int32)[::-1].copy()  # the LAST request arrived first
    sec = oracle.sections(h, bo, np.zeros(N, np.int32), 0, arrival)
    assert sec.tolist() == [2] * (N - 1) + [1]
    # a deep lightly shared prefix above a heavily shared one: the max in Eq. 2 picks the ancestor
    heavy = [np.arange(B).tolist() + [7] * B * 2 + [i] * B for i in range(10)]   # 10 share 3 blocks
    bo, h = _hashes(heavy)
    t_keys = W.build_table(np.unique(h), 64)
    ev = oracle.evict_score(h, bo, t_keys, B)
    leaf = int(h[bo[0] + 3])  # request 0's own 4th block: count 1 at depth 64 -> ancestor 10 * 48 wins
    assert int(ev[int(np.nonzero(t_keys == np.uint64(leaf))[0][0])]) == 10 * B * 3


def test_worked_example_sections_and_full_key():
    """PAPER.md:55 queue A1,B1,C1,A2,B2,C2,A3,B3, all cold: the first request of each tenant is the
    pioneer, the others are siblings, and Eq. 1 admits every pioneer before any
    sibling; inside a section ties on h fall to the score (tenants of three before the tenant of
    two), then arrival."""
    rng = np.random.default_rng(1)
    pre = {t: rng.integers(0, 1000, size=2048).tolist() for t in "ABC"}
    names = ["A1", "B1", "C1", "A2", "B2", "C2", "A3", "B3"]
    reqs = [pre[n[0]] + rng.integers(0, 1000, size=32).tolist() for n in names]
    bo, h = _hashes(reqs)
    N = len(reqs)
    hit = np.zeros(N, np.int32)
    arrival = np.arange(N, dtype=np.int32)
    sec = oracle.sections(h, bo, hit, 0, arrival)
    assert sec.tolist() == [1, 1, 1, 2, 2, 2, 2, 2]
    sc = oracle.score(h, bo, B)
    # 128 shared blocks counted by the tenant's size, 2 own blocks counted once
    assert sc.tolist() == [B * (128 * n + 2) for n in (3, 3, 2, 3, 3, 2, 3, 3)]
    cs = oracle.pending_tree(h, bo).cluster_size
    order = oracle.clpm_order_full(sec, hit, sc, cs, arrival)
    assert [names[i] for i in order] == ["A1", "B1", "C1", "A2", "B2", "A3", "B3", "C2"]
    # a warm request (h > tau) goes first whatever its cluster
    hit[5] = 512
    sec = oracle.sections(h, bo, hit, 0, arrival)
    assert sec[5] == 0
    assert names[oracle.clpm_order_full(sec, hit, sc, cs, arrival)[0]] == "C2"


def test_group_major_reproduces_the_papers_printed_order():
    """"PEEK reorders the queue by cluster via the pending tree to
    A1, A2, A3, B1, B2, B3, C1, C2" - the one admission order the paper prints."""
    rng = np.random.default_rng(1)
    pre = {t: rng.integers(0, 1000, size=2048).tolist() for t in "ABC"}
    names = ["A1", "B1", "C1", "A2", "B2", "C2", "A3", "B3"]
    reqs = [pre[n[0]] + rng.integers(0, 1000, size=32).tolist() for n in names]
    bo, h = _hashes(reqs)
    N = len(reqs)
    hit = np.zeros(N, np.int32)
    arrival = np.arange(N, dtype=np.int32)
    tr = oracle.pending_tree(h, bo)
    sec = oracle.sections(h, bo, hit, 0, arrival)
    lane_a = oracle.clpm_order_full(sec, hit, oracle.score(h, bo, B), tr.cluster_size, arrival)
    gm = oracle.group_major(lane_a, tr.cluster_id)
    assert [names[i] for i in gm] == ["A1", "A2", "A3", "B1", "B2", "B3", "C1", "C2"]


@pytest.mark.parametrize("seed", range(4))
def test_group_major_definition(seed):
    """Brute force of the reading: walk the lane; an unseen cluster emits all its members in lane
    order.  Clusters come out contiguous and the result is a permutation."""
    rng = np.random.default_rng(300 + seed)
    seqs = _tiny(rng, 50)
    N = len(seqs)
    bo, h = _hashes(seqs)
    tr = oracle.pending_tree(h, bo)
    lane = rng.permutation(N).astype(np.int32)
    want, done = [], set()
    for r in lane.tolist():
        c = int(tr.cluster_id[r])
        if c in done:
            continue
        done.add(c)
        want += [x for x in lane.tolist() if int(tr.cluster_id[x]) == c]
    got = oracle.group_major(lane, tr.cluster_id).tolist()
    assert got == want
    assert sorted(got) == list(range(N))


def bf_offline(seqs, depth_blocks=8):
    """PAPER.md:572 written with token tuples: trie over the first depth_blocks blocks, DFS with the
    children of a node in descending subtree count (ties: smallest request index below), the
    requests ending at a node first."""
    N = len(seqs)
    key = [tuple(s[:B * min(len(s) // B, depth_blocks)]) for s in seqs]   # truncated, whole blocks

    def below(prefix):
        return [r for r in range(N) if key[r][:len(prefix)] == prefix]

    out = []

    def visit(prefix):
        out.extend(r for r in range(N) if key[r] == prefix)
        kids = sorted({key[r][:len(prefix) + B] for r in below(prefix) if len(key[r]) > len(prefix)},
                      key=lambda c: (-len(below(c)), min(below(c))))
        for c in kids:
            visit(c)

    visit(())
    return out


@pytest.mark.parametrize("seed", range(4))
def test_offline_phase1_bruteforce(seed):
    rng = np.random.default_rng(500 + seed)
    seqs = _tiny(rng, 40)
    seqs += [list(rng.integers(0, 3, size=200)) for _ in range(6)]
    for d in (8, 2):
        bo, h = _hashes(seqs)
        order, guards = oracle.offline_phase1(h, bo, d)
        assert order.tolist() == bf_offline(seqs, d)
    # guards from the definitions
    N = len(seqs)
    bo, h = _hashes(seqs)
    order, guards = oracle.offline_phase1(h, bo, 8)
    blocks = [tuple(s[:B * (len(s) // B)]) for s in seqs]
    dup = sum(1 for r in range(N) if any(blocks[q] == blocks[r] for q in range(r)))
    cov = sum(1 for r in range(N) if len(blocks[r]) >= 2 * B and
              any(q != r and blocks[q][:2 * B] == blocks[r][:2 * B] for q in range(N)))
    depth = 0
    for r in range(N):
        d = 0
        while d < min(len(blocks[r]) // B, 8) and any(q != r and blocks[q][:B * (d + 1)] == blocks[r][:B * (d + 1)]
                                                     for q in range(N)):
            d += 1
        depth += B * d
    assert abs(guards[0] - dup / N) < 1e-12 and abs(guards[1] - cov / N) < 1e-12 and abs(guards[2] - depth / N) < 1e-9


def test_offline_phase1_worked_example_and_guards():
    """The tenants of PAPER.md:55 share their first 128 tokens, so phase 1 emits the tenants in
    descending size (ties by first request): the printed A1,A2,A3,B1,B2,B3,C1,C2.  A queue of
    unrelated prompts trips the coverage guard; a queue of exact duplicates the duplication guard."""
    rng = np.random.default_rng(1)
    pre = {t: rng.integers(0, 1000, size=2048).tolist() for t in "ABC"}
    names = ["A1", "B1", "C1", "A2", "B2", "C2", "A3", "B3"]
    reqs = [pre[n[0]] + rng.integers(0, 1000, size=32).tolist() for n in names]
    bo, h = _hashes(reqs)
    order, guards = oracle.offline_phase1(h, bo, 8)
    assert [names[i] for i in order] == ["A1", "A2", "A3", "B1", "B2", "B3", "C1", "C2"]
    assert guards.tolist() == [0.0, 1.0, 128.0, 0.0]
    lonely = [rng.integers(0, 1000, size=300).tolist() for _ in range(20)]
    bo, h = _hashes(lonely)
    order, guards = oracle.offline_phase1(h, bo, 8)
    assert order.tolist() == list(range(20)) and guards[1] == 0.0 and guards[3] == 1.0
    same = [list(lonely[0]) for _ in range(10)]
    bo, h = _hashes(same)
    order, guards = oracle.offline_phase1(h, bo, 8)
    assert guards[0] == 0.9 and guards[3] == 1.0


def _radix_of(seqs):
    toks, off = _csr(seqs)
    n = len(seqs)
    pcs = W.Pieces(np.ascontiguousarray(toks), off[:-1].copy(), np.diff(off), np.arange(n + 1, dtype=np.int64))
    radix, _ = W.build_radix(pcs, B, 0)
    return radix


@pytest.mark.parametrize("seed", range(4))
def test_radix_demand_bruteforce(seed):
    """node_demand[v] = requests whose LCP with the cached string spelled root -> v goes past the
    depth at which v starts (R26); the root counts every request."""
    rng = np.random.default_rng(700 + seed)
    cached = [s for s in _tiny(rng, 12) if len(s)]
    reqs = _tiny(rng, 50)
    radix = _radix_of(cached)
    orad = oracle.Radix(radix.c_tokens, radix.n_tok_off, radix.n_tok_len, radix.n_child_off,
                        radix.e_first_tok, radix.e_child)
    toks, off = _csr(reqs)
    got = oracle.radix_demand(toks, off, orad)
    V = radix.n_tok_len.shape[0]
    # path string and start depth of every node, by a walk over the flattened arrays
    path = {0: []}
    stack = [0]
    while stack:
        v = stack.pop()
        for e in range(int(radix.n_child_off[v]), int(radix.n_child_off[v + 1])):
            u = int(radix.e_child[e])
            lab = radix.c_tokens[int(radix.n_tok_off[u]): int(radix.n_tok_off[u]) + int(radix.n_tok_len[u])].tolist()
            path[u] = path[v] + lab
            stack.append(u)
    assert len(path) == V

    def lcp(a, b):
        n = 0
        for x, y in zip(a, b):
            if x != y:
                break
            n += 1
        return n

    for v in range(V):
        start = len(path[v]) - int(radix.n_tok_len[v])
        want = len(reqs) if v == 0 else sum(1 for r in reqs if lcp(r, path[v]) > start)
        assert int(got[v]) == want, v
    assert int(got[0]) == len(reqs)
    # consistency with the hit lengths: a request enters exactly the nodes above its hit depth
    hr = oracle.lpm_radix(toks, off, orad)
    assert int(got.sum()) - len(reqs) == sum(
        sum(1 for v in range(1, V) if lcp(r, path[v]) > len(path[v]) - int(radix.n_tok_len[v])) for r in reqs)
    assert all(int(h) <= len(r) for h, r in zip(hr, reqs))


def test_lane_b_and_dynamic_lane():
    rng = np.random.default_rng(9)
    N = 200
    sec = rng.integers(0, 3, size=N).astype(np.int32)
    hit = rng.integers(0, 5, size=N).astype(np.int32)
    arr = rng.integers(0, 40, size=N).astype(np.int32)   # many duplicate arrivals
    want = sorted(range(N), key=lambda r: (int(sec[r]), int(arr[r]), -int(hit[r]), r))
    assert oracle.lane_b(sec, hit, arr).tolist() == want
    assert oracle.lane_b(sec, hit, None).tolist() == sorted(range(N), key=lambda r: (int(sec[r]), r))
    # the fairness share ramps from 0.15 (cluster dominated) toward 0.60
    cs = np.full(100, 7, np.int32)
    new, sf = oracle.dynamic_lane(cs, 0.0, 0.15)
    assert sf == 0.0 and abs(new - 0.15) < 1e-15            # fixed point of the EMA at the floor
    cs[:] = 1
    new, sf = oracle.dynamic_lane(cs, 1.0, 0.60)
    assert sf == 1.0 and abs(new - 0.60) < 1e-15            # clamp(0.95) = 0.60
    cs[:50] = 3
    new, sf = oracle.dynamic_lane(cs, 0.5, 0.3)
    x = min(max(0.15 + 0.5 * 0.5 + 0.3 * 0.5, 0.10), 0.60)
    assert sf == 0.5 and abs(new - (0.3 * x + 0.7 * 0.3)) < 1e-15


def test_stride_interleave_properties_and_closed_forms():
    """a fraction alpha of the admissions come from Lane A; the fairness lane (whose
    head is the oldest request) advances at least every ceil(1 / (1 - alpha)) slots."""
    import math
    rng = np.random.default_rng(4)
    N = 500
    a = rng.permutation(N).astype(np.int32)
    b = rng.permutation(N).astype(np.int32)
    pos_a = np.argsort(a)
    pos_b = np.argsort(b)
    for alpha in (0.7, 0.4, 0.85, 0.9):
        out = oracle.stride_interleave(a, b, alpha)
        assert sorted(out.tolist()) == list(range(N))
        # replay: which lane admitted each slot is fixed by alpha alone
        from_a = [math.floor((k + 1) * alpha) > math.floor(k * alpha) for k in range(N)]
        for k in (10, 100, 499):
            assert sum(from_a[:k]) == math.floor(k * alpha)
        gaps = np.diff([k for k in range(N) if not from_a[k]])
        assert gaps.max() <= math.ceil(1 / (1 - alpha))
        # every slot admits, from its lane, a request all of whose lane predecessors are admitted
        seen = set()
        for k, r in enumerate(out.tolist()):
            lane_pos, lane = (pos_a, a) if from_a[k] else (pos_b, b)
            assert all(int(x) in seen for x in lane[: lane_pos[r]])
            seen.add(r)
    assert oracle.stride_interleave(a, b, 1.0).tolist() == a.tolist()
    assert oracle.stride_interleave(a, b, 0.0).tolist() == b.tolist()
    assert oracle.stride_interleave(a, a, 0.7).tolist() == a.tolist()
    # A ascending, B descending, alpha = 1/2: B, A, B, A ... from the two ends
    up = np.arange(10, dtype=np.int32)
    assert oracle.stride_interleave(up, up[::-1].copy(), 0.5).tolist() == [9, 0, 8, 1, 7, 2, 6, 3, 5, 4]
