"""Seeded synthetic workloads: the five configs of BASELINE.json.

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none
of the method's arithmetic: no hash function, no prefix walk, no probe, no sort of
chains.  It draws random numbers (numpy ``default_rng([seed, config])``; seeds 42,
142, 242 as in PAPER.md:362), lays requests out as CSR int32 token arrays, and asks
``harness/engine_sim.cpp`` (a stand-in for the engine's prefix cache) to
build the read-only cache inputs.  Chained hashes needed for the table keys are
produced by a ``hash_fn`` the caller passes in (the oracle's in oracle tests, the
CUDA call in GPU tests and bench.py).

The paper measures on LooGLE, RepoBench-Python, the Mooncake trace and LMSYS chat
(PAPER.md:349-353); none is available here and none of their items is reproduced.
These configs stand in for the *shapes* of W1, W2, W5, W4.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass, field
from typing import Callable, Optional

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_ESIM_SRC = os.path.join(_HERE, "engine_sim.cpp")
_ESIM_LIB = os.path.join(_HERE, "libpeek_engine_sim.so")
_esim = None

VOCAB = 128256
EMPTY = np.uint64(0xFFFFFFFFFFFFFFFF)


def build_engine_sim(force: bool = False) -> str:
    if (not force and os.path.exists(_ESIM_LIB)
            and os.path.getmtime(_ESIM_LIB) >= os.path.getmtime(_ESIM_SRC)):
        return _ESIM_LIB
    subprocess.run(["g++", "-O2", "-std=c++17", "-fPIC", "-shared", _ESIM_SRC, "-o", _ESIM_LIB],
                   check=True)
    return _ESIM_LIB


def _lib():
    global _esim
    if _esim is None:
        build_engine_sim()
        L = ctypes.CDLL(_ESIM_LIB)
        L.esim_radix_new.restype = ctypes.c_void_p
        L.esim_radix_new.argtypes = [ctypes.c_int32, ctypes.c_int64]
        L.esim_radix_free.argtypes = [ctypes.c_void_p]
        L.esim_radix_insert.restype = ctypes.c_int64
        L.esim_radix_insert.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p,
                                        ctypes.c_int64, ctypes.c_void_p]
        L.esim_radix_sizes.argtypes = [ctypes.c_void_p] + [ctypes.c_void_p] * 5
        L.esim_radix_export.argtypes = [ctypes.c_void_p] + [ctypes.c_void_p] * 6
        L.esim_table_insert.restype = ctypes.c_int64
        L.esim_table_insert.argtypes = [ctypes.c_void_p, ctypes.c_int64, ctypes.c_void_p,
                                        ctypes.c_int64, ctypes.c_int64, ctypes.c_int64]
        _esim = L
    return _esim


# ---------------------------------------------------------------------------
# Sequences as concatenations of slices of a token pool
# ---------------------------------------------------------------------------
@dataclass
class Pieces:
    """n sequences; sequence i = concat of pool[src[p] : src[p]+length[p]] for its pieces."""
    pool: np.ndarray      # int32[P]
    src: np.ndarray       # int64[n_pieces]
    length: np.ndarray    # int64[n_pieces]
    seq_off: np.ndarray   # int64[n+1] CSR over pieces
    _pool_dev: dict = field(default_factory=dict, repr=False)

    @property
    def n(self) -> int:
        return int(self.seq_off.shape[0] - 1)

    def seq_lens(self) -> np.ndarray:
        c = np.concatenate([[0], np.cumsum(self.length)])
        return (c[self.seq_off[1:]] - c[self.seq_off[:-1]]).astype(np.int64)

    def select(self, idx) -> "Pieces":
        idx = np.asarray(idx, dtype=np.int64)
        cnt = self.seq_off[idx + 1] - self.seq_off[idx]
        new_off = np.concatenate([[0], np.cumsum(cnt)]).astype(np.int64)
        total = int(new_off[-1])
        which = np.repeat(np.arange(idx.shape[0], dtype=np.int64), cnt)
        within = np.arange(total, dtype=np.int64) - new_off[which]
        p = self.seq_off[idx][which] + within
        out = Pieces(self.pool, self.src[p], self.length[p], new_off)
        out._pool_dev = self._pool_dev
        return out

    def truncated(self, new_lens) -> "Pieces":
        """Keep the first new_lens[i] tokens of sequence i (new_lens[i] <= len_i)."""
        new_lens = np.asarray(new_lens, dtype=np.int64)
        cum = np.concatenate([[0], np.cumsum(self.length)])
        which = np.repeat(np.arange(self.n, dtype=np.int64), np.diff(self.seq_off))
        start_in_seq = cum[:-1] - cum[self.seq_off[:-1]][which]
        keep = np.clip(new_lens[which] - start_in_seq, 0, self.length)
        out = Pieces(self.pool, self.src.copy(), keep.astype(np.int64), self.seq_off.copy())
        out._pool_dev = self._pool_dev
        return out

    def materialize(self, device="cpu", chunk_tokens: int = 1 << 26):
        """-> (tokens int32[T], tok_off int64[n+1]) torch tensors on `device`."""
        dev = torch.device(device)
        key = str(dev)
        if key not in self._pool_dev:
            self._pool_dev[key] = torch.from_numpy(self.pool).to(dev)
        pool = self._pool_dev[key]
        lens = self.seq_lens()
        tok_off = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
        T = int(tok_off[-1])
        out = torch.empty(max(T, 1), dtype=torch.int32, device=dev)
        pc_end = np.cumsum(self.length)
        n_p = self.length.shape[0]
        a = 0
        while a < n_p:
            base = int(pc_end[a - 1]) if a > 0 else 0
            b = int(np.searchsorted(pc_end, base + chunk_tokens, side="right"))
            b = max(b, a + 1)
            b = min(b, n_p)
            ln = torch.from_numpy(self.length[a:b]).to(dev)
            sr = torch.from_numpy(self.src[a:b]).to(dev)
            tot = int(pc_end[b - 1]) - base
            if tot > 0:
                starts = torch.cumsum(ln, 0) - ln
                pid = torch.repeat_interleave(torch.arange(b - a, device=dev), ln, output_size=tot)
                idx = torch.arange(tot, device=dev) - starts[pid] + sr[pid]
                out[base:base + tot] = pool[idx]
                del pid, idx
            a = b
        return out[:T] if T > 0 else out[:0], torch.from_numpy(tok_off).to(dev)

    def materialize_np(self):
        t, o = self.materialize("cpu")
        return t.numpy(), o.numpy()


def _pieces_from_lists(pool, per_seq):
    """per_seq: list of lists of (src, len)."""
    src, ln, off = [], [], [0]
    for ps in per_seq:
        for s, l in ps:
            src.append(s)
            ln.append(l)
        off.append(len(src))
    return Pieces(pool, np.asarray(src, dtype=np.int64), np.asarray(ln, dtype=np.int64),
                  np.asarray(off, dtype=np.int64))


# ---------------------------------------------------------------------------
# Engine-side cache construction (inputs, not method)
# ---------------------------------------------------------------------------
@dataclass
class RadixArrays:
    c_tokens: np.ndarray
    n_tok_off: np.ndarray
    n_tok_len: np.ndarray
    n_child_off: np.ndarray
    e_first_tok: np.ndarray
    e_child: np.ndarray
    blocks: int = 0

    @property
    def V(self) -> int:
        return int(self.n_tok_len.shape[0])

    @property
    def E(self) -> int:
        return int(self.e_child.shape[0])


def build_radix(cache: Optional[Pieces], block_size: int, max_blocks: int, batch: int = 4096):
    """Insert candidate sequences in order until `max_blocks` distinct full blocks
    are cached (last one truncated at a block boundary).  Returns (RadixArrays,
    accepted Pieces = exactly the token sequences the cache now holds)."""
    L = _lib()
    h = L.esim_radix_new(block_size, int(max_blocks))
    acc_idx, acc_len = [], []
    try:
        n = cache.n if cache is not None else 0
        a = 0
        while a < n:
            b = min(n, a + batch)
            sub = cache.select(np.arange(a, b))
            toks, off = sub.materialize_np()
            toks = np.ascontiguousarray(toks)
            off = np.ascontiguousarray(off)
            al = np.zeros(b - a, dtype=np.int64)
            L.esim_radix_insert(h, toks.ctypes.data, off.ctypes.data, b - a, al.ctypes.data)
            keep = np.nonzero(al > 0)[0]
            acc_idx.append(keep + a)
            acc_len.append(al[keep])
            V = ctypes.c_int64(); E = ctypes.c_int64(); CT = ctypes.c_int64()
            BL = ctypes.c_int64(); FU = ctypes.c_int32()
            L.esim_radix_sizes(h, ctypes.byref(V), ctypes.byref(E), ctypes.byref(CT),
                               ctypes.byref(BL), ctypes.byref(FU))
            if FU.value:
                break
            a = b
        V = ctypes.c_int64(); E = ctypes.c_int64(); CT = ctypes.c_int64()
        BL = ctypes.c_int64(); FU = ctypes.c_int32()
        L.esim_radix_sizes(h, ctypes.byref(V), ctypes.byref(E), ctypes.byref(CT),
                           ctypes.byref(BL), ctypes.byref(FU))
        r = RadixArrays(np.zeros(max(CT.value, 1), np.int32), np.zeros(V.value, np.int64),
                        np.zeros(V.value, np.int32), np.zeros(V.value + 1, np.int32),
                        np.zeros(max(E.value, 1), np.int32), np.zeros(max(E.value, 1), np.int32),
                        int(BL.value))
        L.esim_radix_export(h, r.c_tokens.ctypes.data, r.n_tok_off.ctypes.data,
                            r.n_tok_len.ctypes.data, r.n_child_off.ctypes.data,
                            r.e_first_tok.ctypes.data, r.e_child.ctypes.data)
        r.c_tokens = r.c_tokens[:CT.value]
        r.e_first_tok = r.e_first_tok[:E.value]
        r.e_child = r.e_child[:E.value]
    finally:
        L.esim_radix_free(h)
    if acc_idx:
        idx = np.concatenate(acc_idx)
        ln = np.concatenate(acc_len)
        accepted = cache.select(idx).truncated(ln)
    else:
        accepted = None
    return r, accepted


def build_table(keys: np.ndarray, slots: int, max_keys: int = 0) -> np.ndarray:
    """Open-addressed key table (linear probing, home = key & (S-1), EMPTY = ~0):
    insert `keys` in order, skipping duplicates, up to `max_keys`."""
    assert slots & (slots - 1) == 0
    t = np.full(slots, EMPTY, dtype=np.uint64)
    keys = np.ascontiguousarray(keys, dtype=np.uint64)
    _lib().esim_table_insert(t.ctypes.data, slots, keys.ctypes.data, keys.shape[0], 0, int(max_keys))
    return t


# ---------------------------------------------------------------------------
# The five configs
# ---------------------------------------------------------------------------
@dataclass
class Workload:
    config: int
    seed: int
    name: str
    block_size: int
    queue: Pieces                 # N pending requests (shuffled: index carries no cluster info)
    arrival: np.ndarray           # int32[N], an independent random permutation
    cache_candidates: Optional[Pieces]   # in insertion order
    cache_blocks: int             # X: distinct full blocks the cache holds
    table_slots: int              # S
    has_radix: bool
    planted: dict

    @property
    def N(self) -> int:
        return self.queue.n


def zipf_sizes(M: int, C: int, a: float) -> np.ndarray:
    """Sizes of C clusters summing to M, w_c ~ (c+1)^-a, each >= 2 (DESIGN.md recipe)."""
    w = (np.arange(C) + 1.0) ** (-a)
    q = M * w / w.sum()
    size = np.maximum(np.floor(q), 2).astype(np.int64)
    frac = q - np.floor(q)
    order = np.argsort(-frac, kind="stable")
    i = 0
    while size.sum() < M:
        size[order[i % C]] += 1
        i += 1
    while size.sum() > M:
        size[int(np.argmax(size))] -= 1
    return size


def _rand_tokens(rng, n):
    return rng.integers(0, VOCAB, size=int(n), dtype=np.int32)


def _finish(config, seed, name, rng, pool_parts, per_seq, cache_per_seq, cache_blocks,
            table_slots, has_radix, planted, cluster_of):
    pool = np.concatenate(pool_parts) if pool_parts else np.zeros(0, np.int32)
    queue = _pieces_from_lists(pool, per_seq)
    N = queue.n
    perm = rng.permutation(N)
    queue = queue.select(perm)
    planted = dict(planted)
    planted["cluster_of"] = np.asarray(cluster_of, dtype=np.int64)[perm]
    arrival = rng.permutation(N).astype(np.int32)
    cache = _pieces_from_lists(pool, cache_per_seq) if cache_per_seq is not None else None
    if cache is not None:
        cache._pool_dev = queue._pool_dev
    return Workload(config, seed, name, 16, queue, arrival, cache, int(cache_blocks),
                    int(table_slots), has_radix, planted)


class _Pool:
    def __init__(self):
        self.parts = []
        self.size = 0

    def add(self, arr) -> int:
        s = self.size
        self.parts.append(arr)
        self.size += int(arr.shape[0])
        return s


def config1(seed=42, N=256, n_clusters=8, prefix_len=512, cache_blocks=4096, n_cached=4,
            n_distractors=200):
    """Tiny shared-prompt chat (BASELINE.json configs[0]; shape of W1)."""
    rng = np.random.default_rng([seed, 1])
    P = _Pool()
    sizes = zipf_sizes(N, n_clusters, 1.1)
    pre = [P.add(_rand_tokens(rng, prefix_len)) for _ in range(n_clusters)]
    per_seq, cluster_of = [], []
    for c in range(n_clusters):
        for _ in range(int(sizes[c])):
            sl = int(rng.integers(64, 257))
            s = P.add(_rand_tokens(rng, sl))
            per_seq.append([(pre[c], prefix_len), (s, sl)])
            cluster_of.append(c)
    cached = rng.permutation(n_clusters)[:n_cached]
    cache = [[(pre[int(c)], prefix_len)] for c in cached]
    for _ in range(n_distractors):
        dl = int(rng.integers(128, 1025))
        cache.append([(P.add(_rand_tokens(rng, dl)), dl)])
    return _finish(1, seed, "tiny_shared_prompt_chat", rng, P.parts, per_seq, cache, cache_blocks,
                   2 * cache_blocks, True,
                   {"cluster_sizes": sizes, "cached_clusters": np.sort(cached), "prefix_len": prefix_len},
                   cluster_of)


def config2(seed=42, N=16384, n_clusters=64, singleton_frac=0.2, cache_blocks=262144,
            cached_frac=0.4, prefix_range=(1024, 2048), n_filler=9000):
    """Shared-prompt chat at scale (configs[1]; W1)."""
    rng = np.random.default_rng([seed, 2])
    P = _Pool()
    n_single = int(round(N * singleton_frac))
    sizes = zipf_sizes(N - n_single, n_clusters, 1.1)
    plen = rng.integers(prefix_range[0], prefix_range[1] + 1, size=n_clusters)
    pre = [P.add(_rand_tokens(rng, plen[c])) for c in range(n_clusters)]
    per_seq, cluster_of = [], []
    for c in range(n_clusters):
        sls = rng.integers(50, 501, size=int(sizes[c]))
        base = P.add(_rand_tokens(rng, sls.sum()))
        o = 0
        for sl in sls:
            per_seq.append([(pre[c], int(plen[c])), (base + o, int(sl))])
            cluster_of.append(c)
            o += int(sl)
    sls = rng.integers(200, 2001, size=n_single)
    base = P.add(_rand_tokens(rng, sls.sum()))
    o = 0
    for sl in sls:
        per_seq.append([(base + o, int(sl))])
        cluster_of.append(-1)
        o += int(sl)
    n_cached = int(round(n_clusters * cached_frac))
    cached = rng.permutation(n_clusters)[:n_cached]
    cache = [[(pre[int(c)], int(plen[int(c)]))] for c in cached]
    fls = rng.integers(128, 1025, size=n_filler)
    base = P.add(_rand_tokens(rng, fls.sum()))
    o = 0
    for fl in fls:
        cache.append([(base + o, int(fl))])
        o += int(fl)
    return _finish(2, seed, "shared_prompt_chat_at_scale", rng, P.parts, per_seq, cache,
                   cache_blocks, 2 * cache_blocks, True,
                   {"cluster_sizes": sizes, "cached_clusters": np.sort(cached), "prefix_len": plen},
                   cluster_of)


def config3(seed=42, N=8192, n_docs=256, doc_range=(4096, 16384), instr_len=256,
            cache_blocks=1048576):
    """Long-prefix RAG (configs[2]; W2)."""
    rng = np.random.default_rng([seed, 3])
    P = _Pool()
    instr = P.add(_rand_tokens(rng, instr_len))
    dlen = rng.integers(doc_range[0], doc_range[1] + 1, size=n_docs)
    docs = [P.add(_rand_tokens(rng, dlen[i])) for i in range(n_docs)]
    w = (np.arange(n_docs) + 1.0) ** (-1.2)
    w /= w.sum()
    nd = rng.integers(1, 4, size=N)
    qls = rng.integers(32, 129, size=N)
    qbase = P.add(_rand_tokens(rng, qls.sum()))
    per_seq, ctx, cluster_of = [], [], []
    o = 0
    for r in range(N):
        ds = rng.choice(n_docs, size=int(nd[r]), p=w)
        pcs = [(instr, instr_len)] + [(docs[int(d)], int(dlen[int(d)])) for d in ds]
        ctx.append(list(pcs))
        per_seq.append(pcs + [(qbase + o, int(qls[r]))])
        cluster_of.append(int(ds[0]))
        o += int(qls[r])
    cache = [ctx[int(r)] for r in rng.permutation(N)]
    return _finish(3, seed, "long_prefix_rag", rng, P.parts, per_seq, cache, cache_blocks,
                   2 * cache_blocks, True, {"instr_len": instr_len}, cluster_of)


def config4(seed=42, N=65536, shared_frac=0.05, n_prefixes=32, prefix_len=512,
            table_slots=1 << 22, n_filler=20000, filler_range=(128, 4096),
            single_range=(200, 4000)):
    """Singleton-dominated chat, block-hash-table mode only (configs[3]; W5)."""
    rng = np.random.default_rng([seed, 4])
    P = _Pool()
    n_shared = int(round(N * shared_frac))
    pre = [P.add(_rand_tokens(rng, prefix_len)) for _ in range(n_prefixes)]
    per_seq, cluster_of = [], []
    sls = rng.integers(single_range[0], single_range[1] + 1, size=N - n_shared)
    base = P.add(_rand_tokens(rng, sls.sum()))
    o = 0
    for sl in sls:
        per_seq.append([(base + o, int(sl))])
        cluster_of.append(-1)
        o += int(sl)
    which = rng.integers(0, n_prefixes, size=n_shared)
    sls = rng.integers(64, max(65, single_range[1] - prefix_len + 1), size=n_shared)
    base = P.add(_rand_tokens(rng, sls.sum()))
    o = 0
    for i in range(n_shared):
        per_seq.append([(pre[int(which[i])], prefix_len), (base + o, int(sls[i]))])
        cluster_of.append(int(which[i]))
        o += int(sls[i])
    cache = [[(pre[c], prefix_len)] for c in range(n_prefixes)]
    fls = rng.integers(filler_range[0], filler_range[1] + 1, size=n_filler)
    base = P.add(_rand_tokens(rng, fls.sum()))
    o = 0
    for fl in fls:
        cache.append([(base + o, int(fl))])
        o += int(fl)
    return _finish(4, seed, "singleton_chat_table_only", rng, P.parts, per_seq, cache,
                   table_slots // 2, table_slots, False,
                   {"prefix_len": prefix_len, "n_prefixes": n_prefixes, "n_shared": n_shared},
                   cluster_of)


def config5(seed=42, N=1048576, n_conv=65536, n_prompts=128, prompt_len=1024,
            turn_range=(4, 32), seg_range=(64, 512), cache_blocks=4194304,
            n_cache_candidates=60000):
    """Agentic multi-turn at scale (configs[4]; W4): the full pipeline."""
    rng = np.random.default_rng([seed, 5])
    P = _Pool()
    prompts = P.add(_rand_tokens(rng, n_prompts * prompt_len))
    turns = rng.integers(turn_range[0], turn_range[1] + 1, size=n_conv).astype(np.int64)
    # rebalance to sum exactly N: walk conversations cyclically
    diff = int(turns.sum() - N)
    c = 0
    guard = 0
    while diff != 0 and guard < 200 * n_conv:
        if diff > 0 and turns[c] > turn_range[0]:
            turns[c] -= 1
            diff -= 1
        elif diff < 0 and turns[c] < turn_range[1]:
            turns[c] += 1
            diff += 1
        c = (c + 1) % n_conv
        guard += 1
    assert diff == 0, "N not reachable with this turn range"
    which = rng.integers(0, n_prompts, size=n_conv)
    tot_turns = int(turns.sum())
    seg = rng.integers(seg_range[0], seg_range[1] + 1, size=tot_turns).astype(np.int64)
    base = P.add(_rand_tokens(rng, seg.sum()))
    conv_of = np.repeat(np.arange(n_conv, dtype=np.int64), turns)
    turn_off = np.concatenate([[0], np.cumsum(turns)])
    seg_cum = np.cumsum(seg)
    conv_base = np.concatenate([[0], seg_cum])[turn_off[:-1]]        # pool offset of conv's stream
    ctx_len = seg_cum - conv_base[conv_of]                            # tokens after the prompt
    n_req = tot_turns
    src = np.empty(2 * n_req, dtype=np.int64)
    ln = np.empty(2 * n_req, dtype=np.int64)
    src[0::2] = prompts + which[conv_of] * prompt_len
    ln[0::2] = prompt_len
    src[1::2] = base + conv_base[conv_of]
    ln[1::2] = ctx_len
    pool = np.concatenate(P.parts)
    queue = Pieces(pool, src, ln, np.arange(0, 2 * n_req + 1, 2, dtype=np.int64))
    perm = rng.permutation(n_req)
    cand = rng.permutation(n_req)[:min(n_cache_candidates, n_req)]
    cache = queue.select(cand)
    queue = queue.select(perm)
    cache._pool_dev = queue._pool_dev
    arrival = rng.permutation(n_req).astype(np.int32)
    planted = {"cluster_of": conv_of[perm], "prompt_of": which[conv_of][perm],
               "prompt_len": prompt_len, "turns": turns}
    return Workload(5, seed, "agentic_multi_turn_at_scale", 16, queue, arrival, cache,
                    int(cache_blocks), int(2 * cache_blocks), True, planted)


CONFIGS = {1: config1, 2: config2, 3: config3, 4: config4, 5: config5}

# Reduced sizes with the same structure, for CPU tests and the oracle-sized parity cases.
SMALL = {
    1: dict(),
    2: dict(N=1024, n_clusters=12, cache_blocks=8192, n_filler=400),
    3: dict(N=256, n_docs=12, doc_range=(300, 1200), instr_len=64, cache_blocks=4096),
    4: dict(N=2048, n_prefixes=6, prefix_len=128, table_slots=1 << 14, n_filler=300,
            filler_range=(64, 600), single_range=(40, 700)),
    5: dict(N=1024, n_conv=96, n_prompts=5, prompt_len=128, turn_range=(4, 18),
            seg_range=(20, 90), cache_blocks=2048, n_cache_candidates=300),
}


def make(config: int, seed: int = 42, small: bool = False, **over) -> Workload:
    kw = dict(SMALL[config]) if small else {}
    kw.update(over)
    return CONFIGS[config](seed=seed, **kw)


@dataclass
class CacheInputs:
    radix: Optional[RadixArrays]
    t_keys: np.ndarray
    cached: Pieces     # the token sequences the cache holds
    n_keys: int


def build_cache(wl: Workload, hash_fn: Callable) -> CacheInputs:
    """Radix arrays + mirrored table for a workload.  `hash_fn(tokens, tok_off) ->
    (blk_off, hashes)` (numpy in, numpy out) supplies the chained hashes of the
    cached sequences; the table gets every distinct one (S = 2X, load 0.5)."""
    if wl.has_radix:
        radix, cached = build_radix(wl.cache_candidates, wl.block_size, wl.cache_blocks)
        toks, off = cached.materialize_np()
        _, keys = hash_fn(toks, off)
        t = build_table(keys, wl.table_slots, 0)
    else:
        radix, cached = None, wl.cache_candidates
        toks, off = cached.materialize_np()
        _, keys = hash_fn(toks, off)
        t = build_table(keys, wl.table_slots, wl.cache_blocks)
    n_keys = int((t != EMPTY).sum())
    return CacheInputs(radix, t, cached, n_keys)
