// peek_lpm.cu — a5/a6 peek_lpm: per-request longest prefix match against the engine's cache.
//
// Radix mode (the result of Alg. 1; "a partial match terminates the branch",
// PAPER.md:291): one warp per request.  Child lookup: a coalesced ballot over the sorted edge
// slice (32-ary narrowing when a node has more than 32 children, e.g. the root).  Edge labels are
// compared 32 lanes x CMP_UNROLL tokens per step, both streams coalesced.
// Hash mode ("per-request find_longest_cache_hit"): one warp per request, 32
// consecutive blocks probed per step in the open-addressed table, first miss wins.
//
// Without a peek_tree_view every request walks on its own (k_lpm_radix / k_lpm_hash, one warp per
// request).  With it the call co-descends over the sorted order: k_lpm_dual<RADIX> below
// ("one cache walk per pending edge"), one persistent kernel per mode.  Queues of
// at most LPM_SMALL_MAX requests take one launch for both modes (k_lpm_small).  The speculative
// variant (k_lpm_*_spec + the resolve scan) is kept as an explicit strategy.
#include <stdlib.h>

#include "peek_common.cuh"

namespace peek {

static constexpr int LPM_THREADS = 256;
static constexpr int LPM_SMALL_MAX = 2048;  // queues up to this size: one launch, a warp per request, both modes
static constexpr int CMP_UNROLL = 8;

struct RadixDev {
    const i32* c_tokens;
    const i64* n_tok_off;
    const i32* n_tok_len;
    const i32* n_child_off;
    const i32* e_first_tok;
    const i32* e_child;
};

// edge index in [e0, e1) whose first token equals t, or -1 (edges sorted ascending, distinct)
__device__ __forceinline__ i32 find_child(const i32* __restrict__ e_first_tok, i32 e0, i32 e1, i32 t,
                                          int lane) {
    // 32-ary narrowing: lanes sample 32 pivots of the range, keep the sub-range that can hold t
    while (e1 - e0 > 32) {
        i32 n = e1 - e0;
        i32 step = (n + 31) >> 5;  // ceil(n / 32)
        i32 pos = e0 + lane * step;
        bool le = pos < e1 && __ldg(e_first_tok + pos) <= t;
        unsigned m = __ballot_sync(0xffffffffu, le);
        if (m == 0) return -1;                 // t below the smallest first token
        int k = 31 - __clz(m);                 // last pivot <= t
        e0 = e0 + k * step;
        e1 = min(e0 + step, e1);
    }
    i32 f = (e0 + lane < e1) ? __ldg(e_first_tok + e0 + lane) : 0;
    unsigned m = __ballot_sync(0xffffffffu, (e0 + lane < e1) && f == t);
    return m ? e0 + (__ffs(m) - 1) : -1;
}

// number of leading equal tokens of a[0..limit) and b[0..limit), warp-cooperative.  Most compares
// end at once (a random token differs) or run the whole edge: the first step looks at 64 tokens,
// later steps at 32 x CMP_UNROLL tokens per round trip.
template <int U>
__device__ __forceinline__ bool match_step(const i32* __restrict__ a, const i32* __restrict__ b, i64 base,
                                           i64 limit, int lane, i64* m) {
    i32 x[U], y[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
        const i64 i = base + u * 32 + lane;
        const bool in = i < limit;
        x[u] = in ? __ldg(a + i) : 0;
        y[u] = in ? __ldg(b + i) : 1;
    }
#pragma unroll
    for (int u = 0; u < U; ++u) {
        const unsigned neq = __ballot_sync(0xffffffffu, x[u] != y[u]);
        if (neq) {
            const i64 f = base + u * 32 + (__ffs(neq) - 1);
            *m = f < limit ? f : limit;
            return true;
        }
    }
    return false;
}
__device__ __forceinline__ i64 match_len(const i32* __restrict__ a, const i32* __restrict__ b, i64 limit,
                                         int lane) {
    i64 m = limit;
    if (limit <= 0) return 0;
    if (match_step<2>(a, b, 0, limit, lane, &m)) return m;
    for (i64 base = 64; base < limit; base += 32 * CMP_UNROLL)
        if (match_step<CMP_UNROLL>(a, b, base, limit, lane, &m)) return m;
    return limit;
}

// the dual walk's compare: every round trip looks at up to 32 x 10 tokens (a turn's new segment, the
// run of tokens a resumed walk usually has to confirm, fits one trip).  Three unrollings - 2, 4 or
// 10 rows - picked by the remaining length (warp uniform), so a short compare does not pay for the
// loads and votes of rows past its end; 32-bit indices (a label is shorter than 2^31 tokens).
template <int U>
__device__ __forceinline__ bool match_rows(const i32* __restrict__ pa, const i32* __restrict__ pb, i32 mine, i32* f) {
    i32 x[U], y[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
        const bool in = u * 32 < mine;  // this lane's token of row u is inside the compare
        x[u] = in ? __ldg(pa + u * 32) : 0;
        y[u] = in ? __ldg(pb + u * 32) : 1;
    }
#pragma unroll
    for (int u = 0; u < U; ++u) {
        const unsigned neq = __ballot_sync(0xffffffffu, x[u] != y[u]);
        if (neq) { *f = u * 32 + (__ffs(neq) - 1); return true; }
    }
    return false;
}
__device__ __forceinline__ i32 match_len_wide(const i32* __restrict__ a, const i32* __restrict__ b, i32 limit,
                                              int lane) {
    for (i32 base = 0; base < limit; base += 320) {
        const i32* __restrict__ pa = a + base + lane;
        const i32* __restrict__ pb = b + base + lane;
        const i32 rem = limit - base, mine = rem - lane;
        i32 f = 0;
        bool hit;
        if (rem <= 64) hit = match_rows<2>(pa, pb, mine, &f);
        else if (rem <= 128) hit = match_rows<4>(pa, pb, mine, &f);
        else hit = match_rows<10>(pa, pb, mine, &f);
        if (hit) { f += base; return f < limit ? f : limit; }
    }
    return limit > 0 ? limit : 0;
}

// Walk request tokens s[0..len) from the root.  start > 0: first re-descend to depth `start` by
// child lookups only (valid when the first `start` tokens are known to be cached).
__device__ __forceinline__ i32 radix_walk(const RadixDev& R, const i32* __restrict__ s, i64 len,
                                          i64 start, int lane, u32& c_look, u32& c_tok) {
    i32 v = 0;
    i64 d = 0;
    for (;;) {
        if (d >= len) break;
        i32 t = __ldg(s + d);
        ++c_look;
        i32 e = find_child(R.e_first_tok, __ldg(R.n_child_off + v), __ldg(R.n_child_off + v + 1), t, lane);
        if (e < 0) break;
        i32 u = __ldg(R.e_child + e);
        i64 L = __ldg(R.n_tok_len + u);
        if (d + L <= start) {  // whole edge inside the prefix known to be cached: no compares
            d += L;
            v = u;
            continue;
        }
        i64 skip = start > d ? start - d : 0;  // leading part of this edge already known equal
        const i32* lab = R.c_tokens + __ldg(R.n_tok_off + u);
        i64 limit = min(L, len - d);
        i64 m = skip + match_len(lab + skip, s + d + skip, limit - skip, lane);
        c_tok += (u32)(m - skip) + (m < limit ? 1u : 0u);
        d += m;
        if (m < L) break;
        v = u;
    }
    return (i32)d;
}

__global__ void __launch_bounds__(LPM_THREADS) k_lpm_radix(const i32* __restrict__ tokens,
                                                          const i64* __restrict__ tok_off, i64 N,
                                                          RadixDev R, i32* __restrict__ out,
                                                          unsigned long long* counters) {
    const int lane = threadIdx.x & 31;
    i64 r = ((i64)blockIdx.x * LPM_THREADS + threadIdx.x) >> 5;
    if (r >= N) return;
    i64 o = tok_off[r];
    i64 len = tok_off[r + 1] - o;
    u32 c_look = 0, c_tok = 0;
    i32 h = radix_walk(R, tokens + o, len, 0, lane, c_look, c_tok);
    if (lane == 0) out[r] = h;
    if (counters && lane == 0) {
        atomicAdd(counters + 0, 1ull);
        atomicAdd(counters + 1, (unsigned long long)c_look);
        atomicAdd(counters + 2, (unsigned long long)c_tok);
    }
}

__device__ __forceinline__ bool table_has(const u64* __restrict__ t_keys, u64 mask, u64 key) {
    u64 p = key & mask;
    for (;;) {
        u64 tk = ld_u64_keep(t_keys + p);
        if (tk == key) return true;
        if (tk == PEEK_EMPTY) return false;
        p = (p + 1) & mask;
    }
}

__global__ void __launch_bounds__(LPM_THREADS) k_lpm_hash(const u64* __restrict__ hashes,
                                                         const i64* __restrict__ blk_off, i64 N,
                                                         const u64* __restrict__ t_keys, u64 mask,
                                                         i32* __restrict__ out, unsigned long long* counters) {
    const int lane = threadIdx.x & 31;
    i64 r = ((i64)blockIdx.x * LPM_THREADS + threadIdx.x) >> 5;
    if (r >= N) return;
    i64 b0 = blk_off[r];
    i64 nb = blk_off[r + 1] - b0;
    i64 i0 = 0;
    i64 hit = nb;
    u32 c_probe = 0;
    for (; i0 < nb; i0 += 32) {
        i64 i = i0 + lane;
        bool miss = false;
        if (i < nb) miss = !table_has(t_keys, mask, hashes[b0 + i]);
        c_probe += (u32)__popc(__ballot_sync(0xffffffffu, i < nb));
        unsigned m = __ballot_sync(0xffffffffu, miss);
        if (m) { hit = i0 + (__ffs(m) - 1); break; }
    }
    if (lane == 0) out[r] = (i32)(hit * 16);
    if (counters && lane == 0) { atomicAdd(counters + 0, 1ull); atomicAdd(counters + 3, (unsigned long long)c_probe); }
}

// ---- small queues: both modes in ONE launch, a warp per request ------------------------------------
// The paper's queues hold 60-200 requests: there the call is bound by launches, not by
// the walks, so the co-descent machinery (edge table, counters, scans) is skipped: every request
// walks on its own, radix mode then hash mode, in one kernel.
__global__ void __launch_bounds__(LPM_THREADS) k_lpm_small(const i32* __restrict__ tokens,
                                                          const i64* __restrict__ tok_off,
                                                          const u64* __restrict__ hashes,
                                                          const i64* __restrict__ blk_off, i64 N, RadixDev R,
                                                          const u64* __restrict__ t_keys, u64 mask,
                                                          i32* __restrict__ hit_radix, i32* __restrict__ hit_hash,
                                                          unsigned long long* counters) {
    const int lane = threadIdx.x & 31;
    const i64 r = ((i64)blockIdx.x * LPM_THREADS + threadIdx.x) >> 5;
    if (r >= N) return;
    u32 c_look = 0, c_tok = 0, c_probe = 0;
    if (hit_radix) {
        const i64 o = tok_off[r];
        const i32 h = radix_walk(R, tokens + o, tok_off[r + 1] - o, 0, lane, c_look, c_tok);
        if (lane == 0) hit_radix[r] = h;
    }
    if (hit_hash) {
        const i64 b0 = blk_off[r], nb = blk_off[r + 1] - b0;
        i64 hit = nb;
        for (i64 i0 = 0; i0 < nb; i0 += 32) {
            const i64 i = i0 + lane;
            bool miss = false;
            if (i < nb) miss = !table_has(t_keys, mask, hashes[b0 + i]);
            c_probe += (u32)__popc(__ballot_sync(0xffffffffu, i < nb));
            const unsigned m = __ballot_sync(0xffffffffu, miss);
            if (m) { hit = i0 + (__ffs(m) - 1); break; }
        }
        if (lane == 0) hit_hash[r] = (i32)(hit * 16);
    }
    if (counters && lane == 0) {
        atomicAdd(counters + 0, (unsigned long long)((hit_radix ? 1 : 0) + (hit_hash ? 1 : 0)));
        if (c_look) atomicAdd(counters + 1, (unsigned long long)c_look);
        if (c_tok) atomicAdd(counters + 2, (unsigned long long)c_tok);
        if (c_probe) atomicAdd(counters + 3, (unsigned long long)c_probe);
    }
}

// ---- speculative co-descent (small N, long requests) -----------------------------------------
// Every sorted position j walks on its own, in parallel, but starts at depth s_j = B*lcp[j] (radix
// mode re-descends to s_j by child lookups only): W_j.  W_j is the true hit whenever
// hit(j-1) >= s_j; otherwise hit(j) = hit(j-1).  The recurrence is resolved by a scan (below).
// Preferred when there are too few requests for the sequential dual-walk to fill the machine.
__global__ void __launch_bounds__(LPM_THREADS) k_lpm_radix_spec(const i32* __restrict__ tokens,
                                                          const i64* __restrict__ tok_off, i64 N,
                                                          RadixDev R, const i32* __restrict__ order,
                                                          const i32* __restrict__ lcp,
                                                          i32* __restrict__ out) {
    const int lane = threadIdx.x & 31;
    i64 j = ((i64)blockIdx.x * LPM_THREADS + threadIdx.x) >> 5;
    if (j >= N) return;
    i64 r = order ? order[j] : j;
    i64 start = order ? (i64)lcp[j] * 16 : 0;
    i64 o = tok_off[r];
    i64 len = tok_off[r + 1] - o;
    u32 c_look = 0, c_tok = 0;
    i32 h = radix_walk(R, tokens + o, len, start, lane, c_look, c_tok);
    if (lane == 0) out[j] = h;  // by sorted position when co-descending, by request otherwise
}

__global__ void __launch_bounds__(LPM_THREADS) k_lpm_hash_spec(const u64* __restrict__ hashes,
                                                         const i64* __restrict__ blk_off, i64 N,
                                                         const u64* __restrict__ t_keys, u64 mask,
                                                         const i32* __restrict__ order,
                                                         const i32* __restrict__ lcp,
                                                         i32* __restrict__ out) {
    const int lane = threadIdx.x & 31;
    i64 j = ((i64)blockIdx.x * LPM_THREADS + threadIdx.x) >> 5;
    if (j >= N) return;
    i64 r = order ? order[j] : j;
    i64 b0 = blk_off[r];
    i64 nb = blk_off[r + 1] - b0;
    i64 i0 = order ? lcp[j] : 0;
    i64 hit = nb;
    for (; i0 < nb; i0 += 32) {
        i64 i = i0 + lane;
        bool miss = false;
        if (i < nb) miss = !table_has(t_keys, mask, hashes[b0 + i]);
        unsigned m = __ballot_sync(0xffffffffu, miss);
        if (m) { hit = i0 + (__ffs(m) - 1); break; }
    }
    if (lane == 0) out[j] = (i32)(hit * 16);
}

// ---- resolve: H_j = (H_{j-1} >= s_j) ? W_j : H_{j-1},  s_j = B*lcp[j] -------------------------
// Each position is the function f_j(x) = x if x < s_j else W'_j with W'_j = max(W_j, s_j) (W_j is
// only used when the resumed walk was valid, and then W_j >= s_j).  Functions "x below a
// threshold a, else the constant c >= a" are closed under composition:
//   (t,U) o (s,W) = (t,U) if t <= s, else (s, W < t ? W : U)
// so the recurrence is an inclusive scan with an associative operator; a group start has s = 0,
// which makes every later composite a constant, i.e. groups need no explicit segmentation.
struct Fn { i32 a, c; };
__device__ __forceinline__ Fn fn_id() { return Fn{0x7fffffff, 0x7fffffff}; }
__device__ __forceinline__ Fn fn_comb(Fn f, Fn g) {  // g after f
    if (g.a <= f.a) return g;
    return Fn{f.a, f.c < g.a ? f.c : g.c};
}
__device__ __forceinline__ Fn fn_shfl_up(Fn v, int o) {
    Fn r;
    r.a = __shfl_up_sync(0xffffffffu, v.a, o);
    r.c = __shfl_up_sync(0xffffffffu, v.c, o);
    return r;
}
__device__ __forceinline__ Fn fn_load(const i32* __restrict__ lcp, const i32* __restrict__ W, i64 j, i64 N) {
    if (j >= N) return fn_id();
    i64 s = (i64)lcp[j] * 16;
    i32 w = W[j];
    Fn f;
    f.a = (i32)s;
    f.c = (i64)w > s ? w : (i32)s;
    return f;
}

static constexpr int RS_THREADS = 256, RS_ITEMS = 8, RS_CHUNK = RS_THREADS * RS_ITEMS;

// CTA-wide exclusive scan of one Fn per thread; *total = composite of the whole CTA
__device__ __forceinline__ Fn block_exscan_fn(Fn v, Fn* sm, Fn* total) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
    Fn inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        Fn t = fn_shfl_up(inc, o);
        if (lane >= o) inc = fn_comb(t, inc);
    }
    Fn exw = fn_shfl_up(inc, 1);
    if (lane == 0) exw = fn_id();
    if (lane == 31) sm[w] = inc;
    __syncthreads();
    if (w == 0) {
        Fn s = lane < nw ? sm[lane] : fn_id();
        Fn si = s;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            Fn t = fn_shfl_up(si, o);
            if (lane >= o) si = fn_comb(t, si);
        }
        Fn ex = fn_shfl_up(si, 1);
        if (lane == 0) ex = fn_id();
        if (lane < nw) sm[lane] = ex;
        if (lane == 31) sm[32] = si;
    }
    __syncthreads();
    Fn r = fn_comb(sm[w], exw);
    *total = sm[32];
    __syncthreads();
    return r;
}

__global__ void __launch_bounds__(RS_THREADS) k_resolve_partial(const i32* __restrict__ lcp,
                                                               const i32* __restrict__ W, i64 N,
                                                               Fn* __restrict__ partial) {
    __shared__ Fn sm[34];
    i64 j0 = (i64)blockIdx.x * RS_CHUNK + (i64)threadIdx.x * RS_ITEMS;
    Fn acc = fn_id();
#pragma unroll
    for (int it = 0; it < RS_ITEMS; ++it) acc = fn_comb(acc, fn_load(lcp, W, j0 + it, N));
    Fn tot;
    block_exscan_fn(acc, sm, &tot);
    if (threadIdx.x == 0) partial[blockIdx.x] = tot;
}

__global__ void __launch_bounds__(1024) k_resolve_scan(Fn* __restrict__ partial, i64 n) {
    __shared__ Fn sm[34];
    Fn carry = fn_id();
    for (i64 b = 0; b < n; b += 1024) {
        i64 i = b + threadIdx.x;
        Fn v = i < n ? partial[i] : fn_id();
        Fn tot;
        Fn ex = block_exscan_fn(v, sm, &tot);
        if (i < n) partial[i] = fn_comb(carry, ex);
        carry = fn_comb(carry, tot);
    }
}

__global__ void __launch_bounds__(RS_THREADS) k_resolve_apply(const i32* __restrict__ order,
                                                             const i32* __restrict__ lcp,
                                                             const i32* __restrict__ W, i64 N,
                                                             const Fn* __restrict__ partial,
                                                             i32* __restrict__ hit) {
    __shared__ Fn sm[34];
    i64 j0 = (i64)blockIdx.x * RS_CHUNK + (i64)threadIdx.x * RS_ITEMS;
    Fn f[RS_ITEMS];
    Fn acc = fn_id();
#pragma unroll
    for (int it = 0; it < RS_ITEMS; ++it) {
        f[it] = fn_load(lcp, W, j0 + it, N);
        acc = fn_comb(acc, f[it]);
    }
    Fn tot;
    Fn ex = fn_comb(partial[blockIdx.x], block_exscan_fn(acc, sm, &tot));
#pragma unroll
    for (int it = 0; it < RS_ITEMS; ++it) {
        ex = fn_comb(ex, f[it]);
        // position 0 has s = 0, so every inclusive composite is a constant: its value is c
        if (j0 + it < N) hit[order[j0 + it]] = ex.c;
    }
}

// one CTA does the whole scan (small N: one launch instead of three)
__global__ void __launch_bounds__(1024) k_resolve_single(const i32* __restrict__ order,
                                                         const i32* __restrict__ lcp,
                                                         const i32* __restrict__ W, i64 N,
                                                         i32* __restrict__ hit) {
    __shared__ Fn sm[34];
    Fn carry = fn_id();
    for (i64 base = 0; base < N; base += 1024 * RS_ITEMS) {
        const i64 j0 = base + (i64)threadIdx.x * RS_ITEMS;
        Fn f[RS_ITEMS];
        Fn acc = fn_id();
#pragma unroll
        for (int it = 0; it < RS_ITEMS; ++it) {
            f[it] = fn_load(lcp, W, j0 + it, N);
            acc = fn_comb(acc, f[it]);
        }
        Fn tot;
        Fn ex = fn_comb(carry, block_exscan_fn(acc, sm, &tot));
#pragma unroll
        for (int it = 0; it < RS_ITEMS; ++it) {
            ex = fn_comb(ex, f[it]);
            if (j0 + it < N) hit[order[j0 + it]] = ex.c;
        }
        carry = fn_comb(carry, tot);
    }
}

// ---- dual-walk over the sorted order (PAPER.md:65-90 Alg. 1, :96) ------------------------------
// A warp owns a RUN of consecutive sorted positions and processes it in order, carrying the
// predecessor's hit and - in radix mode - the predecessor's path through the cache (the nodes it
// entered and the depth it entered them at; a stack in shared memory).  For position j with
// s = B*lcp[j] tokens shared with j-1:
//     hit(j-1) <  s : hit(j) = hit(j-1), nothing is read from the cache
//     hit(j-1) >= s : pop the path back to depth s and resume the walk inside the node that covers
//                     s - no re-descent from the root, no compares below s
// which is the co-descent of the pending trie (order + lcp) against the radix cache: one cache
// walk per pending edge.  Runs are cut at the position of minimal lcp inside fixed windows of
// `win` positions (cheap heads: a run head has no predecessor and does a full walk from the root).
//
// ONE persistent kernel serves both modes: its warps draw work items from an atomic counter, the
// radix windows first (they are the longer ones), then the hash windows, so the two modes overlap
// and the tail of one is filled by the other.  What the radix walk reads per node is packed:
//   * k_lpm_prep builds one 32-byte EdgeInfo per child edge (child, label length and offset, the
//     child's own edge range), so a child lookup costs the search over first tokens + ONE sector
//     instead of four dependent reads (e_child -> n_tok_len, n_tok_off -> n_child_off);
//   * the first tokens of the root's edges (the hottest node: every run head searches it) are
//     staged in shared memory by every CTA (north_star: "staging of the hot top levels").
// Labels are compared 32 lanes x CMP_UNROLL tokens per round trip with coalesced 32-bit loads: the
// kernel is bound by dependent round trips, one register holds one token in flight whatever the
// load width, and the two streams are misaligned against each other by an arbitrary number of
// tokens, so 128-bit loads would cost a second load on one stream for the same tokens in flight.
struct __align__(32) EdgeInfo {
    i32 child, tok_len;
    i64 tok_off;
    i32 ce0, ce1;  // the child's edge range
    i32 pad[2];
};

__global__ void __launch_bounds__(256) k_lpm_prep(RadixDev R, i32 E, EdgeInfo* __restrict__ info) {
    const i32 e = blockIdx.x * 256 + threadIdx.x;
    if (e >= E) return;
    const i32 u = R.e_child[e];
    EdgeInfo x;
    x.child = u; x.tok_len = R.n_tok_len[u]; x.tok_off = R.n_tok_off[u];
    x.ce0 = R.n_child_off[u]; x.ce1 = R.n_child_off[u + 1];
    x.pad[0] = x.pad[1] = 0;
    info[e] = x;
}

#ifndef PEEK_DW_THREADS
#define PEEK_DW_THREADS 256
#endif
#ifndef PEEK_DW_CAP
#define PEEK_DW_CAP 8
#endif
static constexpr int DW_THREADS = PEEK_DW_THREADS;   // k_lpm_dual: several CTAs per SM
static constexpr int DW_WARPS = DW_THREADS / 32;
static constexpr int DW_ROOT_STAGE = 2048;  // first tokens of the root's edges kept in shared memory

// first position of minimal lcp in [w0, w0 + win) (clipped to N); w0 = 0 gives 0 (lcp[0] = 0)
__device__ __forceinline__ i64 window_head(const i32* __restrict__ lcp, i64 w0, int win, i64 N, int lane) {
    if (w0 >= N) return N;
    i32 best = 0x7fffffff, bidx = 0x7fffffff;
    for (int t = 0; t < win; t += 32) {
        i64 j = w0 + t + lane;
        i32 v = (t + lane < win && j < N) ? __ldg(lcp + j) : 0x7fffffff;
        i32 m = __reduce_min_sync(0xffffffffu, v);
        i32 idx = __reduce_min_sync(0xffffffffu, v == m ? t + lane : 0x7fffffff);
        if (m < best) { best = m; bidx = idx; }
    }
    return w0 + bidx;
}

struct PathEntry { i32 ds, L, ce0, ce1; i64 lab; };  // node entered at token depth ds; label length, offset; its edges

struct DualArgs {
    const i32* tokens; const i64* tok_off;
    const u64* hashes; const i64* blk_off;
    i64 N;
    RadixDev R; const EdgeInfo* info;                // radix mode (hit_radix != NULL)
    const u64* t_keys; u64 mask;                     // hash mode (hit_hash != NULL)
    const i32* order; const i32* lcp;
    i32 V, E; i64 CT;  // extents of the radix arrays (range checks of the checked build)
    int win;
    i32 *hit_radix, *hit_hash;
    u32* ctr;             // work-item counter (zero on entry)
    unsigned long long* counters;  // NULL or [4]: walks, child lookups, tokens compared, table probes
};

// edge index in [e0, e1) whose first token equals t, or -1; `ft` = the first-token array the range
// indexes (global, or the staged copy of the root's)
__device__ __forceinline__ i32 find_child_in(const i32* ft, i32 e0, i32 e1, i32 t, int lane, bool smem) {
    while (e1 - e0 > 32) {
        i32 n = e1 - e0;
        i32 step = (n + 31) >> 5;
        i32 pos = e0 + lane * step;
        bool le = pos < e1 && (smem ? ft[pos] : __ldg(ft + pos)) <= t;
        unsigned m = __ballot_sync(0xffffffffu, le);
        if (m == 0) return -1;
        int k = 31 - __clz(m);
        e0 = e0 + k * step;
        e1 = min(e0 + step, e1);
    }
    i32 f = (e0 + lane < e1) ? (smem ? ft[e0 + lane] : __ldg(ft + e0 + lane)) : 0;
    unsigned m = __ballot_sync(0xffffffffu, (e0 + lane < e1) && f == t);
    return m ? e0 + (__ffs(m) - 1) : -1;
}

#ifndef PEEK_DW_MINB
#define PEEK_DW_MINB 4
#endif
// RADIX selects the mode at compile time: the two instantiations get their own register budgets
// (the hash probe loop is lean and wants every warp slot of the SM; the radix walk is not)
template <bool RADIX, bool UPFRONT>
__global__ void __launch_bounds__(DW_THREADS, RADIX ? PEEK_DW_MINB : 8) k_lpm_dual(DualArgs A) {
    __shared__ i32 root_ft[DW_ROOT_STAGE];
    __shared__ PathEntry stack[DW_WARPS][32];
    const unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31, wi = threadIdx.x >> 5;
    const i64 N = A.N;
    const int win = A.win;
    const i64 nwin = (N + win - 1) / win;
    const i64 n_items = nwin;
    const i32 root_e0 = RADIX ? __ldg(A.R.n_child_off) : 0, root_e1 = RADIX ? __ldg(A.R.n_child_off + 1) : 0;
    const i32 root_staged = root_e0 == 0 ? min(root_e1, (i32)DW_ROOT_STAGE) : 0;  // node 0 = root: edges [0, root_e1)
    for (int i = threadIdx.x; i < root_staged; i += DW_THREADS) root_ft[i] = __ldg(A.R.e_first_tok + i);
    __syncthreads();
    PathEntry* st = stack[wi];
    u32 c_walks = 0, c_look = 0, c_tok = 0, c_probe = 0;
    for (;;) {
        u32 item = 0;
        if (lane == 0) item = atomicAdd(A.ctr, 1u);
        item = __shfl_sync(FULL, item, 0);
        if ((i64)item >= n_items) break;
        const i64 w0 = (i64)item * win;
        const i64 head = window_head(A.lcp, w0, win, N, lane);
        const i64 end = window_head(A.lcp, w0 + win, win, N, lane);
        if (RADIX) {
            int top = 0;  // stack entries in use (<= 32; deeper nodes are not recorded)
            i32 Hprev = 0;
            for (i64 jb = head; jb < end; jb += 32) {
                const i64 jl = jb + lane;
                const bool valid = jl < end;
                const i32 r_l = valid ? __ldg(A.order + jl) : 0;
                PEEK_CHECK(r_l >= 0 && (i64)r_l < N, "order[] entry out of range");
                const i32 s_l = valid ? 16 * __ldg(A.lcp + jl) : 0;
                const i64 o_l = valid ? __ldg(A.tok_off + r_l) : 0;
                const i32 len_l = valid ? (i32)(__ldg(A.tok_off + r_l + 1) - o_l) : 0;
                i32 H_l = 0;
                const int cnt = (int)min((i64)32, end - jb);
                // positions that only copy their predecessor's hit are skipped in one vote: the next
                // position that has to touch the cache is the first one whose shared depth the
                // current hit reaches (the run's first position always walks)
                for (int i = 0; i < cnt; ++i) {
                    const bool first = (jb == head && i == 0);
                    if (!first) {
                        const unsigned wm = __ballot_sync(FULL, lane >= i && lane < cnt && s_l <= Hprev);
                        const int nx = wm ? __ffs(wm) - 1 : cnt;
                        if (lane >= i && lane < nx) H_l = Hprev;
                        i = nx;
                        if (i >= cnt) break;
                    }
                    i32 s = __shfl_sync(FULL, s_l, i);
                    if (first) s = 0;
                    i32 H;
                    {
                        const i64 o = __shfl_sync(FULL, o_l, i);
                        const i32 len = __shfl_sync(FULL, len_l, i);
                        const i32* __restrict__ q = A.tokens + o;
                        if (first) ++c_walks;
                        // deepest recorded entry entered strictly above depth s
                        const unsigned mk = __ballot_sync(FULL, lane < top && st[lane].ds < s);
                        i32 d = 0, ce0 = root_e0, ce1 = root_e1;  // position in the cache: depth, edges of the node below
                        bool at_root = true, stop = false;
                        if (mk) {
                            const int k = 31 - __clz(mk);
                            top = k + 1;
                            const PathEntry pe = st[k];
                            const i32 off = s - pe.ds;
                            if (off >= pe.L) {  // node fully inside the shared prefix: continue below it
                                d = pe.ds + pe.L;
                            } else {
                                const i32 limit = min(pe.L, len - pe.ds);
                                const i32 m = off + (i32)match_len_wide(A.R.c_tokens + pe.lab + off, q + pe.ds + off, limit - off, lane);
                                c_tok += (u32)(m - off) + (m < limit ? 1u : 0u);
                                d = pe.ds + m;
                                if (m < pe.L) stop = true;
                            }
                            ce0 = pe.ce0; ce1 = pe.ce1; at_root = false;
                        } else {
                            top = 0;
                        }
                        while (!stop && d < len) {
                            const i32 t = __ldg(q + d);
                            ++c_look;
                            const bool sm = at_root && ce1 <= root_staged;
                            const i32 e = find_child_in(sm ? root_ft : A.R.e_first_tok, ce0, ce1, t, lane, sm);
                            if (e < 0) break;
                            PEEK_CHECK(e < A.E, "edge index out of range");
                            const EdgeInfo ei = A.info[e];
                            PEEK_CHECK(ei.child > 0 && ei.child < A.V && ei.tok_off >= 0 && ei.tok_off + ei.tok_len <= A.CT &&
                                       ei.ce0 <= ei.ce1 && ei.ce1 <= A.E, "radix node out of range");
                            if (top < 32) {
                                if (lane == 0) st[top] = PathEntry{d, ei.tok_len, ei.ce0, ei.ce1, ei.tok_off};
                                ++top;
                            }
                            __syncwarp();
                            ce0 = ei.ce0; ce1 = ei.ce1; at_root = false;
                            const i32 L = ei.tok_len;
                            if (d + L <= s) { d += L; continue; }  // still inside the shared prefix: no compares
                            const i32 skip = s > d ? s - d : 0;
                            const i32 limit = min(L, len - d);
                            const i32 m = skip + (i32)match_len_wide(A.R.c_tokens + ei.tok_off + skip, q + d + skip, limit - skip, lane);
                            c_tok += (u32)(m - skip) + (m < limit ? 1u : 0u);
                            d += m;
                            if (m < L) break;
                        }
                        H = d;
                    }
                    Hprev = H;
                    if (lane == i) H_l = H;
                }
                if (valid) A.hit_radix[r_l] = H_l;
            }
        } else {
            i32 Hprev = 0;  // in blocks
            for (i64 jb = head; jb < end; jb += 32) {
                const i64 jl = jb + lane;
                const bool valid = jl < end;
                const i32 r_l = valid ? __ldg(A.order + jl) : 0;
                PEEK_CHECK(r_l >= 0 && (i64)r_l < N, "order[] entry out of range");
                const i32 s_l = valid ? __ldg(A.lcp + jl) : 0;
                const i64 b_l = valid ? __ldg(A.blk_off + r_l) : 0;
                const i32 nb_l = valid ? (i32)(__ldg(A.blk_off + r_l + 1) - b_l) : 0;
                i32 H_l = 0;
                const int cnt = (int)min((i64)32, end - jb);
                // A walk resumed at the shared depth often misses at once (the branch below the shared
                // prefix is not cached), and that first probe does not depend on the predecessor's hit.
                // When the queue has too few windows to fill the machine (UPFRONT: the call is bound by
                // the chain of dependent trips inside a window, not by throughput), every position of the
                // batch makes it up front, side by side, and a miss there costs the sequential loop no
                // memory round trip.  On a full machine the extra probes cost more than they save.
                const bool up_l = UPFRONT && valid && s_l < nb_l;
                bool miss0_l = false;
                if (UPFRONT && up_l) miss0_l = !table_has(A.t_keys, A.mask, ld_u64_once(A.hashes + b_l + s_l));
                if (UPFRONT) c_probe += (u32)__popc(__ballot_sync(FULL, up_l));
                for (int i = 0; i < cnt; ++i) {
                    const bool first = (jb == head && i == 0);
                    if (!first) {  // skip the positions that only copy (see the radix loop)
                        const unsigned wm = __ballot_sync(FULL, lane >= i && lane < cnt && s_l <= Hprev);
                        const int nx = wm ? __ffs(wm) - 1 : cnt;
                        if (lane >= i && lane < nx) H_l = Hprev;
                        i = nx;
                        if (i >= cnt) break;
                    }
                    i32 s = __shfl_sync(FULL, s_l, i);
                    if (first) s = 0;
                    i32 H;
                    {
                        const i64 b0 = __shfl_sync(FULL, b_l, i);
                        const i32 nb = __shfl_sync(FULL, nb_l, i);
                        if (first) ++c_walks;
                        H = nb;
                        i32 from = s;
                        if (UPFRONT && !first && s < nb) {  // the block at the shared depth was probed up front
                            if (__shfl_sync(FULL, (int)miss0_l, i)) { H = s; from = nb; }
                            else from = s + 1;
                        }
                        int batch = 32;
                        for (i32 i0 = from; i0 < nb; i0 += batch, batch = 32) {
                            const i32 x = i0 + lane;
                            bool miss = false;
                            const bool act = lane < batch && x < nb;
                            if (act) miss = !table_has(A.t_keys, A.mask, ld_u64_once(A.hashes + b0 + x));
                            c_probe += (u32)__popc(__ballot_sync(FULL, act));
                            const unsigned m = __ballot_sync(FULL, miss);
                            if (m) { H = i0 + (__ffs(m) - 1); break; }
                        }
                    }
                    Hprev = H;
                    if (lane == i) H_l = H;
                }
                if (valid) A.hit_hash[r_l] = H_l * 16;
            }
        }
    }
    if (A.counters && lane == 0) {
        if (c_walks) atomicAdd(A.counters + 0, (unsigned long long)c_walks);
        if (c_look) atomicAdd(A.counters + 1, (unsigned long long)c_look);
        if (c_tok) atomicAdd(A.counters + 2, (unsigned long long)c_tok);
        if (c_probe) atomicAdd(A.counters + 3, (unsigned long long)c_probe);
    }
}

// ---- per-radix-node pending demand (R26) ------------------------
// node_demand[v] = pending requests whose match enters node v.  The hit length is known, so a warp
// re-descends its request by child lookups only (no label compares) down to depth hit[r] and counts
// every node on the way; the root (entered by all) is written directly.
__global__ void __launch_bounds__(LPM_THREADS) k_radix_demand(const i32* __restrict__ tokens,
                                                             const i64* __restrict__ tok_off, i64 N,
                                                             RadixDev R, const i32* __restrict__ hit,
                                                             i32* __restrict__ node_demand) {
    const int lane = threadIdx.x & 31;
    const i64 r = ((i64)blockIdx.x * LPM_THREADS + threadIdx.x) >> 5;
    if (r >= N) return;
    const i32* __restrict__ s = tokens + tok_off[r];
    const i64 h = hit[r];
    i32 v = 0;
    i64 d = 0;
    while (d < h) {  // tokens [0, h) are cached: the edge starting with s[d] exists
        const i32 e = find_child(R.e_first_tok, __ldg(R.n_child_off + v), __ldg(R.n_child_off + v + 1), __ldg(s + d), lane);
        if (e < 0) break;  // cannot happen for a hit produced by peek_lpm on the same cache
        const i32 u = __ldg(R.e_child + e);
        if (lane == 0) atomicAdd(node_demand + u, 1);
        d += __ldg(R.n_tok_len + u);
        v = u;
    }
}
__global__ void k_radix_demand_root(i32* node_demand, i32 n) { node_demand[0] = n; }

i64 lpm_ws_bytes(i64 N, i64 V) {  // speculative path: W per mode and the scan partials; dual walk: edge table + counter
    Arena a(nullptr);
    a.take<i32>(N);
    a.take<i32>(N);
    a.take<Fn>((N + RS_CHUNK - 1) / RS_CHUNK + 1);
    a.take<EdgeInfo>(V);
    a.take<u32>(64);
    return a.used;
}

static unsigned long long* g_lpm_counters = nullptr;  // peek_lpm_counters
static int g_lpm_strategy = 0;  // PEEK_OPT_LPM_STRATEGY
static int g_lpm_window = 0;    // PEEK_OPT_LPM_WINDOW
void lpm_set_option(int key, i64 v) {
    if (key == PEEK_OPT_LPM_STRATEGY) g_lpm_strategy = (int)v;
    if (key == PEEK_OPT_LPM_WINDOW) g_lpm_window = (int)v;
}

}  // namespace peek

using namespace peek;

extern "C" peek_status peek_lpm(const int32_t* tokens, const int64_t* tok_off, const uint64_t* hashes,
                                const int64_t* blk_off, int64_t N, int32_t block_size,
                                const peek_radix* radix, const peek_table* table,
                                const peek_tree_view* tree, int32_t* hit_radix, int32_t* hit_hash,
                                void* ws, int64_t ws_bytes, void* stream) {
    if (N < 0 || N >= 0x7fffffffLL) { set_error("peek_lpm: N out of range"); return PEEK_ERR_INVALID_ARG; }
    if (block_size != 16) { set_error("peek_lpm: block_size must be 16"); return PEEK_ERR_UNSUPPORTED; }
    if (hit_radix && (!radix || !tokens || !tok_off)) {
        set_error("peek_lpm: hit_radix needs radix, tokens and tok_off");
        return PEEK_ERR_INVALID_ARG;
    }
    if (hit_hash && (!table || !hashes || !blk_off)) {
        set_error("peek_lpm: hit_hash needs table, hashes and blk_off");
        return PEEK_ERR_INVALID_ARG;
    }
    if (hit_radix && (radix->V < 1 || !radix->n_child_off || !radix->n_tok_off || !radix->n_tok_len ||
                      (radix->E > 0 && (!radix->e_first_tok || !radix->e_child || !radix->c_tokens)))) {
        set_error("peek_lpm: incomplete peek_radix");
        return PEEK_ERR_INVALID_ARG;
    }
    if (hit_hash && (!table->t_keys || table->S < 2 || (table->S & (table->S - 1)))) {
        set_error("peek_lpm: table.S must be a power of two >= 2");
        return PEEK_ERR_INVALID_ARG;
    }
    if (tree && (!tree->order || !tree->lcp)) {
        set_error("peek_lpm: tree view needs order and lcp");
        return PEEK_ERR_INVALID_ARG;
    }
    if (N == 0 || (!hit_radix && !hit_hash)) return PEEK_OK;
    const i64 VE = hit_radix ? (radix->V > radix->E ? radix->V : radix->E) : 0;
    if (!ws || ((uintptr_t)ws & 255) || ws_bytes < lpm_ws_bytes(N, VE)) {
        set_error("peek_lpm: workspace NULL, misaligned or too small");
        return PEEK_ERR_WORKSPACE;
    }
    cudaStream_t st = (cudaStream_t)stream;
    const i32* order = tree ? tree->order : nullptr;
    const i32* lcp = tree ? tree->lcp : nullptr;
    const unsigned warps_grid = (unsigned)((N * 32 + LPM_THREADS - 1) / LPM_THREADS);
    // co-descent strategy: sequential dual-walk needs many runs to fill the machine
    const bool dual = tree && (g_lpm_strategy == PEEK_LPM_DUAL_WALK ||
                               g_lpm_strategy == PEEK_LPM_AUTO);  // (queues of <= LPM_SMALL_MAX requests took the one-launch path above)
    const bool spec = tree && !dual;
    // sorted positions per dual-walk window: enough windows to fill the machine (~8K warps), at
    // most 32 positions (a run head pays a full walk from the root)
    int win = 1;
    while (win < 32 && N / win > 8192) win *= 2;
    if (g_lpm_window > 0) win = g_lpm_window;
    Arena a(ws);
    i32* Wr = a.take<i32>(N);
    i32* Wh = a.take<i32>(N);
    const i64 nchunks = (N + RS_CHUNK - 1) / RS_CHUNK;
    Fn* partial = a.take<Fn>(nchunks + 1);
    EdgeInfo* info = a.take<EdgeInfo>(VE);
    u32* ctr = a.take<u32>(64);
    a.arm(st);
    auto resolve = [&](const i32* W, i32* hit) {
        if (N <= 65536) {
            Prof pr(PROF_LPM_RESOLVE, st, 1);
            k_resolve_single<<<1, 1024, 0, st>>>(order, lcp, W, N, hit);
        } else {
            Prof pr(PROF_LPM_RESOLVE, st, 3);
            k_resolve_partial<<<(unsigned)nchunks, RS_THREADS, 0, st>>>(lcp, W, N, partial);
            k_resolve_scan<<<1, 1024, 0, st>>>(partial, nchunks);
            k_resolve_apply<<<(unsigned)nchunks, RS_THREADS, 0, st>>>(order, lcp, W, N, partial, hit);
        }
    };
    RadixDev R{nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    if (hit_radix) R = RadixDev{radix->c_tokens, radix->n_tok_off, radix->n_tok_len,
                                radix->n_child_off, radix->e_first_tok, radix->e_child};
    if (g_lpm_strategy == PEEK_LPM_AUTO && N <= LPM_SMALL_MAX) {  // small queue: one launch for both modes
        Prof pr(hit_radix ? PROF_LPM_RADIX : PROF_LPM_HASH, st, 1);
        k_lpm_small<<<warps_grid, LPM_THREADS, 0, st>>>(tokens, tok_off, hashes, blk_off, N, R,
                                                        hit_hash ? table->t_keys : nullptr,
                                                        hit_hash ? (u64)(table->S - 1) : 0, hit_radix, hit_hash,
                                                        g_lpm_counters);
    } else if (dual) {  // persistent kernels, one per mode (plus the edge table of the radix cache)
        PEEK_CUDA(cudaMemsetAsync(ctr, 0, 256, st));
        DualArgs D;
        D.tokens = tokens; D.tok_off = tok_off; D.hashes = hashes; D.blk_off = blk_off; D.N = N;
        D.R = R; D.info = info;
        D.V = hit_radix ? radix->V : 0; D.E = hit_radix ? radix->E : 0; D.CT = hit_radix ? radix->CT : 0;
        D.t_keys = hit_hash ? table->t_keys : nullptr; D.mask = hit_hash ? (u64)(table->S - 1) : 0;
        D.order = order; D.lcp = lcp; D.win = win; D.hit_radix = hit_radix; D.hit_hash = hit_hash;
        D.counters = g_lpm_counters;
        const i64 items = (N + win - 1) / win;
        const bool upfront = items <= (i64)sm_count() * 64;  // fewer windows than warp slots: the call is latency bound
        i64 ctas = (items + DW_WARPS - 1) / DW_WARPS;
        const i64 cap = (i64)sm_count() * PEEK_DW_CAP;  // resident CTAs per SM - the warps loop over the items
        if (ctas > cap) ctas = cap;
        // both modes: the two walks are independent, so the hash probes run on the library's side
        // stream next to the radix walk (each is bound by dependent trips, not by the machine)
        SideStream ss;
        if (hit_radix && hit_hash && side_fork(st, &ss)) {
            Prof pr(PROF_LPM_DUAL, st, radix->E > 0 ? 3 : 2);
            D.ctr = ctr + 32;
            if (upfront) k_lpm_dual<false, true><<<(unsigned)ctas, DW_THREADS, 0, ss.side>>>(D);
            else k_lpm_dual<false, false><<<(unsigned)ctas, DW_THREADS, 0, ss.side>>>(D);
            if (radix->E > 0) k_lpm_prep<<<(unsigned)((radix->E + 255) / 256), 256, 0, st>>>(R, radix->E, info);
            D.ctr = ctr;
            k_lpm_dual<true, false><<<(unsigned)ctas, DW_THREADS, 0, st>>>(D);
            PEEK_CUDA(side_join(st, ss));
        } else {
            if (hit_radix) {
                Prof pr(PROF_LPM_RADIX, st, radix->E > 0 ? 2 : 1);
                if (radix->E > 0) k_lpm_prep<<<(unsigned)((radix->E + 255) / 256), 256, 0, st>>>(R, radix->E, info);
                D.ctr = ctr;
                k_lpm_dual<true, false><<<(unsigned)ctas, DW_THREADS, 0, st>>>(D);
            }
            if (hit_hash) {
                Prof pr(PROF_LPM_HASH, st, 1);
                D.ctr = ctr + 32;
                if (upfront) k_lpm_dual<false, true><<<(unsigned)ctas, DW_THREADS, 0, st>>>(D);
                else k_lpm_dual<false, false><<<(unsigned)ctas, DW_THREADS, 0, st>>>(D);
            }
        }
    } else {
        if (hit_radix) {
            {
                Prof pr(PROF_LPM_RADIX, st, 1);
                if (spec) k_lpm_radix_spec<<<warps_grid, LPM_THREADS, 0, st>>>(tokens, tok_off, N, R, order, lcp, Wr);
                else k_lpm_radix<<<warps_grid, LPM_THREADS, 0, st>>>(tokens, tok_off, N, R, hit_radix, g_lpm_counters);
            }
            if (spec) resolve(Wr, hit_radix);
        }
        if (hit_hash) {
            {
                Prof pr(PROF_LPM_HASH, st, 1);
                if (spec) k_lpm_hash_spec<<<warps_grid, LPM_THREADS, 0, st>>>(hashes, blk_off, N, table->t_keys, (u64)(table->S - 1), order, lcp, Wh);
                else k_lpm_hash<<<warps_grid, LPM_THREADS, 0, st>>>(hashes, blk_off, N, table->t_keys, (u64)(table->S - 1), hit_hash, g_lpm_counters);
            }
            if (spec) resolve(Wh, hit_hash);
        }
    }
    PEEK_CUDA(cudaGetLastError());
    return PEEK_OK;
}


extern "C" peek_status peek_lpm_counters(uint64_t* counters) {
    g_lpm_counters = (unsigned long long*)counters;
    return PEEK_OK;
}

extern "C" peek_status peek_radix_demand(const int32_t* tokens, const int64_t* tok_off, int64_t N,
                                         const peek_radix* radix, const int32_t* hit_radix,
                                         int32_t* node_demand, void* stream) {
    if (N < 0 || N >= 0x7fffffffLL) { set_error("peek_radix_demand: N out of range"); return PEEK_ERR_INVALID_ARG; }
    if (!radix || radix->V < 1 || !node_demand || !radix->n_child_off || !radix->n_tok_len ||
        (radix->E > 0 && (!radix->e_first_tok || !radix->e_child))) {
        set_error("peek_radix_demand: incomplete peek_radix or NULL output");
        return PEEK_ERR_INVALID_ARG;
    }
    if (N > 0 && (!tokens || !tok_off || !hit_radix)) {
        set_error("peek_radix_demand: NULL argument");
        return PEEK_ERR_INVALID_ARG;
    }
    cudaStream_t st = (cudaStream_t)stream;
    PEEK_CUDA(cudaMemsetAsync(node_demand, 0, sizeof(i32) * (size_t)radix->V, st));
    Prof pr(PROF_SIGNALS, st, 2);
    k_radix_demand_root<<<1, 1, 0, st>>>(node_demand, (i32)N);
    if (N > 0) {
        RadixDev R{radix->c_tokens, radix->n_tok_off, radix->n_tok_len, radix->n_child_off, radix->e_first_tok, radix->e_child};
        const unsigned grid = (unsigned)((N * 32 + LPM_THREADS - 1) / LPM_THREADS);
        k_radix_demand<<<grid, LPM_THREADS, 0, st>>>(tokens, tok_off, N, R, hit_radix, node_demand);
    }
    PEEK_CUDA(cudaGetLastError());
    return PEEK_OK;
}
