// peek_lpm.cu — a5/a6 peek_lpm: per-request longest prefix match against the engine's cache.
//
// Radix mode (the result of Alg. 1; "a partial match terminates the branch",
// PAPER.md:291): one warp per request.  Child lookup: a coalesced ballot over the sorted edge
// slice (32-ary narrowing when a node has more than 32 children, e.g. the root).  Edge labels are
// compared 32 lanes x CMP_UNROLL tokens per step, both streams coalesced.
// Hash mode ("per-request find_longest_cache_hit"): one warp per request, 32
// consecutive blocks probed per step in the open-addressed table, first miss wins.
//
// Co-descent ("one cache walk per pending edge"): with a peek_tree_view the
// request at sorted position j starts at depth s_j = B*lcp[j] (the prefix it shares with its sorted
// predecessor) instead of 0: W_j = the walk resumed at s_j (radix mode re-descends to s_j by child
// lookups only, no token compares).  A per-group pass then resolves
//   H_j = (H_{j-1} >= s_j) ? W_j : H_{j-1}
// (if the predecessor's hit ends inside the shared prefix, so does this request's, at the same
// place; otherwise the shared prefix is fully cached and the resumed walk is exact).
#include "peek_common.cuh"

namespace peek {

static constexpr int LPM_THREADS = 256;
static constexpr int CMP_UNROLL = 4;

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

// number of leading equal tokens of a[0..limit) and b[0..limit), warp-cooperative
__device__ __forceinline__ i64 match_len(const i32* __restrict__ a, const i32* __restrict__ b, i64 limit,
                                         int lane) {
    for (i64 base = 0; base < limit; base += 32 * CMP_UNROLL) {
        i32 x[CMP_UNROLL], y[CMP_UNROLL];
#pragma unroll
        for (int u = 0; u < CMP_UNROLL; ++u) {
            i64 i = base + u * 32 + lane;
            bool in = i < limit;
            x[u] = in ? __ldg(a + i) : 0;
            y[u] = in ? __ldg(b + i) : 1;
        }
#pragma unroll
        for (int u = 0; u < CMP_UNROLL; ++u) {
            unsigned neq = __ballot_sync(0xffffffffu, x[u] != y[u]);
            if (neq) {
                i64 m = base + u * 32 + (__ffs(neq) - 1);
                return m < limit ? m : limit;
            }
        }
    }
    return limit;
}

// Walk request tokens s[0..len) from the root.  start > 0: first re-descend to depth `start` by
// child lookups only (valid when the first `start` tokens are known to be cached).
__device__ __forceinline__ i32 radix_walk(const RadixDev& R, const i32* __restrict__ s, i64 len,
                                          i64 start, int lane) {
    i32 v = 0;
    i64 d = 0;
    for (;;) {
        if (d >= len) break;
        i32 t = __ldg(s + d);
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
        d += m;
        if (m < L) break;
        v = u;
    }
    return (i32)d;
}

__global__ void __launch_bounds__(LPM_THREADS) k_lpm_radix(const i32* __restrict__ tokens,
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
    i32 h = radix_walk(R, tokens + o, len, start, lane);
    if (lane == 0) out[j] = h;  // by sorted position when co-descending, by request otherwise
}

__device__ __forceinline__ bool table_has(const u64* __restrict__ t_keys, u64 mask, u64 key) {
    u64 p = key & mask;
    for (;;) {
        u64 tk = __ldg(t_keys + p);
        if (tk == key) return true;
        if (tk == PEEK_EMPTY) return false;
        p = (p + 1) & mask;
    }
}

__global__ void __launch_bounds__(LPM_THREADS) k_lpm_hash(const u64* __restrict__ hashes,
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

i64 lpm_ws_bytes(i64 N) {
    Arena a(nullptr);
    a.take<i32>(N);
    a.take<i32>(N);
    a.take<Fn>((N + RS_CHUNK - 1) / RS_CHUNK + 1);
    return a.used;
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
    if (!ws || ((uintptr_t)ws & 255) || ws_bytes < lpm_ws_bytes(N)) {
        set_error("peek_lpm: workspace NULL, misaligned or too small");
        return PEEK_ERR_WORKSPACE;
    }
    cudaStream_t st = (cudaStream_t)stream;
    Arena a(ws);
    i32* Wr = a.take<i32>(N);
    i32* Wh = a.take<i32>(N);
    const i32* order = tree ? tree->order : nullptr;
    const i32* lcp = tree ? tree->lcp : nullptr;
    unsigned warps_grid = (unsigned)((N * 32 + LPM_THREADS - 1) / LPM_THREADS);
    i64 nchunks = (N + RS_CHUNK - 1) / RS_CHUNK;
    Fn* partial = a.take<Fn>(nchunks + 1);
    if (hit_radix) {
        RadixDev R{radix->c_tokens, radix->n_tok_off, radix->n_tok_len,
                   radix->n_child_off, radix->e_first_tok, radix->e_child};
        {
            Prof pr(PROF_LPM_RADIX, st, 1);
            k_lpm_radix<<<warps_grid, LPM_THREADS, 0, st>>>(tokens, tok_off, N, R, order, lcp,
                                                           tree ? Wr : hit_radix);
        }
        if (tree) {
            Prof pr(PROF_LPM_RESOLVE, st, 3);
            k_resolve_partial<<<(unsigned)nchunks, RS_THREADS, 0, st>>>(lcp, Wr, N, partial);
            k_resolve_scan<<<1, 1024, 0, st>>>(partial, nchunks);
            k_resolve_apply<<<(unsigned)nchunks, RS_THREADS, 0, st>>>(order, lcp, Wr, N, partial, hit_radix);
        }
    }
    if (hit_hash) {
        {
            Prof pr(PROF_LPM_HASH, st, 1);
            k_lpm_hash<<<warps_grid, LPM_THREADS, 0, st>>>(hashes, blk_off, N, table->t_keys,
                                                          (u64)(table->S - 1), order, lcp,
                                                          tree ? Wh : hit_hash);
        }
        if (tree) {
            Prof pr(PROF_LPM_RESOLVE, st, 3);
            k_resolve_partial<<<(unsigned)nchunks, RS_THREADS, 0, st>>>(lcp, Wh, N, partial);
            k_resolve_scan<<<1, 1024, 0, st>>>(partial, nchunks);
            k_resolve_apply<<<(unsigned)nchunks, RS_THREADS, 0, st>>>(order, lcp, Wh, N, partial, hit_hash);
        }
    }
    PEEK_CUDA(cudaGetLastError());
    return PEEK_OK;
}
