// peek_signals.cu — a9 peek_clpm_signals: the remaining signals of Eq. 1 and Eq. 2
// (R20-R23):
//   section[r]      warm / pioneer / sibling            (PAPER.md:102; Alg. 2 lines 3-13, :325)
//   score[r]        ancestor score sum pending_count(v) * |edge(v)|
//   evict_score[p]  max over the ancestors of the cached block in slot p of
//                   pending_count * depth                                 (Eq. 2)
// All three are read off the pending trie as peek_pending_tree leaves it: sorted order + adjacent
// LCP.  For sorted position j the blocks [lcp[j], nb) first appear at j; walking the LCP array to
// the right with next-smaller-value searches splits them into STEPS of constant pending_count
// (each step is a trie edge, or the part of one that starts at j):
//   step (i_lo..i_hi, t):  blocks i_lo..i_hi of j are shared by exactly the positions j..t-1.
// score   every step adds count * length * B to all positions j..t-1: two atomics into a difference
//         array, then one prefix sum over the positions.
// evict   the value of a block is the prefix maximum of count * depth down its path.  The part
//         of the path above lcp[j] belongs to the position par(j) that introduced block lcp[j]-1
//         (a previous-smaller-value search); E_in(j) = max(g(j), E_in(par(j))) with g(j) the
//         maximum over par(j)'s own steps down to that block, resolved for all positions by
//         pointer jumping (log depth rounds).  Each position then walks its own steps shallow to
//         deep and writes the running maximum into the slot of every block that is cached.
// section the requests sharing the first two blocks are a run of sorted positions (lcp >= 2);
//         the pioneer of a run is the minimum (arrival, index) over its cold members.
#include "peek_grid.cuh"

namespace peek {

static constexpr int SG_THREADS = 256;

// ---- steps of one position, deep to shallow ------------------------------------------------------
// calls f(i_lo, i_hi, t) for every step of position j inside the depth range [d_lo, d_hi]
template <typename F>
__device__ __forceinline__ void for_steps_desc(const MinTree& mt, i64 j, i64 d_lo, i64 d_hi, F f) {
    i64 i_hi = d_hi, t = j + 1;
    while (i_hi >= d_lo) {
        t = nsv_next_less(mt, t, (i32)(i_hi + 1));  // first later position sharing <= i_hi blocks
        const i64 lt = mt.val(0, t);
        const i64 i_lo = lt > d_lo ? lt : d_lo;
        f(i_lo, i_hi, t);
        i_hi = i_lo - 1;
    }
}

// ---- score ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(SG_THREADS) k_score_steps(const i64* __restrict__ blk_off, i64 N,
                                                           const i32* __restrict__ order,
                                                           const i32* __restrict__ lcp, MinTree mt,
                                                           unsigned long long* __restrict__ diff) {
    for (i64 j = (i64)blockIdx.x * SG_THREADS + threadIdx.x; j < N; j += (i64)gridDim.x * SG_THREADS) {
        const i64 r = order[j];
        const i64 nb = blk_off[r + 1] - blk_off[r];
        const i64 l0 = lcp[j], l1 = j + 1 < N ? lcp[j + 1] : 0;
        const i64 own_lo = l0 > l1 ? l0 : l1;  // blocks only this request has
        unsigned long long add = (unsigned long long)((nb - own_lo) * 16);
        unsigned long long sub_next = add;     // what stops applying at position j + 1
        for_steps_desc(mt, j, l0, l1 - 1, [&](i64 i_lo, i64 i_hi, i64 t) {
            const unsigned long long v = (unsigned long long)((t - j) * (i_hi - i_lo + 1) * 16);
            add += v;
            if (t == j + 1) sub_next += v;
            else atomicAdd(diff + t, 0ull - v);
        });
        atomicAdd(diff + j, add);
        atomicAdd(diff + j + 1, 0ull - sub_next);  // diff has N + 1 entries
    }
}

// inclusive prefix sum of diff[0..N) (three launches), scattered to score[order[j]]
static constexpr int SC_ITEMS = 8, SC_CHUNK = SG_THREADS * SC_ITEMS;
__global__ void __launch_bounds__(SG_THREADS) k_sum_partial(const unsigned long long* __restrict__ v, i64 N,
                                                           i64* __restrict__ partial) {
    __shared__ i64 sm[34];
    const i64 j0 = (i64)blockIdx.x * SC_CHUNK + (i64)threadIdx.x * SC_ITEMS;
    i64 s = 0;
#pragma unroll
    for (int it = 0; it < SC_ITEMS; ++it) if (j0 + it < N) s += (i64)v[j0 + it];
    i64 tot;
    block_exscan_i64(s, sm, &tot);
    if (threadIdx.x == 0) partial[blockIdx.x] = tot;
}
__global__ void __launch_bounds__(1024) k_sum_scan(i64* __restrict__ partial, i64 n) {
    __shared__ i64 sm[34];
    i64 carry = 0;
    for (i64 b = 0; b < n; b += 1024) {
        const i64 i = b + threadIdx.x;
        const i64 v = i < n ? partial[i] : 0;
        i64 tot;
        const i64 ex = block_exscan_i64(v, sm, &tot);
        if (i < n) partial[i] = carry + ex;
        carry += tot;
    }
}
__global__ void __launch_bounds__(SG_THREADS) k_sum_apply(const unsigned long long* __restrict__ v, i64 N,
                                                         const i64* __restrict__ partial,
                                                         const i32* __restrict__ order,
                                                         i64* __restrict__ score) {
    __shared__ i64 sm[34];
    const i64 j0 = (i64)blockIdx.x * SC_CHUNK + (i64)threadIdx.x * SC_ITEMS;
    i64 x[SC_ITEMS], s = 0;
#pragma unroll
    for (int it = 0; it < SC_ITEMS; ++it) { x[it] = j0 + it < N ? (i64)v[j0 + it] : 0; s += x[it]; }
    i64 tot;
    i64 run = block_exscan_i64(s, sm, &tot) + partial[blockIdx.x];
#pragma unroll
    for (int it = 0; it < SC_ITEMS; ++it) {
        run += x[it];
        if (j0 + it < N) score[order[j0 + it]] = run;
    }
}

// ---- eviction score ------------------------------------------------------------------------------
// maximum of pending_count * depth (tokens) over position j's own steps inside depths [d_lo, d_hi]
__device__ __forceinline__ i64 own_max(const MinTree& mt, i64 j, i64 d_lo, i64 d_hi) {
    i64 g = 0;
    for_steps_desc(mt, j, d_lo, d_hi, [&](i64, i64 i_hi, i64 t) {
        const i64 v = (t - j) * 16 * (i_hi + 1);  // a step's maximum sits at its deepest block
        if (v > g) g = v;
    });
    return g;
}

// par[j] = the position that introduced block lcp[j] - 1 of j's path (-1 for a root child),
// ein[j] = the maximum over that position's own steps down to that block
__global__ void __launch_bounds__(SG_THREADS) k_evict_parent(i64 N, const i32* __restrict__ lcp, MinTree mt,
                                                            i32* __restrict__ par, i64* __restrict__ ein) {
    for (i64 j = (i64)blockIdx.x * SG_THREADS + threadIdx.x; j < N; j += (i64)gridDim.x * SG_THREADS) {
        const i64 l0 = lcp[j];
        if (l0 == 0) { par[j] = -1; ein[j] = 0; continue; }
        const i64 p = nsv_prev_less(mt, j - 1, (i32)l0);
        par[j] = (i32)p;
        ein[j] = own_max(mt, p, mt.val(0, p), l0 - 1);
    }
}

struct JumpCtl { u32 bar; u32 changed[2]; u32 pad; };

// ein[j] = max over the whole parent chain: pointer jumping, ping-pong buffers, until no pointer is left
__global__ void __launch_bounds__(1024, 1) k_evict_jump(i64 N, i32* par0, i64* ein0, i32* par1, i64* ein1,
                                                       JumpCtl* ctl, i32* result_buf) {
    Grid g{&ctl->bar, 0};
    const i64 gtid = (i64)blockIdx.x * blockDim.x + threadIdx.x, gsize = (i64)gridDim.x * blockDim.x;
    int cur = 0;
    for (int round = 0;; ++round) {
        const i32* ps = cur ? par1 : par0;
        const i64* es = cur ? ein1 : ein0;
        i32* pd = cur ? par0 : par1;
        i64* ed = cur ? ein0 : ein1;
        if (gtid == 0) ctl->changed[(round + 1) & 1] = 0;
        bool any = false;
        for (i64 j = gtid; j < N; j += gsize) {
            const i32 p = ps[j];
            i64 e = es[j];
            i32 np = -1;
            if (p >= 0) {
                const i64 ep = es[p];
                if (ep > e) e = ep;
                np = ps[p];
                any = true;
            }
            pd[j] = np;
            ed[j] = e;
        }
        if (__any_sync(0xffffffffu, any) && (threadIdx.x & 31) == 0) atomicOr(&ctl->changed[round & 1], 1u);
        g.sync();
        cur ^= 1;
        if (__ldcg(&ctl->changed[round & 1]) == 0) break;
        g.sync();  // the flag of this round is reset two rounds later: keep the rounds apart
    }
    if (gtid == 0) *result_buf = cur;
}

__device__ __forceinline__ i64 sg_table_slot(const u64* __restrict__ t_keys, u64 mask, u64 key) {
    u64 p = key & mask;
    for (;;) {
        const u64 tk = __ldg(t_keys + p);
        if (tk == key) return (i64)p;
        if (tk == PEEK_EMPTY) return -1;
        p = (p + 1) & mask;
    }
}

// A warp owns 32 consecutive sorted positions (the work distribution of k_demand): lane q describes
// position j0 + q - its chain, the range [l0, nb) of blocks that first appear there, its deepest
// shared step (blocks [lo1, l1) shared with positions j+1 .. t1-1) and the running maxima that
// apply above that step and above the unshared tail - then the new blocks of the 32 positions are
// flattened and handed out one per lane.  The value of a block is max(E_in, own steps down to it);
// blocks of shallower nested steps take a per-lane walk.
static constexpr int EV_WARPS = SG_THREADS / 32;
struct EvictMeta {
    i64 b0[32], above1[32], above_tail[32];
    i32 l0[32], l1[32], lo1[32], cnt1[32];
};

__global__ void __launch_bounds__(SG_THREADS) k_evict_write(const u64* __restrict__ hashes,
                                                           const i64* __restrict__ blk_off, i64 N,
                                                           const i32* __restrict__ order,
                                                           const i32* __restrict__ lcp, MinTree mt,
                                                           const i64* ein_a, const i64* ein_b,
                                                           const i32* __restrict__ which,
                                                           const u64* __restrict__ t_keys, u64 mask,
                                                           const unsigned char* __restrict__ tags,
                                                           i64* __restrict__ evict, int ppw) {
    __shared__ EvictMeta sm[EV_WARPS];
    const unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const i64 j0 = (((i64)blockIdx.x * SG_THREADS + threadIdx.x) >> 5) * ppw;  // ppw positions per warp
    if (j0 >= N) return;
    const i64* ein = *which ? ein_b : ein_a;
    EvictMeta& M = sm[w];
    const i64 j = j0 + lane;
    i32 n_new = 0;
    i64 e_in = 0;
    {
        const bool valid = lane < ppw && j < N;
        i64 b0 = 0;
        i32 nb = 0, l0 = 0, l1 = 0;
        if (valid) {
            const i64 r = __ldg(order + j);
            b0 = __ldg(blk_off + r);
            nb = (i32)(__ldg(blk_off + r + 1) - b0);
            l0 = __ldg(lcp + j);
            l1 = j + 1 < N ? __ldg(lcp + j + 1) : 0;
            n_new = nb - l0;
            e_in = ein[j];
        }
        i32 lo1 = l1, cnt1 = 1;
        i64 above1 = e_in, above_tail = e_in;
        if (valid && l1 > l0) {
            const i64 t = nsv_next_less(mt, j + 1, l1);
            const i32 lt = mt.val(0, t);
            lo1 = lt > l0 ? lt : l0;
            cnt1 = (i32)(t - j);
            if (lo1 > l0) { const i64 o = own_max(mt, j, l0, lo1 - 1); if (o > above1) above1 = o; }
            const i64 v1 = (i64)cnt1 * 16 * l1;  // the deepest shared step's maximum
            above_tail = v1 > above1 ? v1 : above1;
        }
        M.b0[lane] = b0; M.l0[lane] = l0; M.l1[lane] = l1; M.lo1[lane] = lo1; M.cnt1[lane] = cnt1;
        M.above1[lane] = above1; M.above_tail[lane] = above_tail;
    }
    i32 pre = n_new;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const i32 t = __shfl_up_sync(FULL, pre, o);
        if (lane >= o) pre += t;
    }
    const i32 total = __shfl_sync(FULL, pre, 31);
    const i32 excl = pre - n_new;
    __syncwarp();
    for (i32 base = 0; base < total; base += 32) {
        const i32 it = base + lane;
        const bool act = it < total;
        const i32 itc = act ? it : total - 1;
        int lo = 0, hi = 31;  // first position q with pre[q] > itc
#pragma unroll
        for (int s = 0; s < 5; ++s) {
            const int mid = (lo + hi) >> 1;
            const i32 v = __shfl_sync(FULL, pre, mid);
            if (v > itc) hi = mid; else lo = mid + 1;
        }
        const int q = lo;
        const i32 i = M.l0[q] + (itc - __shfl_sync(FULL, excl, q));
        const u64 key = __ldg(hashes + M.b0[q] + i);
        const i64 eq = __shfl_sync(FULL, e_in, q);
        i64 val;
        if (i >= M.l1[q]) {
            const i64 own = (i64)16 * (i + 1);
            val = own > M.above_tail[q] ? own : M.above_tail[q];
        } else if (i >= M.lo1[q]) {
            const i64 own = (i64)M.cnt1[q] * 16 * (i + 1);
            val = own > M.above1[q] ? own : M.above1[q];
        } else {
            const i64 own = own_max(mt, j0 + q, M.l0[q], i);
            val = own > eq ? own : eq;
        }
        if (act) {
            const i64 p = tags ? table_slot_tagged(t_keys, tags, mask, key, key & mask, ld_tagword(tags + ((key & mask) & ~7ull)))
                               : sg_table_slot(t_keys, mask, key);
            if (p >= 0) evict[p] = val;
        }
    }
}

// ---- sections ------------------------------------------------------------------------------------
__device__ __forceinline__ u64 sec_key(const i32* __restrict__ arrival, i64 r) {
    const u32 a = arrival ? ((u32)arrival[r] ^ 0x80000000u) : (u32)r;
    return ((u64)a << 32) | (u64)(u32)r;
}

__global__ void __launch_bounds__(SG_THREADS) k_section_min(const i64* __restrict__ blk_off, i64 N,
                                                           const i32* __restrict__ order, MinTree mt,
                                                           const i32* __restrict__ hit, i32 tau,
                                                           const i32* __restrict__ arrival,
                                                           i32* __restrict__ start,
                                                           unsigned long long* __restrict__ runmin) {
    for (i64 j = (i64)blockIdx.x * SG_THREADS + threadIdx.x; j < N; j += (i64)gridDim.x * SG_THREADS) {
        const i64 r = order[j];
        const i64 nb = blk_off[r + 1] - blk_off[r];
        i32 s = -1;  // warm, or no full block: no run
        if (hit[r] <= tau && nb > 0) {
            // the requests sharing the first two blocks (one, for a one-block prompt) are the run
            // of positions around j whose adjacent LCPs stay >= 2 (>= 1)
            s = (i32)nsv_prev_less(mt, j, nb >= 2 ? 2 : 1);
            atomicMin(runmin + s, (unsigned long long)sec_key(arrival, r));
        }
        start[j] = s;
    }
}

__global__ void __launch_bounds__(SG_THREADS) k_section_write(const i64* __restrict__ blk_off, i64 N,
                                                             const i32* __restrict__ order,
                                                             const i32* __restrict__ hit, i32 tau,
                                                             const i32* __restrict__ arrival,
                                                             const i32* __restrict__ start,
                                                             const unsigned long long* __restrict__ runmin,
                                                             i32* __restrict__ section) {
    for (i64 j = (i64)blockIdx.x * SG_THREADS + threadIdx.x; j < N; j += (i64)gridDim.x * SG_THREADS) {
        const i64 r = order[j];
        i32 sec;
        if (hit[r] > tau) sec = 0;
        else if (start[j] < 0) sec = 1;
        else sec = runmin[start[j]] == (unsigned long long)sec_key(arrival, r) ? 1 : 2;
        section[r] = sec;
    }
}

// ---- workspace ------------------------------------------------------------------------------------
struct SignalsWs {
    JumpCtl* ctl;
    i32* which;
    i32* mt_buf;
    unsigned long long* diff;   // N + 1
    i64* partial;
    i32* par[2];
    i64* ein[2];
    i32* start;
    unsigned long long* runmin;
};
static void signals_layout(Arena& a, i64 N, SignalsWs& W) {
    W.ctl = a.take<JumpCtl>(1);
    W.which = a.take<i32>(1);
    W.mt_buf = a.take<i32>(mintree_words(N));
    W.diff = a.take<unsigned long long>(N + 1);
    W.partial = a.take<i64>((N + SC_CHUNK - 1) / SC_CHUNK + 1);
    W.par[0] = a.take<i32>(N); W.par[1] = a.take<i32>(N);
    W.ein[0] = a.take<i64>(N); W.ein[1] = a.take<i64>(N);
    W.start = a.take<i32>(N);
    W.runmin = a.take<unsigned long long>(N);
}
// S > 0: room for the table's tags (peek_common.cuh), used when the workspace has it
i64 clpm_signals_ws_bytes(i64 N, i64 S) {
    Arena a(nullptr);
    SignalsWs W;
    signals_layout(a, N, W);
    if (S >= TAGS_MIN_S) a.take<unsigned char>(S);
    return a.used;
}

}  // namespace peek

using namespace peek;

extern "C" peek_status peek_clpm_signals(const uint64_t* hashes, const int64_t* blk_off, int64_t N,
                                         const int32_t* order, const int32_t* lcp, const int32_t* hit,
                                         int32_t tau, const int32_t* arrival, const peek_table* table,
                                         int32_t* section, int64_t* score, int64_t* evict_score,
                                         void* ws, int64_t ws_bytes, void* stream) {
    if (N < 0 || N >= 0x7fffffffLL) { set_error("peek_clpm_signals: N out of range"); return PEEK_ERR_INVALID_ARG; }
    if (evict_score && (!table || !table->t_keys || table->S < 2 || (table->S & (table->S - 1)))) {
        set_error("peek_clpm_signals: evict_score needs a table with S a power of two >= 2");
        return PEEK_ERR_INVALID_ARG;
    }
    if (section && N > 0 && !hit) { set_error("peek_clpm_signals: section needs hit"); return PEEK_ERR_INVALID_ARG; }
    cudaStream_t st = (cudaStream_t)stream;
    const bool work = N > 0 && (section || score || evict_score);
    if (work && (!blk_off || !order || !lcp || (evict_score && !hashes))) {
        set_error("peek_clpm_signals: NULL argument");
        return PEEK_ERR_INVALID_ARG;
    }
    if (work && (!ws || ((uintptr_t)ws & 255) || ws_bytes < clpm_signals_ws_bytes(N, 0))) {
        set_error("peek_clpm_signals: workspace NULL, misaligned or too small");
        return PEEK_ERR_WORKSPACE;
    }
    // every argument is checked: from here on work is enqueued
    if (evict_score) PEEK_CUDA(cudaMemsetAsync(evict_score, 0, sizeof(i64) * (size_t)table->S, st));
    if (!work) return PEEK_OK;
    Arena a(ws);
    SignalsWs W;
    signals_layout(a, N, W);
    unsigned char* tags = nullptr;  // big table: absent keys (most pending blocks) are answered by its tags
    if (evict_score && table->S >= TAGS_MIN_S && ((uintptr_t)table->t_keys & 15) == 0 &&
        ws_bytes >= clpm_signals_ws_bytes(N, table->S))
        tags = a.take<unsigned char>(table->S);
    a.arm(st);
    MinTree mt;
    mintree_layout(mt, lcp, N, W.mt_buf);
    Prof pr(PROF_SIGNALS, st, mintree_launches(mt) + (score ? 4 : 0) + (evict_score ? (tags ? 4 : 3) : 0) + (section ? 2 : 0));
    mintree_build(mt, st);
    unsigned grid = (unsigned)((N + SG_THREADS - 1) / SG_THREADS);
    if (grid > 148u * 16u) grid = 148u * 16u;
    const i64 nchunks = (N + SC_CHUNK - 1) / SC_CHUNK;
    if (score) {
        PEEK_CUDA(cudaMemsetAsync(W.diff, 0, sizeof(unsigned long long) * (size_t)(N + 1), st));
        k_score_steps<<<grid, SG_THREADS, 0, st>>>(blk_off, N, order, lcp, mt, W.diff);
        k_sum_partial<<<(unsigned)nchunks, SG_THREADS, 0, st>>>(W.diff, N, W.partial);
        k_sum_scan<<<1, 1024, 0, st>>>(W.partial, nchunks);
        k_sum_apply<<<(unsigned)nchunks, SG_THREADS, 0, st>>>(W.diff, N, W.partial, order, score);
    }
    if (evict_score) {
        k_evict_parent<<<grid, SG_THREADS, 0, st>>>(N, lcp, mt, W.par[0], W.ein[0]);
        PEEK_CUDA(cudaMemsetAsync(W.ctl, 0, sizeof(JumpCtl), st));
        int jgrid = persistent_ctas();
        i64 want = (N + 1023) / 1024;
        if (want < jgrid) jgrid = (int)(want < 1 ? 1 : want);
        i64 n = N;
        void* params[] = {&n, &W.par[0], &W.ein[0], &W.par[1], &W.ein[1], &W.ctl, &W.which};
        PEEK_CUDA(cudaLaunchCooperativeKernel((const void*)k_evict_jump, dim3(jgrid), dim3(1024), params, 0, st));
        int ppw = 32;
        while (ppw > 1 && N / ppw < 16384) ppw >>= 1;
        const i64 ewarps = (N + ppw - 1) / ppw;
        const unsigned wgrid = (unsigned)((ewarps * 32 + SG_THREADS - 1) / SG_THREADS);
        if (tags) k_table_tags<<<(unsigned)((table->S / 8 + 255) / 256), 256, 0, st>>>(table->t_keys, table->S, tags, nullptr);
        k_evict_write<<<wgrid, SG_THREADS, 0, st>>>(hashes, blk_off, N, order, lcp, mt, W.ein[0], W.ein[1], W.which,
                                                   table->t_keys, (u64)(table->S - 1), tags, evict_score, ppw);
    }
    if (section) {
        PEEK_CUDA(cudaMemsetAsync(W.runmin, 0xff, sizeof(unsigned long long) * (size_t)N, st));
        k_section_min<<<grid, SG_THREADS, 0, st>>>(blk_off, N, order, mt, hit, tau, arrival, W.start, W.runmin);
        k_section_write<<<grid, SG_THREADS, 0, st>>>(blk_off, N, order, hit, tau, arrival, W.start, W.runmin, section);
    }
    PEEK_CUDA(cudaGetLastError());
    return PEEK_OK;
}
