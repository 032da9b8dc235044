// peek_sort.cuh — CUB-free stable LSD radix sort of (u64 key, u32 value) pairs for the persistent
// cooperative kernels (one CTA of GS_THREADS per SM, all co-resident).
//
// CTA c owns the contiguous chunk [c*C, (c+1)*C) of the current buffer for the whole pass.  A pass:
//   1  load the chunk (registers), rank every element among the equal digits of the chunk
//      (warp match + per-warp digit counters in shared memory), publish the chunk's digit histogram
//   -- grid barrier --
//   2  base[d] = (elements with a smaller digit anywhere) + (elements with digit d in earlier chunks)
//   3  scatter key and value to base[d] + rank
//   -- grid barrier --
// so a pass reads and writes every pair once and costs two grid barriers.  When N fits one tile per
// CTA (N <= gridDim * GS_TILE, e.g. 1.2 M pairs on 148 SMs) the keys never leave the registers
// between steps 1 and 3; larger inputs loop over tiles and reload.  Digits are 8 bits wide and are
// taken only where `vary` (the OR of key ^ key' over all pairs, or any superset) has bits set:
// constant bit ranges cost nothing.
#pragma once
#include <type_traits>

#include "peek_grid.cuh"

namespace peek {

#ifndef PEEK_GS_THREADS
#define PEEK_GS_THREADS 1024
#endif
#ifndef PEEK_GS_KPT
#define PEEK_GS_KPT 8
#endif
static constexpr int GS_THREADS = PEEK_GS_THREADS;
static constexpr int GS_WARPS = GS_THREADS / 32;
static constexpr int GS_KPT = PEEK_GS_KPT;
static constexpr int GS_TILE = GS_THREADS * GS_KPT;

struct GsSmem {
    unsigned short wcnt[GS_WARPS][256];  // per-warp digit counts, then exclusive prefix over warps
    u32 base[256];                       // where this CTA's next element with digit d goes
    u32 tot[256];                        // digit counts of the tile / chunk
    u32 dstart[256];                     // exclusive prefix of the tile's digit counts
    u32 scan[GS_WARPS + 2];
};

// dynamic shared memory of a kernel that sorts: one tile of pairs, staged in digit order so that
// the scatter writes runs of consecutive addresses (full sectors instead of one sector per pair)
static constexpr int GS_STAGE_BYTES = GS_TILE * (int)(sizeof(u64) + sizeof(u32));
struct GsStage {
    u64* key;
    u32* val;
};
__device__ __forceinline__ GsStage gs_stage(void* dyn_smem) {
    return GsStage{(u64*)dyn_smem, (u32*)((char*)dyn_smem + (size_t)GS_TILE * sizeof(u64))};
}

struct GsBufs {
    u64* key[2];
    u32* val[2];
    u32* hist;  // gs_hist_words(gridDim.x) words; the accumulator part must be zero on entry
};

// lanes of the warp whose 8-bit digit equals this lane's (ballot per bit: cheaper than MATCH.ANY
// on near-distinct digits); a lane with dg >= 256 (padding) must not take part in any group
__device__ __forceinline__ unsigned gs_peers(u32 dg) {
    unsigned m = __ballot_sync(0xffffffffu, dg < 256u);
#pragma unroll
    for (int bit = 0; bit < 8; ++bit) {
        const bool one = (dg >> bit) & 1u;
        const unsigned bal = __ballot_sync(0xffffffffu, one);
        m &= one ? bal : ~bal;
    }
    return m;
}

// rank the tile's elements: meta[k] = digit | (elements with the same digit earlier in this warp's
// rows) << 16; afterwards sm.wcnt[w][d] = elements with digit d in warps < w, sm.tot[d] = tile count
template <int K>
__device__ __forceinline__ void gs_rank_tile(u32 (&meta)[K], GsSmem& sm) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const unsigned lt = (1u << lane) - 1u;
    for (int d = threadIdx.x; d < GS_WARPS * 256 / 2; d += GS_THREADS) ((u32*)&sm.wcnt[0][0])[d] = 0;
    unsigned peers[K];
    unsigned live = 0;  // rows of this warp that hold any pair (small inputs fill only the first)
#pragma unroll
    for (int k = 0; k < K; ++k) {
        peers[k] = 0;
        if (__any_sync(0xffffffffu, meta[k] < 256u)) { peers[k] = gs_peers(meta[k]); live |= 1u << k; }
    }
    __syncthreads();
    PEEK_MARK(110);
#pragma unroll
    for (int k = 0; k < K; ++k) {
        if (!((live >> k) & 1u)) continue;  // warp-uniform
        const u32 dg = meta[k];
        const bool valid = dg < 256u;
        const u32 old = valid ? sm.wcnt[w][dg] : 0;
        meta[k] = dg | ((old + __popc(peers[k] & lt)) << 16);
        __syncwarp();
        if (valid && (peers[k] & lt) == 0) sm.wcnt[w][dg] = (unsigned short)(old + __popc(peers[k]));
        __syncwarp();
    }
    __syncthreads();
    PEEK_MARK(111);
    if (threadIdx.x < 256) {
        u32 run = 0;
        for (int w0 = 0; w0 < GS_WARPS; w0 += 8) {
            u32 c[8];
#pragma unroll
            for (int ww = 0; ww < 8; ++ww) c[ww] = sm.wcnt[w0 + ww][threadIdx.x];
#pragma unroll
            for (int ww = 0; ww < 8; ++ww) {
                sm.wcnt[w0 + ww][threadIdx.x] = (unsigned short)run;
                run += c[ww];
            }
        }
        sm.tot[threadIdx.x] = run;
    }
    __syncthreads();
    PEEK_MARK(112);
    {
        const u32 t = threadIdx.x < 256 ? sm.tot[threadIdx.x] : 0;
        u32 all;
        const u32 inc = block_inscan(t, [](u32 a, u32 b) { return a + b; }, 0u, sm.scan, &all);
        if (threadIdx.x < 256) sm.dstart[threadIdx.x] = inc - t;
        __syncthreads();
    }
}

// ---- digit bases without an all-to-all read ------------------------------------------------------
// Every CTA needs, per digit, the elements with a smaller digit anywhere plus those with the same
// digit in earlier chunks.  Reading all G histograms in all G CTAs is G*G KB of L2 traffic on the
// same lines (measured 8 us per pass at G = 148).  Instead a CTA publishes its histogram row AND adds
// it (fire-and-forget reductions) to the digit totals and to the row of its group of GS_GROUP
// chunks; after the barrier it reads the totals, the rows of the groups before its own and the rows
// of the chunks before it inside its group: <= 1 + G/GS_GROUP + GS_GROUP rows instead of G.
// The accumulators come in two sets (passes alternate); the set a pass does not use is zeroed
// during that pass, and both must be zero when a sort starts (host memset, and restored on exit).
static constexpr int GS_GROUP = 16;
__host__ __device__ inline i64 gs_hist_words(int grid) {
    return 256 * ((i64)grid + 2 * ((grid + GS_GROUP - 1) / GS_GROUP + 1));
}
struct GsHist {
    u32* rows;    // [G][256] per-chunk histograms
    u32* acc[2];  // [1 + NG][256]: row 0 digit totals, row 1 + g the sum over group g
    int ng;
};
__device__ __forceinline__ GsHist gs_hist(u32* hist) {
    const int G = gridDim.x, ng = (G + GS_GROUP - 1) / GS_GROUP;
    GsHist h;
    h.rows = hist;
    h.acc[0] = hist + (size_t)256 * G;
    h.acc[1] = h.acc[0] + (size_t)256 * (ng + 1);
    h.ng = ng;
    return h;
}

// before the barrier: publish sm.tot (this chunk's digit counts); `set` = pass parity
__device__ __forceinline__ void gs_publish(const GsHist& h, int set, const GsSmem& sm) {
    if (threadIdx.x < 256) {
        const u32 v = sm.tot[threadIdx.x];
        h.rows[(size_t)blockIdx.x * 256 + threadIdx.x] = v;
        if (v) {
            atomicAdd(h.acc[set] + threadIdx.x, v);
            atomicAdd(h.acc[set] + (size_t)256 * (1 + blockIdx.x / GS_GROUP) + threadIdx.x, v);
        }
    }
}

// after the barrier: sm.base[d]; also zeroes the other accumulator set for the next pass
__device__ __forceinline__ void gs_bases(const GsHist& h, int set, GsSmem& sm) {
    const int me = blockIdx.x, grp = me / GS_GROUP, d = threadIdx.x & 255, part = threadIdx.x >> 8;
    constexpr int PARTS = GS_THREADS / 256;  // thread groups that split the rows between them
    // rows to add up for "same digit, earlier chunks": groups < grp, then chunks grp*GS_GROUP .. me-1
    const int nrows = grp + (me - grp * GS_GROUP);
    u32 below = 0;
    for (int r0 = part; r0 < nrows; r0 += PARTS * 8) {
        u32 v[8];
#pragma unroll
        for (int x = 0; x < 8; ++x) {
            const int r = r0 + x * PARTS;
            const u32* row = r < grp ? h.acc[set] + (size_t)256 * (1 + r)
                                     : h.rows + (size_t)256 * (grp * GS_GROUP + (r - grp));
            v[x] = r < nrows ? __ldcg(row + d) : 0u;
        }
#pragma unroll
        for (int x = 0; x < 8; ++x) below += v[x];
    }
    const u32 total = part == 0 ? __ldcg(h.acc[set] + d) : 0u;
    if (PARTS > 1) {
        if (part == 0) sm.base[d] = 0;
        __syncthreads();
        if (below) atomicAdd(&sm.base[d], below);
        __syncthreads();
        below = part == 0 ? sm.base[d] : 0u;
    }
    u32 all;
    const u32 inc = block_inscan(total, [](u32 a, u32 b) { return a + b; }, 0u, sm.scan, &all);
    if (part == 0) sm.base[d] = below + inc - total;
    // the other set was last read before the previous pass's closing barrier
    const int words = 256 * (h.ng + 1);
    for (int i = blockIdx.x * GS_THREADS + threadIdx.x; i < words; i += gridDim.x * GS_THREADS) h.acc[set ^ 1][i] = 0;
    __syncthreads();
}

struct GsNoGen {};  // tag: pass 0 reads buffer 0

// Stable sort of n (key, value) pairs.  With a generator `gen(i, key&, val&)` the pairs of pass 0
// are produced on the fly (position i of the input order) instead of being read from buffer 0, and
// pass 0 writes buffer 0; without one the input is buffer 0.  Returns the buffer (0 or 1) that
// holds the result; with a generator and vary == 0 the pairs are materialised into buffer 0.
// Must be called by all threads of all CTAs of a cooperative launch with blockDim.x == GS_THREADS.
template <typename Gen>
__device__ __forceinline__ int grid_sort_pairs_gen(const GsBufs& b, i64 n, u64 vary, Grid& g, GsSmem& sm,
                                                   GsStage stg, Gen gen, int start_buf = 0) {
    constexpr bool HAS_GEN = !std::is_same<Gen, GsNoGen>::value;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const i64 C = (n + gridDim.x - 1) / gridDim.x;
    const i64 c0 = min((i64)blockIdx.x * C, n), c1 = min(c0 + C, n);
    const int ntiles = (int)((C + GS_TILE - 1) / GS_TILE);
    int cur = HAS_GEN ? -1 : start_buf;  // -1: the generator is the source
    if (gridDim.x == 1 && n <= GS_THREADS) {
        // Small inputs (one CTA, one pair per thread): no passes at all - every pair counts the
        // pairs that sort before it (smaller key, or equal key and earlier position) against the
        // keys held in shared memory, and is written straight to that rank.  Queues of the size
        // the paper runs (60-200 requests) take this path.
        if (!HAS_GEN && vary == 0) return start_buf;
        const int dstb = cur < 0 ? 0 : cur ^ 1;
        const int t = threadIdx.x;
        u64 key = ~0ull;
        u32 val = 0;
        if (t < n) {
            if constexpr (HAS_GEN) gen((i64)t, key, val);
            else { key = __ldcg(b.key[cur] + t); val = __ldcg(b.val[cur] + t); }
        }
        stg.key[t] = key;
        __syncthreads();
        u32 rank = 0;
        const int nn = (int)n;
#pragma unroll 4
        for (int j = 0; j < nn; ++j) {
            const u64 kj = stg.key[j];
            rank += (kj < key || (kj == key && j < t)) ? 1u : 0u;
        }
        if (t < n) { b.key[dstb][rank] = key; b.val[dstb][rank] = val; }
        __syncthreads();
        return dstb;
    }
    const GsHist gh = gs_hist(b.hist);
    int pass = 0;
    if (HAS_GEN && vary == 0) vary = 1;  // one (trivial) pass materialises the pairs
    while (vary) {
        const int sh = __ffsll((long long)vary) - 1;
        vary &= ~(0xffull << sh);
        const int dstb = cur < 0 ? 0 : cur ^ 1;
        const u64* __restrict__ ks = b.key[cur < 0 ? 0 : cur];
        const u32* __restrict__ vs = b.val[cur < 0 ? 0 : cur];
        u64* __restrict__ kd = b.key[dstb];
        u32* __restrict__ vd = b.val[dstb];
        u64 key[GS_KPT];
        u32 val[GS_KPT], meta[GS_KPT];
        auto load_tile = [&](int t) {
#pragma unroll
            for (int k = 0; k < GS_KPT; ++k) {
                const i64 i = c0 + (i64)t * GS_TILE + w * (32 * GS_KPT) + k * 32 + lane;
                const bool valid = i < c1;
                key[k] = 0;
                val[k] = 0;
                if (valid) {
                    if constexpr (HAS_GEN) {
                        if (cur < 0) gen(i, key[k], val[k]);
                        else { key[k] = __ldcg(ks + i); val[k] = __ldcg(vs + i); }
                    } else {
                        key[k] = __ldcg(ks + i);
                        val[k] = __ldcg(vs + i);
                    }
                }
                meta[k] = valid ? (u32)(key[k] >> sh) & 255u : (0x100u | lane);
            }
        };
        if (ntiles == 1) {
            load_tile(0);
            PEEK_MARK(100);
            gs_rank_tile<GS_KPT>(meta, sm);
        } else {
            if (threadIdx.x < 256) sm.tot[threadIdx.x] = 0;
            __syncthreads();
            for (int t = 0; t < ntiles; ++t) {
                load_tile(t);
#pragma unroll
                for (int k = 0; k < GS_KPT; ++k)
                    if (meta[k] < 256u) atomicAdd(&sm.tot[meta[k]], 1u);
            }
            __syncthreads();
        }
        gs_publish(gh, pass & 1, sm);
        PEEK_MARK(101);
        g.sync();
        PEEK_MARK(102);
        gs_bases(gh, pass & 1, sm);
        PEEK_MARK(103);
        for (int t = 0; t < ntiles; ++t) {
            if (ntiles > 1) {
                load_tile(t);
                gs_rank_tile<GS_KPT>(meta, sm);
            }
#pragma unroll
            for (int k = 0; k < GS_KPT; ++k) {  // stage the tile in digit order
                const i64 i = c0 + (i64)t * GS_TILE + w * (32 * GS_KPT) + k * 32 + lane;
                if (i < c1) {
                    const u32 d = meta[k] & 0xffffu;
                    const u32 lp = sm.dstart[d] + sm.wcnt[w][d] + (meta[k] >> 16);
                    stg.key[lp] = key[k];
                    stg.val[lp] = val[k];
                }
            }
            __syncthreads();
            {
                const i64 tbase = c0 + (i64)t * GS_TILE;
                const int tcount = (int)min((i64)GS_TILE, c1 - tbase);
#pragma unroll
                for (int k = 0; k < GS_KPT; ++k) {  // runs of equal digits go to consecutive addresses
                    const int q = k * GS_THREADS + threadIdx.x;
                    if (q < tcount) {
                        const u64 kk = stg.key[q];
                        const u32 d = (u32)(kk >> sh) & 255u;
                        const u32 pos = sm.base[d] + ((u32)q - sm.dstart[d]);
                        kd[pos] = kk;
                        vd[pos] = stg.val[q];
                    }
                }
            }
            __syncthreads();  // the stage is reused by the next tile / pass
            if (ntiles > 1) {
                if (threadIdx.x < 256) sm.base[threadIdx.x] += sm.tot[threadIdx.x];
                __syncthreads();
            }
        }
        PEEK_MARK(104);
        g.sync();
        PEEK_MARK(105);
        cur = dstb;
        ++pass;
    }
    // leave both accumulator sets zero: the last pass's set is dirty, nobody reads it any more
    if (pass > 0) {
        const int words = 256 * (gh.ng + 1);
        for (int i = blockIdx.x * GS_THREADS + threadIdx.x; i < words; i += gridDim.x * GS_THREADS)
            gh.acc[(pass - 1) & 1][i] = 0;
    }
    return cur < 0 ? 0 : cur;
}

// input in buffer `start_buf`
__device__ __forceinline__ int grid_sort_pairs(const GsBufs& b, i64 n, u64 vary, Grid& g, GsSmem& sm,
                                               GsStage stg, int start_buf = 0) {
    return grid_sort_pairs_gen(b, n, vary, g, sm, stg, GsNoGen{}, start_buf);
}

// OR-accumulate (x ^ ref) of a grid-stride loop into a 64-bit device word: call once per thread
__device__ __forceinline__ void gs_vary_accumulate(u64 diff, unsigned long long* vary) {
    const u32 lo = __reduce_or_sync(0xffffffffu, (u32)diff);
    const u32 hi = __reduce_or_sync(0xffffffffu, (u32)(diff >> 32));
    if ((threadIdx.x & 31) == 0 && (lo | hi)) atomicOr(vary, ((unsigned long long)hi << 32) | lo);
}

}  // namespace peek
