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
#include "peek_grid.cuh"

namespace peek {

static constexpr int GS_THREADS = 1024;
static constexpr int GS_WARPS = GS_THREADS / 32;
static constexpr int GS_KPT = 8;
static constexpr int GS_TILE = GS_THREADS * GS_KPT;

struct GsSmem {
    unsigned short wcnt[GS_WARPS][256];  // per-warp digit counts, then exclusive prefix over warps
    u32 base[256];                       // where this CTA's next element with digit d goes
    u32 tot[256];                        // digit counts of the tile / chunk
    u32 scan[GS_WARPS + 2];
};

struct GsBufs {
    u64* key[2];
    u32* val[2];
    u32* hist;  // 256 * gridDim.x, digit-major
};

// rank the tile's elements: pre[k] = elements with the same digit earlier in this warp's rows;
// afterwards sm.wcnt[w][d] = elements with digit d in warps < w, sm.tot[d] = tile count of d
template <int K>
__device__ __forceinline__ void gs_rank_tile(const u32 (&dg)[K], u32 (&pre)[K], GsSmem& sm) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const unsigned lt = (1u << lane) - 1u;
    for (int d = threadIdx.x; d < GS_WARPS * 256 / 2; d += GS_THREADS) ((u32*)&sm.wcnt[0][0])[d] = 0;
    __syncthreads();
#pragma unroll
    for (int k = 0; k < K; ++k) {
        const bool valid = dg[k] < 256u;
        const unsigned peers = __match_any_sync(0xffffffffu, dg[k]);
        const u32 old = valid ? sm.wcnt[w][dg[k]] : 0;
        pre[k] = old + __popc(peers & lt);
        __syncwarp();
        if (valid && (peers & lt) == 0) sm.wcnt[w][dg[k]] = (unsigned short)(old + __popc(peers));
        __syncwarp();
    }
    __syncthreads();
    if (threadIdx.x < 256) {
        u32 run = 0;
#pragma unroll 8
        for (int ww = 0; ww < GS_WARPS; ++ww) {
            const u32 c = sm.wcnt[ww][threadIdx.x];
            sm.wcnt[ww][threadIdx.x] = (unsigned short)run;
            run += c;
        }
        sm.tot[threadIdx.x] = run;
    }
    __syncthreads();
}

// sm.base[d] from the published histograms, digit-major hist[d * G + c] (call after the grid
// barrier): warp w sums digits 8w .. 8w+7 over the G chunks with coalesced loads
__device__ __forceinline__ void gs_bases(const u32* __restrict__ hist, GsSmem& sm) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int G = gridDim.x, me = blockIdx.x;
    constexpr int DPW = 256 / GS_WARPS;
    u32 tot[DPW], bel[DPW];
#pragma unroll
    for (int q = 0; q < DPW; ++q) {
        const u32* row = hist + (size_t)(w * DPW + q) * G;
        u32 t = 0, bl = 0;
        for (int c = lane; c < G; c += 32) {
            const u32 v = __ldcg(row + c);
            t += v;
            if (c < me) bl += v;
        }
        tot[q] = t;
        bel[q] = bl;
    }
#pragma unroll
    for (int q = 0; q < DPW; ++q) {
        tot[q] = __reduce_add_sync(0xffffffffu, tot[q]);
        bel[q] = __reduce_add_sync(0xffffffffu, bel[q]);
    }
    if (lane == 0) {
#pragma unroll
        for (int q = 0; q < DPW; ++q) { sm.tot[w * DPW + q] = tot[q]; sm.base[w * DPW + q] = bel[q]; }
    }
    __syncthreads();
    const u32 total = threadIdx.x < 256 ? sm.tot[threadIdx.x] : 0;
    u32 all;
    const u32 inc = block_inscan(total, [](u32 a, u32 b) { return a + b; }, 0u, sm.scan, &all);
    if (threadIdx.x < 256) sm.base[threadIdx.x] += inc - total;
    __syncthreads();
}

// Sorts n pairs held in buffer 0 of `b`; returns the buffer (0 or 1) that holds the result.
// Must be called by all threads of all CTAs of a cooperative launch with blockDim.x == GS_THREADS.
__device__ inline int grid_sort_pairs(const GsBufs& b, i64 n, u64 vary, Grid& g, GsSmem& sm) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const i64 C = (n + gridDim.x - 1) / gridDim.x;
    const i64 c0 = min((i64)blockIdx.x * C, n), c1 = min(c0 + C, n);
    const int ntiles = (int)((C + GS_TILE - 1) / GS_TILE);
    int cur = 0;
    while (vary) {
        const int sh = __ffsll((long long)vary) - 1;
        vary &= ~(0xffull << sh);
        const u64* __restrict__ ks = b.key[cur];
        const u32* __restrict__ vs = b.val[cur];
        u64* __restrict__ kd = b.key[cur ^ 1];
        u32* __restrict__ vd = b.val[cur ^ 1];
        u64 key[GS_KPT];
        u32 dg[GS_KPT], pre[GS_KPT];
        auto load_tile = [&](int t) {
#pragma unroll
            for (int k = 0; k < GS_KPT; ++k) {
                const i64 i = c0 + (i64)t * GS_TILE + w * (32 * GS_KPT) + k * 32 + lane;
                const bool valid = i < c1;
                key[k] = valid ? __ldcg(ks + i) : 0;
                dg[k] = valid ? (u32)(key[k] >> sh) & 255u : (0x100u | lane);
            }
        };
        if (ntiles == 1) {
            load_tile(0);
            gs_rank_tile<GS_KPT>(dg, pre, sm);
            if (threadIdx.x < 256) b.hist[(size_t)threadIdx.x * gridDim.x + blockIdx.x] = sm.tot[threadIdx.x];
        } else {
            if (threadIdx.x < 256) sm.tot[threadIdx.x] = 0;
            __syncthreads();
            for (int t = 0; t < ntiles; ++t) {
                load_tile(t);
#pragma unroll
                for (int k = 0; k < GS_KPT; ++k)
                    if (dg[k] < 256u) atomicAdd(&sm.tot[dg[k]], 1u);
            }
            __syncthreads();
            if (threadIdx.x < 256) b.hist[(size_t)threadIdx.x * gridDim.x + blockIdx.x] = sm.tot[threadIdx.x];
        }
        PEEK_MARK(101);
        g.sync();
        PEEK_MARK(102);
        gs_bases(b.hist, sm);
        PEEK_MARK(103);
        for (int t = 0; t < ntiles; ++t) {
            if (ntiles > 1) {
                load_tile(t);
                gs_rank_tile<GS_KPT>(dg, pre, sm);
            }
#pragma unroll
            for (int k = 0; k < GS_KPT; ++k) {
                const i64 i = c0 + (i64)t * GS_TILE + w * (32 * GS_KPT) + k * 32 + lane;
                if (i < c1) {
                    const u32 d = dg[k];
                    const u32 pos = sm.base[d] + sm.wcnt[w][d] + pre[k];
                    kd[pos] = key[k];
                    vd[pos] = __ldcg(vs + i);
                }
            }
            if (ntiles > 1) {
                __syncthreads();
                if (threadIdx.x < 256) sm.base[threadIdx.x] += sm.tot[threadIdx.x];
                __syncthreads();
            }
        }
        PEEK_MARK(104);
        g.sync();
        PEEK_MARK(105);
        cur ^= 1;
    }
    return cur;
}

// OR-accumulate (x ^ ref) of a grid-stride loop into a 64-bit device word: call once per thread
__device__ __forceinline__ void gs_vary_accumulate(u64 diff, unsigned long long* vary) {
    const u32 lo = __reduce_or_sync(0xffffffffu, (u32)diff);
    const u32 hi = __reduce_or_sync(0xffffffffu, (u32)(diff >> 32));
    if ((threadIdx.x & 31) == 0 && (lo | hi)) atomicOr(vary, ((unsigned long long)hi << 32) | lo);
}

}  // namespace peek
