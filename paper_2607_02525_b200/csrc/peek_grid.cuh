// peek_grid.cuh — building blocks of the persistent (cooperative, one launch) kernels: CTA scans,
// grid-wide scans over CTA-owned chunks, a CUB-free stable LSD radix sort of u32 indices by a
// gathered digit, and the min-hierarchy used for nearest-smaller-value searches on the LCP array.
// Every routine that contains a grid_barrier must be called by ALL threads of ALL CTAs.
#pragma once
#include "peek_common.cuh"

namespace peek {

static constexpr int PK_THREADS = 512;  // CTA size of the persistent kernels
static constexpr int PK_WARPS = PK_THREADS / 32;

struct Grid {
    u32* bar;   // zero-initialised barrier word
    u32 epoch;  // running target, identical in every thread
    __device__ __forceinline__ void sync() { grid_barrier(bar, epoch); }
};

// ---- CTA scan of one value per thread (commutative or not: order is thread order) ------------
template <typename T, typename Op>
__device__ __forceinline__ T warp_inscan(T v, Op op, int lane) {
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        T t = __shfl_up_sync(0xffffffffu, v, o);
        if (lane >= o) v = op(t, v);
    }
    return v;
}

// inclusive scan; smem >= PK_WARPS + 1 elements of T; *total = reduction of the whole CTA
template <typename T, typename Op>
__device__ __forceinline__ T block_inscan(T v, Op op, T ident, T* smem, T* total) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
    T inc = warp_inscan(v, op, lane);
    if (lane == 31) smem[w] = inc;
    __syncthreads();
    if (w == 0) {
        T s = lane < nw ? smem[lane] : ident;
        T si = warp_inscan(s, op, lane);
        T ex = __shfl_up_sync(0xffffffffu, si, 1);
        if (lane == 0) ex = ident;
        if (lane < nw) smem[lane] = ex;
        if (lane == 31) smem[nw] = si;
    }
    __syncthreads();
    T r = op(smem[w], inc);
    *total = smem[nw];
    __syncthreads();
    return r;
}

// ---- grid-wide inclusive scan (commutative, associative op) ----------------------------------
// CTA c owns the contiguous chunk [c*chunk, (c+1)*chunk).  load(i) -> T, store(i, inclusive).
// agg: gridDim.x elements of T in global memory.  Two grid barriers.
template <typename T, typename Op, typename Load, typename Store>
__device__ void grid_inscan(i64 n, Load load, Store store, Op op, T ident, T* agg, T* smem, Grid& g) {
    const i64 chunk = (((n + gridDim.x - 1) / gridDim.x) + blockDim.x - 1) / blockDim.x * blockDim.x;
    const i64 c0 = min((i64)blockIdx.x * chunk, n), c1 = min(c0 + chunk, n);
    T acc = ident;
    for (i64 i = c0 + threadIdx.x; i < c1; i += blockDim.x) acc = op(acc, load(i));
    T tot;
    block_inscan(acc, op, ident, smem, &tot);
    if (threadIdx.x == 0) agg[blockIdx.x] = tot;
    g.sync();
    acc = ident;
    for (int c = threadIdx.x; c < (int)blockIdx.x; c += blockDim.x) acc = op(acc, agg[c]);
    T carry;
    block_inscan(acc, op, ident, smem, &carry);
    for (i64 b = c0; b < c1; b += blockDim.x) {
        i64 i = b + threadIdx.x;
        T v = i < c1 ? load(i) : ident;
        T tt;
        T inc = block_inscan(v, op, ident, smem, &tt);
        if (i < c1) store(i, op(carry, inc));
        carry = op(carry, tt);
    }
    g.sync();
}

// ---- stable LSD radix sort pass over u32 indices, 8-bit digit gathered through `digit(idx)` ---
static constexpr int SORT_KPT = 4;
static constexpr int SORT_TILE = PK_THREADS * SORT_KPT;

struct SortSmem {
    u32 wcnt[PK_WARPS][256];
    u32 base[256];
    u32 scan[PK_WARPS + 1];
};

struct SortScratch {
    u32* tile_hist;    // 256 * ceil(n / SORT_TILE), digit-major
    u32* digit_total;  // 256
};

__host__ __device__ inline i64 sort_tiles(i64 n) { return (n + SORT_TILE - 1) / SORT_TILE; }

// Returns true if dst now holds the pass result, false if the digit was constant (pass skipped,
// src still current).  The decision is grid-uniform.  Three grid barriers (two when skipped).
template <typename DigitFn>
__device__ bool radix_pass(const u32* src, u32* dst, i64 n, DigitFn digit, SortScratch sc, SortSmem& sm,
                           Grid& g) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const i64 NT = sort_tiles(n);
    // H: per-tile digit histograms
    for (i64 t = blockIdx.x; t < NT; t += gridDim.x) {
        if (threadIdx.x < 256) sm.base[threadIdx.x] = 0;
        __syncthreads();
#pragma unroll
        for (int k = 0; k < SORT_KPT; ++k) {
            i64 i = t * SORT_TILE + (i64)w * (32 * SORT_KPT) + k * 32 + lane;
            if (i < n) atomicAdd(&sm.base[digit(src[i])], 1u);
        }
        __syncthreads();
        if (threadIdx.x < 256) sc.tile_hist[(i64)threadIdx.x * NT + t] = sm.base[threadIdx.x];
        __syncthreads();
    }
    g.sync();
    // S: exclusive scan over tiles, one warp per digit
    {
        const i64 gw = (i64)blockIdx.x * PK_WARPS + w, nw = (i64)gridDim.x * PK_WARPS;
        for (i64 d = gw; d < 256; d += nw) {
            u32 carry = 0;
            u32* row = sc.tile_hist + d * NT;
            for (i64 b = 0; b < NT; b += 32) {
                i64 i = b + lane;
                u32 v = i < NT ? row[i] : 0;
                u32 inc = warp_inscan(v, [](u32 a, u32 b2) { return a + b2; }, lane);
                if (i < NT) row[i] = carry + inc - v;
                carry += __shfl_sync(0xffffffffu, inc, 31);
            }
            if (lane == 0) sc.digit_total[d] = carry;
        }
    }
    g.sync();
    // C: scatter
    u32 tot = threadIdx.x < 256 ? sc.digit_total[threadIdx.x] : 0;
    int constant = __syncthreads_or(tot == (u32)n);
    if (constant) return false;
    {
        u32 all;
        u32 inc = block_inscan(tot, [](u32 a, u32 b2) { return a + b2; }, 0u, sm.scan, &all);
        if (threadIdx.x < 256) sm.base[threadIdx.x] = inc - tot;
        __syncthreads();
    }
    const unsigned lt = (1u << lane) - 1u;
    for (i64 t = blockIdx.x; t < NT; t += gridDim.x) {
        for (int d = threadIdx.x; d < PK_WARPS * 256; d += PK_THREADS) (&sm.wcnt[0][0])[d] = 0;
        __syncthreads();
        u32 idx[SORT_KPT], dg[SORT_KPT], pre[SORT_KPT];
#pragma unroll
        for (int k = 0; k < SORT_KPT; ++k) {
            i64 i = t * SORT_TILE + (i64)w * (32 * SORT_KPT) + k * 32 + lane;
            bool valid = i < n;
            idx[k] = valid ? src[i] : 0;
            dg[k] = valid ? (u32)digit(idx[k]) : (0x100u | lane);
            unsigned peers = __match_any_sync(0xffffffffu, dg[k]);
            u32 old = valid ? sm.wcnt[w][dg[k]] : 0;
            pre[k] = old + __popc(peers & lt);
            __syncwarp();
            if (valid && (peers & lt) == 0) sm.wcnt[w][dg[k]] = old + __popc(peers);
            __syncwarp();
        }
        __syncthreads();
        if (threadIdx.x < 256) {
            u32 run = 0;
#pragma unroll
            for (int ww = 0; ww < PK_WARPS; ++ww) {
                u32 c = sm.wcnt[ww][threadIdx.x];
                sm.wcnt[ww][threadIdx.x] = run;
                run += c;
            }
        }
        __syncthreads();
#pragma unroll
        for (int k = 0; k < SORT_KPT; ++k) {
            i64 i = t * SORT_TILE + (i64)w * (32 * SORT_KPT) + k * 32 + lane;
            if (i < n) {
                u32 d = dg[k];
                u32 pos = sm.base[d] + sc.tile_hist[(i64)d * NT + t] + sm.wcnt[w][d] + pre[k];
                dst[pos] = idx[k];
            }
        }
        __syncthreads();
    }
    g.sync();
    return true;
}

// ---- min hierarchy over L0x[0..N] (L0x[i] = lcp[i] for i < N, L0x[N] = 0) --------------------
// level k (k >= 1) has n_k = ceil(n_{k-1} / 32) entries, each the min of 32 entries below.
static constexpr int NSV_MAX_LEVELS = 8;
struct MinTree {
    const i32* lcp;  // level 0 (N entries, virtual N-th = 0)
    i64 N;
    i32* lvl[NSV_MAX_LEVELS];  // lvl[k] for k >= 1
    i64 n[NSV_MAX_LEVELS];     // n[0] = N + 1
    int levels;                // number of levels including level 0
    __device__ __forceinline__ i32 val(int k, i64 i) const {
        if (k == 0) return i < N ? lcp[i] : 0;
        return lvl[k][i];
    }
};

__host__ __device__ inline i64 mintree_words(i64 N) {
    i64 n = N + 1, tot = 0;
    while (n > 1) { n = (n + 31) / 32; tot += (n + 63) / 64 * 64; }
    return tot + 64;
}

__host__ __device__ inline void mintree_layout(MinTree& mt, const i32* lcp, i64 N, i32* buf) {
    mt.lcp = lcp;
    mt.N = N;
    mt.n[0] = N + 1;
    mt.lvl[0] = nullptr;
    int k = 0;
    i64 n = N + 1;
    while (n > 1 && k + 1 < NSV_MAX_LEVELS) {
        n = (n + 31) / 32;
        ++k;
        mt.lvl[k] = buf;
        mt.n[k] = n;
        buf += (n + 63) / 64 * 64;
    }
    mt.levels = k + 1;
}

// build level k from level k-1 (grid-stride over global warps; one warp per output entry)
__device__ __forceinline__ void mintree_build_level(const MinTree& mt, int k, i64 gwarp, i64 nwarps, int lane) {
    for (i64 c = gwarp; c < mt.n[k]; c += nwarps) {
        i64 i = c * 32 + lane;
        i32 v = i < mt.n[k - 1] ? mt.val(k - 1, i) : 0x7fffffff;
        v = __reduce_min_sync(0xffffffffu, v);
        if (lane == 0) mt.lvl[k][c] = v;
    }
}

// stand-alone build of all levels (one small launch per level) for the non-persistent kernels;
// static: every translation unit that includes this header gets its own copy
static __global__ void __launch_bounds__(256) k_mintree_level(MinTree mt, int k) {
    i64 gw = ((i64)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    i64 nw = ((i64)gridDim.x * blockDim.x) >> 5;
    mintree_build_level(mt, k, gw, nw, threadIdx.x & 31);
}
// small inputs: every level in one launch of one CTA (a CTA barrier between levels)
static __global__ void __launch_bounds__(1024) k_mintree_all(MinTree mt) {
    for (int k = 1; k < mt.levels; ++k) {
        mintree_build_level(mt, k, (i64)(threadIdx.x >> 5), (i64)(blockDim.x >> 5), threadIdx.x & 31);
        __syncthreads();
    }
}
// big inputs: level 1 by the whole grid, then every further level (<= 1/1024 of the input) by one CTA
static __global__ void __launch_bounds__(1024) k_mintree_from(MinTree mt, int k0) {
    for (int k = k0; k < mt.levels; ++k) {
        mintree_build_level(mt, k, (i64)(threadIdx.x >> 5), (i64)(blockDim.x >> 5), threadIdx.x & 31);
        __syncthreads();
    }
}
static constexpr i64 MINTREE_TAIL_MAX = 32768;  // entries of level 2 that one CTA still builds (N <= 2^25)
static inline int mintree_launches(const MinTree& mt) {
    if (mt.levels <= 1) return 0;
    if (mt.n[1] <= 1024) return 1;
    if (mt.levels > 2 && mt.n[2] <= MINTREE_TAIL_MAX) return 2;
    return mt.levels - 1;
}
static inline void mintree_build(const MinTree& mt, cudaStream_t st) {
    if (mt.levels > 1 && mt.n[1] <= 1024) {  // N <= 32768
        k_mintree_all<<<1, 1024, 0, st>>>(mt);
        return;
    }
    const bool tail = mt.levels > 2 && mt.n[2] <= MINTREE_TAIL_MAX;
    for (int k = 1; k < (tail ? 2 : mt.levels); ++k) {
        i64 warps = mt.n[k];
        unsigned grid = (unsigned)((warps * 32 + 255) / 256);
        if (grid > 148u * 8u) grid = 148u * 8u;
        k_mintree_level<<<grid, 256, 0, st>>>(mt, k);
    }
    if (tail) k_mintree_from<<<1, 1024, 0, st>>>(mt, 2);
}

// largest p <= j with L0x[p] < cd   (requires one to exist, e.g. L0x[0] = 0 < cd)
__device__ __forceinline__ i64 nsv_prev_less(const MinTree& mt, i64 j, i32 cd) {
    int k = 0;
    i64 i = j;
    for (;;) {
        for (;;) {
            if (mt.val(k, i) < cd) {
                if (k == 0) return i;
                --k;
                i = min(i * 32 + 31, mt.n[k] - 1);
                continue;
            }
            if ((i & 31) == 0) break;
            --i;
        }
        i = (i >> 5) - 1;
        ++k;
    }
}

// smallest t >= t0 with L0x[t] < cd   (exists: L0x[N] = 0 < cd for cd >= 1)
__device__ __forceinline__ i64 nsv_next_less(const MinTree& mt, i64 t0, i32 cd) {
    int k = 0;
    i64 i = t0;
    for (;;) {
        for (;;) {
            if (mt.val(k, i) < cd) {
                if (k == 0) return i;
                --k;
                i = i * 32;
                continue;
            }
            if ((i & 31) == 31 || i == mt.n[k] - 1) break;
            ++i;
        }
        i = (i >> 5) + 1;
        ++k;
    }
}

}  // namespace peek
