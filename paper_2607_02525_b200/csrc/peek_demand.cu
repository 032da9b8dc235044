// peek_demand.cu — a7/a8 peek_demand_rank.
//
// Demand (PAPER.md:281 inverted index block_hash -> demand; pending_count of Eq. 2):
// the sorted order + adjacent LCP ARE the pending trie, so each distinct pending block is visited
// once (at the sorted position where it first appears, i >= lcp[j]) and its pending_count is the
// width of the run of positions that share it, found with a next-smaller-value search on the LCP
// array.  One table probe per DISTINCT block instead of one per (request, block) pair.
//
// cLPM order (sub-key of Eq. 1): stable LSD radix sort of request indices by
// (-hit, -cluster_size, arrival), digits gathered from the three arrays; constant digits skipped.
#include "peek_grid.cuh"

namespace peek {

// ---- demand -----------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_mintree_level(MinTree mt, int k) {
    i64 gw = ((i64)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    i64 nw = ((i64)gridDim.x * blockDim.x) >> 5;
    mintree_build_level(mt, k, gw, nw, threadIdx.x & 31);
}

__device__ __forceinline__ i64 table_slot(const u64* __restrict__ t_keys, u64 mask, u64 key) {
    u64 p = key & mask;
    for (;;) {
        u64 tk = __ldg(t_keys + p);
        if (tk == key) return (i64)p;
        if (tk == PEEK_EMPTY) return -1;
        p = (p + 1) & mask;
    }
}

__device__ __forceinline__ void demand_range(const u64* __restrict__ chain, i64 i_lo, i64 i_hi, i32 count,
                                             const u64* __restrict__ t_keys, u64 mask, i32* demand,
                                             int lane) {
    for (i64 i = i_lo + lane; i <= i_hi; i += 32) {
        i64 p = table_slot(t_keys, mask, __ldg(chain + i));
        if (p >= 0) atomicAdd(demand + p, count);
    }
}

__global__ void __launch_bounds__(256) k_demand(const u64* __restrict__ hashes, const i64* __restrict__ blk_off,
                                               i64 N, const i32* __restrict__ order,
                                               const i32* __restrict__ lcp, MinTree mt,
                                               const u64* __restrict__ t_keys, u64 mask,
                                               i32* __restrict__ demand) {
    const int lane = threadIdx.x & 31;
    i64 j = ((i64)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    if (j >= N) return;
    i64 r = order[j];
    i64 b0 = blk_off[r], nb = blk_off[r + 1] - b0;
    i64 l0 = lcp[j], l1 = j + 1 < N ? lcp[j + 1] : 0;
    const u64* chain = hashes + b0;
    // blocks [l0, l1) are shared with later positions: runs of equal pending_count
    i64 i_hi = l1 - 1, t = j + 1;
    while (i_hi >= l0) {
        t = nsv_next_less(mt, t, (i32)(i_hi + 1));  // first later position sharing <= i_hi blocks
        i64 lt = mt.val(0, t);
        i64 i_lo = lt > l0 ? lt : l0;
        demand_range(chain, i_lo, i_hi, (i32)(t - j), t_keys, mask, demand, lane);
        i_hi = i_lo - 1;
    }
    // blocks only this request has
    demand_range(chain, l0 > l1 ? l0 : l1, nb - 1, 1, t_keys, mask, demand, lane);
}

// ---- cLPM order ---------------------------------------------------------------------------
struct RankCtl { u32 bar; u32 pad[3]; };

struct RankArgs {
    const i32 *hit, *csize, *arrival;
    i64 N;
    i32* out;
    RankCtl* ctl;
    u32* ord2;
    u32* tile_hist;
    u32* digit_total;
};

__global__ void __launch_bounds__(PK_THREADS) k_clpm_sort(RankArgs A) {
    __shared__ SortSmem ssm;
    const i64 N = A.N;
    const i64 gtid = (i64)blockIdx.x * PK_THREADS + threadIdx.x, gsize = (i64)gridDim.x * PK_THREADS;
    Grid g{&A.ctl->bar, 0};
    u32* cur = (u32*)A.out;
    u32* nxt = A.ord2;
    for (i64 r = gtid; r < N; r += gsize) cur[r] = (u32)r;
    g.sync();
    SortScratch sc{A.tile_hist, A.digit_total};
    const i32* hit = A.hit;
    const i32* cs = A.csize;
    const i32* arr = A.arrival;
    for (int p = 0; p < 12; ++p) {
        const int sh = 8 * (p & 3);
        bool moved;
        if (p < 4) {  // arrival ascending (signed: flip the sign bit); NULL => the index itself
            moved = radix_pass(cur, nxt, N, [=](u32 idx) {
                u32 v = arr ? ((u32)__ldg(arr + idx) ^ 0x80000000u) : idx;
                return (v >> sh) & 255u;
            }, sc, ssm, g);
        } else if (p < 8) {  // cluster size descending
            moved = radix_pass(cur, nxt, N, [=](u32 idx) {
                u32 v = ~(u32)__ldg(cs + idx);
                return (v >> sh) & 255u;
            }, sc, ssm, g);
        } else {  // hit descending
            moved = radix_pass(cur, nxt, N, [=](u32 idx) {
                u32 v = ~(u32)__ldg(hit + idx);
                return (v >> sh) & 255u;
            }, sc, ssm, g);
        }
        if (moved) { u32* t = cur; cur = nxt; nxt = t; }
    }
    if (cur != (u32*)A.out) {
        for (i64 r = gtid; r < N; r += gsize) A.out[r] = (i32)cur[r];
    }
}

static void rank_layout(Arena& a, i64 N, RankArgs& A) {
    A.ctl = a.take<RankCtl>(1);
    A.ord2 = a.take<u32>(N);
    A.tile_hist = a.take<u32>(256 * sort_tiles(N));
    A.digit_total = a.take<u32>(256);
}

i64 demand_rank_ws_bytes(i64 N, i64 S) {
    (void)S;
    Arena a(nullptr);
    RankArgs A;
    rank_layout(a, N, A);
    a.take<i32>(mintree_words(N));
    return a.used;
}

int persistent_grid(const void* kernel);

}  // namespace peek

using namespace peek;

extern "C" peek_status peek_demand_rank(const uint64_t* hashes, const int64_t* blk_off, int64_t N,
                                        const int32_t* order, const int32_t* lcp, const peek_table* table,
                                        const int32_t* hit, const int32_t* cluster_size,
                                        const int32_t* arrival, int32_t* demand, int32_t* clpm_order,
                                        void* ws, int64_t ws_bytes, void* stream) {
    if (N < 0 || N >= 0x7fffffffLL) { set_error("peek_demand_rank: N out of range"); return PEEK_ERR_INVALID_ARG; }
    if (demand && (!table || !table->t_keys || table->S < 2 || (table->S & (table->S - 1)))) {
        set_error("peek_demand_rank: demand needs a table with S a power of two >= 2");
        return PEEK_ERR_INVALID_ARG;
    }
    if (demand && N > 0 && (!hashes || !blk_off || !order || !lcp)) {
        set_error("peek_demand_rank: demand needs hashes, blk_off, order and lcp");
        return PEEK_ERR_INVALID_ARG;
    }
    if (clpm_order && N > 0 && (!hit || !cluster_size)) {
        set_error("peek_demand_rank: clpm_order needs hit and cluster_size");
        return PEEK_ERR_INVALID_ARG;
    }
    cudaStream_t st = (cudaStream_t)stream;
    if (demand) PEEK_CUDA(cudaMemsetAsync(demand, 0, sizeof(i32) * (size_t)table->S, st));
    if (N == 0 || (!demand && !clpm_order)) return PEEK_OK;
    if (!ws || ((uintptr_t)ws & 255) || ws_bytes < demand_rank_ws_bytes(N, table ? table->S : 0)) {
        set_error("peek_demand_rank: workspace NULL, misaligned or too small");
        return PEEK_ERR_WORKSPACE;
    }
    Arena a(ws);
    RankArgs A;
    rank_layout(a, N, A);
    i32* mt_buf = a.take<i32>(mintree_words(N));
    if (demand) {
        MinTree mt;
        mintree_layout(mt, lcp, N, mt_buf);
        Prof pr(PROF_DEMAND, st, mt.levels);
        for (int k = 1; k < mt.levels; ++k) {
            i64 warps = mt.n[k];
            unsigned grid = (unsigned)((warps * 32 + 255) / 256);
            if (grid > 148u * 8u) grid = 148u * 8u;
            k_mintree_level<<<grid, 256, 0, st>>>(mt, k);
        }
        unsigned grid = (unsigned)((N * 32 + 255) / 256);
        k_demand<<<grid, 256, 0, st>>>(hashes, blk_off, N, order, lcp, mt, table->t_keys,
                                      (u64)(table->S - 1), demand);
    }
    if (clpm_order) {
        A.hit = hit; A.csize = cluster_size; A.arrival = arrival; A.N = N; A.out = clpm_order;
        int grid = persistent_grid((const void*)k_clpm_sort);
        i64 want = (N + PK_THREADS - 1) / PK_THREADS;
        if (want < grid) grid = (int)(want < 1 ? 1 : want);
        PEEK_CUDA(cudaMemsetAsync(A.ctl, 0, sizeof(RankCtl), st));
        void* params[] = {&A};
        Prof pr(PROF_RANK, st, 1);
        PEEK_CUDA(cudaLaunchCooperativeKernel((const void*)k_clpm_sort, dim3(grid), dim3(PK_THREADS), params, 0, st));
    }
    PEEK_CUDA(cudaGetLastError());
    return PEEK_OK;
}
