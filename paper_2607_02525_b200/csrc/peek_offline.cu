// peek_offline.cu — a12 peek_offline_phase1: PEEK-offline's prefix-trie DFS
// reordering and its three guards (R25).
//
// The trie over the first D = 128 tokens (8 blocks) is never built.  A chained hash names a trie
// node, so one open-addressed table over the (request, level < 8) hashes gives every node its
// subtree count (atomicAdd) and the smallest request index below it (atomicMin).  "Children in
// descending subtree count, ties by the smallest request below, terminators first" is then a
// lexicographic order of the per-level keys
//     key_i(r) = 0 if r has no block i, else 1 + ((N - count(node_i(r))) << b | minidx(node_i(r)))
// and comes out of one stable pair sort per level, deepest level first (LSD over the levels), on
// the sort engine of peek_sort.cuh; a level whose keys are all equal costs no pass.
// Guards: duplication from a second table over whole chains (the last hash and the length name a
// chain, R15), coverage and sharing depth from the node counts.
#include "peek_sort.cuh"

namespace peek {

static constexpr int OF_THREADS = 256;
static constexpr int OF_MAX_DEPTH = 16;

struct OffCtl {
    u32 bar, pad;
    unsigned long long dup, cov, depth_blocks_sum;
    unsigned long long kor[OF_MAX_DEPTH], kand[OF_MAX_DEPTH];
};

struct OffArgs {
    const u64* hashes;
    const i64* blk_off;
    i64 N;
    int D;
    i32* order;
    double* guards;
    OffCtl* ctl;
    GsBufs bufs;
    unsigned long long* nkeys;  // node table: H slots, all-ones = empty
    u32* ncount;                // H
    u32* nmin;                  // H
    u32* slot;                  // N * D: node slot of (request, level), ~0 = absent
    unsigned long long* ckeys;  // chain table: HC slots
    u64 hmask, cmask;
};

__device__ __forceinline__ u64 of_insert(unsigned long long* keys, u64 mask, unsigned long long key, bool* fresh) {
    u64 h = mix64(key) & mask;
    for (;;) {
        const unsigned long long prev = atomicCAS(keys + h, ~0ull, key);
        if (prev == ~0ull) { *fresh = true; return h; }
        if (prev == key) { *fresh = false; return h; }
        h = (h + 1) & mask;
    }
}

// one thread per (request, level): node counts and smallest index; one per request: distinct chains
__global__ void __launch_bounds__(OF_THREADS) k_offline_insert(OffArgs A) {
    const i64 total = A.N * A.D;
    for (i64 x = (i64)blockIdx.x * OF_THREADS + threadIdx.x; x < total; x += (i64)gridDim.x * OF_THREADS) {
        const i64 r = x / A.D;
        const int i = (int)(x - r * A.D);
        const i64 b0 = A.blk_off[r], nb = A.blk_off[r + 1] - b0;
        u32 s = 0xffffffffu;
        if (i < nb) {
            bool fresh;
            const u64 h = of_insert(A.nkeys, A.hmask, (unsigned long long)A.hashes[b0 + i], &fresh);
            atomicAdd(A.ncount + h, 1u);
            atomicMin(A.nmin + h, (u32)r);
            s = (u32)h;
        }
        A.slot[x] = s;
        if (i == 0) {  // whole-chain identity: (last hash, length) names the chain (R15)
            const unsigned long long ck = nb ? mix64(A.hashes[b0 + nb - 1] ^ mix64((u64)nb)) : 0x1234567ull;
            bool fresh;
            of_insert(A.ckeys, A.cmask, ck == ~0ull ? ck - 1 : ck, &fresh);
            if (!fresh) atomicAdd(&A.ctl->dup, 1ull);
        }
    }
}

// coverage and sharing depth per request
__global__ void __launch_bounds__(OF_THREADS) k_offline_guards(OffArgs A) {
    u32 cov = 0, dsum = 0;
    for (i64 r = (i64)blockIdx.x * OF_THREADS + threadIdx.x; r < A.N; r += (i64)gridDim.x * OF_THREADS) {
        int d = 0;
        for (; d < A.D; ++d) {
            const u32 s = A.slot[r * A.D + d];
            if (s == 0xffffffffu || A.ncount[s] < 2u) break;
        }
        dsum += (u32)d;
        if (A.D >= 2) {
            const u32 s1 = A.slot[r * A.D + 1];
            if (s1 != 0xffffffffu && A.ncount[s1] >= 2u) ++cov;
        }
    }
    cov = __reduce_add_sync(0xffffffffu, cov);
    dsum = __reduce_add_sync(0xffffffffu, dsum);
    if ((threadIdx.x & 31) == 0) {
        if (cov) atomicAdd(&A.ctl->cov, (unsigned long long)cov);
        if (dsum) atomicAdd(&A.ctl->depth_blocks_sum, (unsigned long long)dsum);
    }
}

__global__ void __launch_bounds__(GS_THREADS, 1) k_offline_sort(OffArgs A) {
    extern __shared__ __align__(16) unsigned char dyn_smem[];
    __shared__ GsSmem ssm;
    const GsStage stg = gs_stage(dyn_smem);
    const i64 N = A.N;
    const i64 gtid = (i64)blockIdx.x * GS_THREADS + threadIdx.x, gsize = (i64)gridDim.x * GS_THREADS;
    Grid g{&A.ctl->bar, 0};
    const int nbits = bits_for((u64)(N > 1 ? N - 1 : 1));
    auto level_key = [&](u32 r, int lvl) -> u64 {
        const u32 s = __ldcg(A.slot + (i64)r * A.D + lvl);
        if (s == 0xffffffffu) return 0;
        return 1ull + (((u64)(N - (i64)__ldcg(A.ncount + s)) << nbits) | (u64)__ldcg(A.nmin + s));
    };
    if (gtid == 0) {  // the guards (all counters were final before this launch)
        const double n = (double)N;
        const double dup = (double)A.ctl->dup / n, cov = (double)A.ctl->cov / n;
        const double depth = 16.0 * (double)A.ctl->depth_blocks_sum / n;
        A.guards[0] = dup; A.guards[1] = cov; A.guards[2] = depth;
        A.guards[3] = (dup > 0.5 || cov < 0.1 || depth < 64.0) ? 1.0 : 0.0;
    }
    // identity order into buffer 0, then one stable sort per level, deepest first
    for (i64 j = gtid; j < N; j += gsize) A.bufs.val[0][j] = (u32)j;
    int src = 0;
    for (int lvl = A.D - 1; lvl >= 0; --lvl) {
        g.sync();
        u64 orv = 0, andv = ~0ull;
        for (i64 j = gtid; j < N; j += gsize) {
            const u64 k = level_key(__ldcg(A.bufs.val[src] + j), lvl);
            A.bufs.key[src][j] = k;
            orv |= k;
            andv &= k;
        }
        const u32 olo = __reduce_or_sync(0xffffffffu, (u32)orv), ohi = __reduce_or_sync(0xffffffffu, (u32)(orv >> 32));
        const u32 alo = __reduce_and_sync(0xffffffffu, (u32)andv), ahi = __reduce_and_sync(0xffffffffu, (u32)(andv >> 32));
        if ((threadIdx.x & 31) == 0) {
            atomicOr(&A.ctl->kor[lvl], ((unsigned long long)ohi << 32) | olo);
            atomicAnd(&A.ctl->kand[lvl], ((unsigned long long)ahi << 32) | alo);
        }
        g.sync();
        const u64 vary = __ldcg(&A.ctl->kor[lvl]) & ~__ldcg(&A.ctl->kand[lvl]);
        src = grid_sort_pairs(A.bufs, N, vary, g, ssm, stg, src);
    }
    g.sync();
    const u32* res = A.bufs.val[src];
    for (i64 j = gtid; j < N; j += gsize) A.order[j] = (i32)__ldcg(res + j);
}

static i64 pow2_at_least(i64 x) {
    i64 h = 64;
    while (h < x) h <<= 1;
    return h;
}
static void offline_layout(Arena& a, i64 N, int D, int grid, OffArgs& A) {
    A.ctl = a.take<OffCtl>(1);
    A.bufs.hist = a.take<u32>(gs_hist_words(grid));  // directly after ctl: one memset clears both
    A.bufs.key[0] = a.take<u64>(N);
    A.bufs.key[1] = a.take<u64>(N);
    A.bufs.val[0] = a.take<u32>(N);
    A.bufs.val[1] = a.take<u32>(N);
    const i64 H = pow2_at_least(2 * N * D), HC = pow2_at_least(2 * N);
    A.nkeys = a.take<unsigned long long>(H);
    A.nmin = a.take<u32>(H);                 // directly after nkeys: one 0xff memset covers both
    A.ckeys = a.take<unsigned long long>(HC);  // ... and this one
    A.ncount = a.take<u32>(H);
    A.slot = a.take<u32>(N * D);
    A.hmask = (u64)(H - 1);
    A.cmask = (u64)(HC - 1);
}
i64 offline_phase1_ws_bytes(i64 N) {
    Arena a(nullptr);
    OffArgs A;
    offline_layout(a, N, OF_MAX_DEPTH, 1024, A);
    return a.used;
}

}  // namespace peek

using namespace peek;

extern "C" peek_status peek_offline_phase1(const uint64_t* hashes, const int64_t* blk_off, int64_t N,
                                           int32_t depth_blocks, int32_t* order, double* guards, void* ws,
                                           int64_t ws_bytes, void* stream) {
    if (N < 0 || N >= 0x7fffffffLL) { set_error("peek_offline_phase1: N out of range"); return PEEK_ERR_INVALID_ARG; }
    if (depth_blocks < 1 || depth_blocks > OF_MAX_DEPTH) {
        set_error("peek_offline_phase1: depth_blocks must be 1..%d", OF_MAX_DEPTH);
        return PEEK_ERR_INVALID_ARG;
    }
    if (N == 0) return PEEK_OK;
    if (!hashes || !blk_off || !order || !guards) { set_error("peek_offline_phase1: NULL argument"); return PEEK_ERR_INVALID_ARG; }
    if (!ws || ((uintptr_t)ws & 255) || ws_bytes < offline_phase1_ws_bytes(N)) {
        set_error("peek_offline_phase1: workspace NULL, misaligned or too small");
        return PEEK_ERR_WORKSPACE;
    }
    cudaStream_t st = (cudaStream_t)stream;
    Arena a(ws);
    OffArgs A;
    offline_layout(a, N, depth_blocks, 1024, A);
    A.hashes = hashes; A.blk_off = blk_off; A.N = N; A.D = depth_blocks; A.order = order; A.guards = guards;
    PEEK_CUDA(cudaMemsetAsync(A.ctl, 0, (size_t)((char*)(A.bufs.hist + gs_hist_words(1024)) - (char*)A.ctl), st));
    PEEK_CUDA(cudaMemsetAsync(A.nkeys, 0xff, (size_t)((char*)(A.ckeys + (A.cmask + 1)) - (char*)A.nkeys), st));
    PEEK_CUDA(cudaMemsetAsync(A.ncount, 0, sizeof(u32) * (size_t)(A.hmask + 1), st));
    // kand starts as all ones
    PEEK_CUDA(cudaMemsetAsync(A.ctl->kand, 0xff, sizeof(A.ctl->kand), st));
    a.arm(st);
    Prof pr(PROF_OFFLINE, st, 3);
    i64 work = N * depth_blocks;
    unsigned grid = (unsigned)((work + OF_THREADS - 1) / OF_THREADS);
    if (grid > 148u * 32u) grid = 148u * 32u;
    k_offline_insert<<<grid, OF_THREADS, 0, st>>>(A);
    unsigned g2 = (unsigned)((N + OF_THREADS - 1) / OF_THREADS);
    if (g2 > 148u * 16u) g2 = 148u * 16u;
    k_offline_guards<<<g2, OF_THREADS, 0, st>>>(A);
    int cgrid = persistent_ctas();
    if (cgrid > 1024) cgrid = 1024;
    i64 want = (N + GS_THREADS - 1) / GS_THREADS;
    if (want < cgrid) cgrid = (int)(want < 1 ? 1 : want);
    PEEK_CUDA(func_smem_optin((const void*)k_offline_sort, GS_STAGE_BYTES));
    void* params[] = {&A};
    PEEK_CUDA(cudaLaunchCooperativeKernel((const void*)k_offline_sort, dim3(cgrid), dim3(GS_THREADS), params,
                                          GS_STAGE_BYTES, st));
    PEEK_CUDA(cudaGetLastError());
    return PEEK_OK;
}
