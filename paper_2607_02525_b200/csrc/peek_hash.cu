// peek_hash.cu — a1 peek_block_hash: chained per-block hashes (R1).
//
// Two steps:
//   nb_scan   blk_off = exclusive prefix sum of floor(len_r / B)                 (2 small launches; 3 beyond 2 M requests; 1 up to 8192)
//   fused     k_block_hash_fused: tokens -> per-block sums -> chained hashes in ONE pass over HBM
//             (1-D bulk TMA staging, thread-per-block sums, lane-per-request chain; see below)
#include <mutex>

#include "peek_common.cuh"

namespace peek {

static constexpr int B16 = 16;
__constant__ u64 c_M[16] = {pos_mult(0),  pos_mult(1),  pos_mult(2),  pos_mult(3),
                            pos_mult(4),  pos_mult(5),  pos_mult(6),  pos_mult(7),
                            pos_mult(8),  pos_mult(9),  pos_mult(10), pos_mult(11),
                            pos_mult(12), pos_mult(13), pos_mult(14), pos_mult(15)};
constexpr u64 sum_mult() {
    u64 s = 0;
    for (int j = 0; j < 16; ++j) s += pos_mult(j);
    return s;
}
static constexpr u64 SUM_M = sum_mult();

// ---- nb_scan ---------------------------------------------------------------------------
static constexpr int SCAN_THREADS = 256, SCAN_ITEMS = 8, SCAN_CHUNK = SCAN_THREADS * SCAN_ITEMS;

__global__ void __launch_bounds__(SCAN_THREADS) k_nb_partial(const i64* __restrict__ tok_off, i64 N,
                                                            i64* __restrict__ partial) {
    __shared__ i64 sm[34];
    i64 base = (i64)blockIdx.x * SCAN_CHUNK;
    i64 s = 0;
#pragma unroll
    for (int it = 0; it < SCAN_ITEMS; ++it) {
        i64 r = base + it * SCAN_THREADS + threadIdx.x;
        if (r < N) s += (tok_off[r + 1] - tok_off[r]) / B16;
    }
    i64 tot;
    block_exscan_i64(s, sm, &tot);
    if (threadIdx.x == 0) partial[blockIdx.x] = tot;
}

// single CTA: exclusive scan of partial[0..n) in place
__global__ void __launch_bounds__(1024) k_scan_partials(i64* __restrict__ partial, i64 n,
                                                        unsigned long long* __restrict__ counter) {
    __shared__ i64 sm[34];
    if (threadIdx.x == 0) *counter = 0;  // request queue head of k_block_hash_fused
    i64 carry = 0;
    for (i64 b = 0; b < n; b += 1024) {
        i64 i = b + threadIdx.x;
        i64 v = i < n ? partial[i] : 0;
        i64 tot;
        i64 ex = block_exscan_i64(v, sm, &tot);
        if (i < n) partial[i] = carry + ex;
        carry += tot;
    }
}

// small queues: the whole scan in one CTA, one launch (N <= SCAN_SMALL_MAX)
static constexpr int SCAN_SMALL_MAX = 8192;
__global__ void __launch_bounds__(1024) k_nb_scan_small(const i64* __restrict__ tok_off, i64 N,
                                                        i64* __restrict__ blk_off,
                                                        unsigned long long* __restrict__ counter) {
    __shared__ i64 sm[34];
    if (threadIdx.x == 0) { *counter = 0; blk_off[0] = 0; }
    i64 carry = 0;
    for (i64 b = 0; b < N; b += 1024) {
        const i64 r = b + threadIdx.x;
        const i64 v = r < N ? (tok_off[r + 1] - tok_off[r]) / B16 : 0;
        i64 tot;
        const i64 ex = block_exscan_i64(v, sm, &tot);
        if (r < N) blk_off[r + 1] = carry + ex + v;
        carry += tot;
    }
}

// PRESCANNED: partial[] holds exclusive prefixes (k_scan_partials ran); else it holds the chunks' own
// sums and every CTA adds up the chunks before its own itself (up to SCAN_DIRECT_MAX of them: one
// launch less), CTA 0 also resetting the request counter of k_block_hash_fused
static constexpr int SCAN_DIRECT_MAX = 1024;
template <bool PRESCANNED>
__global__ void __launch_bounds__(SCAN_THREADS) k_nb_apply(const i64* __restrict__ tok_off, i64 N,
                                                          const i64* __restrict__ partial,
                                                          i64* __restrict__ blk_off,
                                                          unsigned long long* __restrict__ counter) {
    __shared__ i64 sm[34];
    i64 base = 0;
    if (PRESCANNED) {
        base = partial[blockIdx.x];
    } else {
        if (blockIdx.x == 0 && threadIdx.x == 0) *counter = 0;
        i64 acc = 0;
        for (int c = threadIdx.x; c < (int)blockIdx.x; c += SCAN_THREADS) acc += partial[c];
        i64 tot0;
        block_exscan_i64(acc, sm, &tot0);
        base = tot0;
        __syncthreads();
    }
    // thread t owns SCAN_ITEMS consecutive requests so the scan is a plain blocked scan; the offsets
    // come in and the results go out through a shared-memory tile, so both global streams are coalesced
    __shared__ i64 tile[SCAN_CHUNK + 1];
    const i64 c0 = (i64)blockIdx.x * SCAN_CHUNK;
    for (int x = threadIdx.x; x <= SCAN_CHUNK; x += SCAN_THREADS) tile[x] = c0 + x <= N ? tok_off[c0 + x] : 0;
    __syncthreads();
    const int t0 = threadIdx.x * SCAN_ITEMS;
    i64 nb[SCAN_ITEMS];
    i64 s = 0;
#pragma unroll
    for (int it = 0; it < SCAN_ITEMS; ++it) {
        nb[it] = c0 + t0 + it < N ? (tile[t0 + it + 1] - tile[t0 + it]) / B16 : 0;
        s += nb[it];
    }
    i64 tot;
    i64 ex = block_exscan_i64(s, sm, &tot) + base;
    __syncthreads();  // every thread has read its offsets: the tile now takes the results
#pragma unroll
    for (int it = 0; it < SCAN_ITEMS; ++it) {
        ex += nb[it];
        tile[t0 + it] = ex;
    }
    __syncthreads();
    if (blockIdx.x == 0 && threadIdx.x == 0) blk_off[0] = 0;
    for (int x = threadIdx.x; x < SCAN_CHUNK; x += SCAN_THREADS)
        if (c0 + x < N) blk_off[c0 + x + 1] = tile[x];
}

// ---- fused content + chain ----------------------------------------------------------------
// One persistent kernel, HF_WARPS independent warps per CTA, one CTA per SM.  Lane l of a warp owns
// one request at a time (taken from a global counter) and carries its chain state k in a register.
// A round of a warp:
//   A  for every owning lane q: the next chunk of <= 32 blocks (<= 2 KB of tokens) of q's request is
//      staged in shared memory by ONE 1-D bulk TMA copy (cp.async.bulk + mbarrier, HF_STAGES deep
//      ring per warp), then lane j computes block j of the chunk on its own: 16 multiply-adds from
//      four conflict-free 128-bit shared loads, no cross-lane reduction; c = mix64(S) goes to the
//      warp's c-buffer in shared memory.  The loop is unrolled over the ring (stage addresses,
//      barriers and parities are static) and a chunk's mix64 runs one trip late, inside the next
//      chunk's multiply-adds, where its dependent chain costs no stalls
//   B  every owning lane runs the serial chain k = mix64(k ^ c) over ITS request's chunk (the chain
//      is inherently serial per request, so lanes = requests)
//   C  the chunk's k values are written to `hashes` with coalesced 256-byte stores
// so tokens are read from HBM once and only the final hashes are written: 4T + 8NB bytes.
// HF_LANES requests per warp: the c-buffer (HF_LANES x 32 values) and the ring share the warp's
// slice of shared memory, and 20 warps x 16 requests beat 15 x 32 (more copies in flight; the chain
// phase runs half empty, but phase A is 70 % of the instructions).
//
// Alignment: a request starts at an arbitrary token, so a chunk starts `a` = 0..3 words past a
// 16-byte boundary.  The copy fetches the 16-byte aligned superset; row j = staged bytes
// [64j, 64j+64).  Block j is words a..15 of row j plus words 0..a-1 of row j+1: lane j also loads
// the first vector of row j+1, which stands in for the first a words of its own row, and the
// multipliers are rotated by a (block_sum<a>).
// Bank conflicts: rows are 64 bytes apart, so lane j reads its four 16-byte vectors in the rotated
// order (c + (j>>1)) & 3 and keeps its multipliers pre-rotated the same way (M[c][e] below).
#ifndef PEEK_HF_WARPS
#define PEEK_HF_WARPS 20
#endif
#ifndef PEEK_HF_STAGES
#define PEEK_HF_STAGES 3
#endif
static constexpr int HF_WARPS = PEEK_HF_WARPS;
static constexpr int HF_THREADS = HF_WARPS * 32;
static constexpr int HF_STAGES = PEEK_HF_STAGES;
static constexpr int HF_STAGE_BYTES = 2176;          // 2048 + 16 rounded up to a multiple of 128
static constexpr int HF_CROW = 33;                   // c-buffer row pitch in u64 (32 + 1: no conflicts)
#ifndef PEEK_HF_LANES
#define PEEK_HF_LANES 16
#endif
static constexpr int HF_LANES = PEEK_HF_LANES;       // owning lanes (requests) per warp = c-buffer rows
static constexpr int HF_WARP_BYTES = HF_STAGES * HF_STAGE_BYTES + HF_LANES * HF_CROW * 8 + 64;
static constexpr int HF_SMEM_BYTES = HF_WARPS * HF_WARP_BYTES + 128;

__device__ __forceinline__ u32 smem_u32(const void* p) { return (u32)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(u32 bar, u32 count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(u32 bar, u32 bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void tma_load_1d(u32 dst, const void* src, u32 bytes, u32 bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(u32 bar, u32 parity) {
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra DONE;\n"
        "bra LAB_WAIT;\n"
        "DONE:\n"
        "}" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ uint4 lds128(u32 addr) {
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
    return v;
}

// Content sum (without SUM_M) of block `lane` of a staged chunk whose first token sits A words past a
// 16-byte boundary.  V[c] is physical vector (c + x) & 3 of row `lane`, M[c][e] = pos_mult(4 * ((c + x) & 3)
// + e).  The block is words A..15 of the row followed by words 0..A-1 of the NEXT row: X (vector 0 of
// row lane + 1) stands in for the first A words of this row's physical vector 0, which V[c0] holds.
// The previous chunk's mix64 rides in the same basic block so that its dependent chain fills the
// multiply-add latencies.
template <int A>
__device__ __forceinline__ u64 block_sum(const uint4 (&V)[4], u32 xaddr, const u64 (&M)[4][4], int c0,
                                         u64 Uprev, u64* cprev) {
    u32 xw[4] = {0, 0, 0, 0};
    if (A > 0) {
        const uint4 X = lds128(xaddr);
        xw[0] = X.x; xw[1] = X.y; xw[2] = X.z; xw[3] = X.w;
    }
    u64 acc0 = 0, acc1 = 0;
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        const u32 w[4] = {V[c].x, V[c].y, V[c].z, V[c].w};
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            u64 p;
            if (e >= A) p = (u64)w[e] * M[c][e - A];
            else p = (u64)(c == c0 ? xw[e] : w[e]) * M[(c + 3) & 3][4 + e - A];
            if (e & 1) acc1 += p;
            else acc0 += p;
        }
    }
    *cprev = mix64(Uprev + SUM_M);
    return acc0 + acc1;
}

struct HashArgs {
    const i32* tokens;
    const i64* tok_off;
    const i64* blk_off;
    i64 N;
    u64 seed;
    u64* hashes;
    i64 cap;
    unsigned long long* counter;  // next request to hand out (zeroed by k_scan_partials)
    int lanes_cap;                // owning lanes per warp (spreads few long requests over all warps)
};

__global__ void __launch_bounds__(HF_THREADS, 1) k_block_hash_fused(HashArgs A) {
    extern __shared__ __align__(128) unsigned char hf_smem[];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const unsigned FULL = 0xffffffffu;
    const unsigned lt = (1u << lane) - 1u;
    unsigned char* wbase = hf_smem + (size_t)wid * HF_WARP_BYTES;
    const u32 stage0 = smem_u32(wbase);
    u64* cbuf = (u64*)(wbase + HF_STAGES * HF_STAGE_BYTES);
    const u32 bar0 = smem_u32(wbase + HF_STAGES * HF_STAGE_BYTES + HF_LANES * HF_CROW * 8);
    if (lane == 0) {
#pragma unroll
        for (int s = 0; s < HF_STAGES; ++s) mbar_init(bar0 + 8 * s, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncwarp();

    const int x = (lane >> 1) & 3, c0 = (4 - x) & 3;
    u64 M[4][4];
#pragma unroll
    for (int c = 0; c < 4; ++c)
#pragma unroll
        for (int e = 0; e < 4; ++e) M[c][e] = pos_mult(4 * ((c + x) & 3) + e);
    u32 voff[4];
#pragma unroll
    for (int c = 0; c < 4; ++c) voff[c] = 64u * lane + 16u * ((c + x) & 3);

    const char* pool_end = (const char*)(A.tokens + A.tok_off[A.N]);
    const char* pool_end16 = (const char*)((uintptr_t)pool_end & ~(uintptr_t)15);

    // request owned by this lane
    bool own = false, exhausted = false;
    i32 pos = 0, nb = 0;
    const char* tptr = nullptr;  // first token of the request
    i64 obase = 0;
    u64 k = A.seed;
    // this lane's chunk of the round being staged: 16-byte aligned source, clipped copy size,
    // meta = n | a << 8 | (words past the last 16-byte boundary of the pool) << 16
    const char* c_src = nullptr;
    u32 c_bytes = 0, c_meta = 0;
    unsigned im = 0, cm = 0;  // lanes whose chunk is still to be issued / consumed
    u32 par[HF_STAGES];       // parity to wait for on each stage
#pragma unroll
    for (int s = 0; s < HF_STAGES; ++s) par[s] = 0;
    const u32 xoff = 64u * lane + 64u;

    // next chunk of `im` -> stage S (static): the owning lane issues its own copy
    auto issue = [&](const int S) {
        const int q = __ffs(im) - 1;
        im &= im - 1;
        if (lane == q) {
            const u32 bar = bar0 + 8 * S;
            mbar_expect_tx(bar, c_bytes);
            if (c_bytes) tma_load_1d(stage0 + S * HF_STAGE_BYTES, (const void*)c_src, c_bytes, bar);
            // the DRAM atom at the end of this chunk is also the first one of the request's next chunk,
            // which is copied a round later: ask L2 to keep it (read amplification 6.4 % -> 5 %)
            if (c_bytes >= 64) asm volatile("prefetch.global.L2::evict_last [%0];" ::"l"(c_src + c_bytes - 16));
        }
    };
    // Take requests for the lanes that have none, describe every owning lane's next chunk and put
    // the first HF_STAGES - 1 copies of the round in flight (every round starts at stage 0: all
    // stages are drained when phase A ends).  Returns false when nothing is left.
    auto next_round = [&]() -> bool {
        bool need = !own && lane < A.lanes_cap && !exhausted;
        for (;;) {
            const unsigned m = __ballot_sync(FULL, need);
            if (!m) break;
            unsigned long long base = 0;
            if (lane == 0) base = atomicAdd(A.counter, (unsigned long long)__popc(m));
            base = __shfl_sync(FULL, base, 0);
            if ((i64)base >= A.N) { exhausted = true; break; }
            if (need) {
                const i64 r = (i64)base + __popc(m & lt);
                if (r < A.N) {
                    const i64 b0 = A.blk_off[r], b1 = A.blk_off[r + 1];
                    if (b1 > b0) {
                        own = true; need = false;
                        pos = 0; nb = (i32)(b1 - b0); obase = b0;
                        tptr = (const char*)(A.tokens + A.tok_off[r]);
                    }
                } else {
                    need = false;
                }
            }
        }
        const unsigned active = __ballot_sync(FULL, own);
        if (!active) return false;
        c_meta = 0;
        if (own) {
            const u32 n = (u32)min(32, nb - pos);
            const uintptr_t ad = (uintptr_t)tptr + (size_t)pos * 64;
            const u32 a4 = (u32)(ad & 15);
            const char* need_end = (const char*)ad + 64 * n;
            c_src = (const char*)(ad - a4);
            c_bytes = 64u * n + (a4 ? 16u : 0u);
            u32 tail = 0;
            if (c_src + c_bytes > pool_end16) {  // the copy stops at the last 16-byte boundary of the pool
                c_bytes = (u32)(pool_end16 - c_src);
                if (need_end > pool_end16) tail = (u32)(need_end - pool_end16) >> 2;
            }
            c_meta = n | (a4 >> 2) << 8 | tail << 16;
        }
        im = cm = active;
#pragma unroll
        for (int s = 0; s < HF_STAGES - 1; ++s)
            if (im) issue(s);
        return true;
    };

    bool more = next_round();
    while (more) {
        // ---- phase A: one thread per block of each staged chunk; the loop is unrolled over the
        //      ring so that stage addresses, barriers and parities are static ----
        u64 Uprev = 0;
        u64* cprev = cbuf + 32;  // first trip: the pad slot of row 0
        while (cm) {
#pragma unroll
            for (int S = 0; S < HF_STAGES; ++S) {
                if (!cm) break;
                issue((S + HF_STAGES - 1) % HF_STAGES);  // no chunk left: no lane matches
                const int q = __ffs(cm) - 1;
                cm &= cm - 1;
                const u32 meta = __shfl_sync(FULL, c_meta, q);
                const int a = (meta >> 8) & 3;
                const u32 sbase = stage0 + S * HF_STAGE_BYTES;
                mbar_wait(bar0 + 8 * S, par[S]);
                par[S] ^= 1u;
                if (meta >> 16) {  // last words of the pool, past its last 16-byte boundary: by hand
                    const u32 src_lo = __shfl_sync(FULL, (u32)(uintptr_t)c_src, q);
                    if (lane < (int)(meta >> 16)) {
                        const u32 v = *(const u32*)(pool_end16 + 4 * lane);
                        asm volatile("st.shared.u32 [%0], %1;" ::"r"(sbase + ((u32)(uintptr_t)pool_end16 - src_lo) + 4u * lane), "r"(v) : "memory");
                    }
                    __syncwarp();
                }
                uint4 V[4];
#pragma unroll
                for (int c = 0; c < 4; ++c) V[c] = lds128(sbase + voff[c]);
                u64 U;
                switch (a) {
                    case 0: U = block_sum<0>(V, sbase + xoff, M, c0, Uprev, cprev); break;
                    case 1: U = block_sum<1>(V, sbase + xoff, M, c0, Uprev, cprev); break;
                    case 2: U = block_sum<2>(V, sbase + xoff, M, c0, Uprev, cprev); break;
                    default: U = block_sum<3>(V, sbase + xoff, M, c0, Uprev, cprev); break;
                }
                Uprev = U;
                cprev = cbuf + q * HF_CROW + lane;
                __syncwarp();  // the stage is fully read before it is refilled
            }
        }
        *cprev = mix64(Uprev + SUM_M);

        // ---- advance, and put the next round's first copies in flight before the chain ----
        const i32 nB = (i32)(c_meta & 0xff);  // this round: chain steps of this lane, output position
        const i64 outp = obase + pos;
        const unsigned done = __ballot_sync(FULL, own);
        bool fresh = false;
        if (own) {
            pos += nB;
            if (pos == nb) { own = false; fresh = true; }
        }
        more = next_round();
        __syncwarp();  // c-buffer rows visible

        // ---- phase B: serial chain, lane = request ----
        // steps every owner has run unguarded (lanes without a request chain row 0 and store nothing)
        const bool ownr = (done >> lane) & 1u;
        const i32 nmax = __reduce_max_sync(FULL, nB);
        const i32 nmin = __reduce_min_sync(FULL, ownr ? nB : 32);
        u64* crow = cbuf + (ownr ? lane : 0) * HF_CROW;
        i32 s = 0;
        for (; s < nmin; ++s) {
            k = mix64(k ^ crow[s]);
            if (k == PEEK_EMPTY) k = PEEK_EMPTY - 1;
            if (ownr) crow[s] = k;
        }
        for (; s < nmax; ++s) {
            if (s < nB) {
                k = mix64(k ^ crow[s]);
                if (k == PEEK_EMPTY) k = PEEK_EMPTY - 1;
                crow[s] = k;
            }
        }
        if (fresh || !ownr) k = A.seed;
        __syncwarp();

        // ---- phase C: coalesced stores of the round's hashes ----
        const i64 room = A.cap - outp;
        const i32 ncl = room < (i64)nB ? (room < 0 ? 0 : (i32)room) : nB;
        u64* const outq = A.hashes + outp;
        unsigned om = done;
        while (om) {
            const int q = __ffs(om) - 1;
            om &= om - 1;
            const i32 n = __shfl_sync(FULL, ncl, q);
            u64* o = (u64*)__shfl_sync(FULL, (unsigned long long)(uintptr_t)outq, q);
            if (lane < n) o[lane] = cbuf[q * HF_CROW + lane];
        }
        __syncwarp();
    }
}

i64 block_hash_ws_bytes(i64 N) {
    Arena a(nullptr);
    a.take<i64>((N + SCAN_CHUNK - 1) / SCAN_CHUNK + 1);
    a.take<unsigned long long>(1);
    return a.used;
}

}  // namespace peek

using namespace peek;

extern "C" peek_status peek_block_hash(const int32_t* tokens, const int64_t* tok_off, int64_t N,
                                       int32_t block_size, uint64_t seed, int64_t* blk_off,
                                       uint64_t* hashes, int64_t hashes_capacity, void* ws,
                                       int64_t ws_bytes, void* stream) {
    if (N < 0 || N >= 0x7fffffffLL) { set_error("peek_block_hash: N out of range"); return PEEK_ERR_INVALID_ARG; }
    if (block_size != B16) { set_error("peek_block_hash: block_size must be 16"); return PEEK_ERR_UNSUPPORTED; }
    if (N == 0) return PEEK_OK;
    if (!tok_off || !blk_off || hashes_capacity < 0 || (hashes_capacity > 0 && (!hashes || !tokens))) {
        set_error("peek_block_hash: NULL argument");
        return PEEK_ERR_INVALID_ARG;
    }
    if ((uintptr_t)tokens & 15) {
        set_error("peek_block_hash: tokens must be 16-byte aligned");
        return PEEK_ERR_INVALID_ARG;
    }
    if (!ws || ((uintptr_t)ws & 255) || ws_bytes < block_hash_ws_bytes(N)) {
        set_error("peek_block_hash: workspace NULL, misaligned or too small");
        return PEEK_ERR_WORKSPACE;
    }
    cudaStream_t st = (cudaStream_t)stream;
    Arena a(ws);
    i64 nchunks = (N + SCAN_CHUNK - 1) / SCAN_CHUNK;
    i64* partial = a.take<i64>(nchunks + 1);
    unsigned long long* counter = a.take<unsigned long long>(1);
    a.arm(st);
    if (N <= SCAN_SMALL_MAX) {
        Prof pr(PROF_HASH_SCAN, st, 1);
        k_nb_scan_small<<<1, 1024, 0, st>>>(tok_off, N, blk_off, counter);
    } else {
        const bool direct = nchunks <= SCAN_DIRECT_MAX;
        Prof pr(PROF_HASH_SCAN, st, direct ? 2 : 3);
        k_nb_partial<<<(unsigned)nchunks, SCAN_THREADS, 0, st>>>(tok_off, N, partial);
        if (direct) {
            k_nb_apply<false><<<(unsigned)nchunks, SCAN_THREADS, 0, st>>>(tok_off, N, partial, blk_off, counter);
        } else {
            k_scan_partials<<<1, 1024, 0, st>>>(partial, nchunks, counter);
            k_nb_apply<true><<<(unsigned)nchunks, SCAN_THREADS, 0, st>>>(tok_off, N, partial, blk_off, counter);
        }
    }
    if (hashes_capacity > 0) {
        PEEK_CUDA(func_smem_optin((const void*)k_block_hash_fused, HF_SMEM_BYTES));
        int grid = sm_count();
        i64 warps = (i64)grid * HF_WARPS;
        if (N < warps) {  // fewer requests than warps: no point in idle CTAs
            grid = (int)((N + HF_WARPS - 1) / HF_WARPS);
            warps = (i64)grid * HF_WARPS;
        }
        i64 per_warp = (N + warps - 1) / warps;
        HashArgs A{tokens, tok_off, blk_off, N, seed, hashes, hashes_capacity, counter,
                   (int)(per_warp < 1 ? 1 : (per_warp > HF_LANES ? HF_LANES : per_warp))};
        Prof pr(PROF_HASH_CONTENT, st, 1);
        k_block_hash_fused<<<grid, HF_THREADS, HF_SMEM_BYTES, st>>>(A);
    }
    PEEK_CUDA(cudaGetLastError());
    return PEEK_OK;
}

// ---- peek_block_hash_static: the same call, its scratch in a file-scope device array -------------
// For callers that cannot allocate device memory (CUDA-graph capture, serving loops and harnesses
// that forbid cudaMalloc).  The scratch of peek_block_hash (the per-chunk partial sums of the block
// scan and the request counter of k_block_hash_fused) lives in g_hash_static_scratch: every GPU that
// loads the library holds these 32 KB until the process exits.  In host code the array's name is a
// host-side stand-in, not a device address, so the address the kernels get comes from
// cudaGetSymbolAddress, asked once per device with that device current.
static constexpr i64 HASH_STATIC_BYTES = 32 * 1024;
static __device__ __align__(256) unsigned char g_hash_static_scratch[HASH_STATIC_BYTES];

static peek_status hash_static_scratch(void** out) {
    static std::mutex mu;
    static void* known[64];  // by device ordinal; no host allocation either
    int dev = 0;
    PEEK_CUDA(cudaGetDevice(&dev));
    std::lock_guard<std::mutex> lock(mu);
    if (dev >= 0 && dev < 64 && known[dev]) {
        *out = known[dev];
        return PEEK_OK;
    }
    void* p = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&p, g_hash_static_scratch);
    if (e != cudaSuccess || !p) return cuda_fail(e, "cudaGetSymbolAddress(g_hash_static_scratch)");
    if (dev >= 0 && dev < 64) known[dev] = p;
    *out = p;
    return PEEK_OK;
}

extern "C" peek_status peek_block_hash_static(const int32_t* tokens, const int64_t* tok_off, int64_t N,
                                              int32_t block_size, uint64_t seed, int64_t* blk_off,
                                              uint64_t* hashes, int64_t hashes_capacity, void* stream) {
    // host-side checks first (they answer before any CUDA call), in the order of peek_block_hash
    if (N < 0) { set_error("peek_block_hash_static: N out of range"); return PEEK_ERR_INVALID_ARG; }
    if (N > PEEK_BLOCK_HASH_STATIC_MAX_N || block_hash_ws_bytes(N) > HASH_STATIC_BYTES) {
        set_error("peek_block_hash_static: N = %lld exceeds the static scratch (at most %lld requests); "
                  "use peek_block_hash with a caller-provided workspace",
                  (long long)N, (long long)PEEK_BLOCK_HASH_STATIC_MAX_N);
        return PEEK_ERR_CAPACITY;
    }
    if (block_size != B16) { set_error("peek_block_hash_static: block_size must be 16"); return PEEK_ERR_UNSUPPORTED; }
    if (N == 0) return PEEK_OK;
    if (!tok_off || !blk_off || hashes_capacity < 0 || (hashes_capacity > 0 && (!hashes || !tokens))) {
        set_error("peek_block_hash_static: NULL argument");
        return PEEK_ERR_INVALID_ARG;
    }
    if ((uintptr_t)tokens & 15) {
        set_error("peek_block_hash_static: tokens must be 16-byte aligned");
        return PEEK_ERR_INVALID_ARG;
    }
    void* scratch = nullptr;
    const peek_status s = hash_static_scratch(&scratch);
    if (s != PEEK_OK) return s;
    // Nothing in the scratch has to start at zero: the scan kernels write every partial sum they
    // later read and reset the request counter, so the previous call's contents are harmless.
    return peek_block_hash(tokens, tok_off, N, block_size, seed, blk_off, hashes, hashes_capacity, scratch,
                           HASH_STATIC_BYTES, stream);
}
