// peek_hash.cu — a1 peek_block_hash: chained per-block hashes (R1).
//
// Three steps, all HBM-streaming:
//   nb_scan      blk_off = exclusive prefix sum of floor(len_r / B)      (3 small launches)
//   content      S_i = sum_j (tok+1) * M_j for EVERY block, flattened over the global block
//                index so the token stream is read with coalesced 128-bit loads regardless of
//                request lengths; 4 lanes per 16-token block, 2-step shuffle reduce
//   chain        k_i = mix64(k_{i-1} ^ mix64(S_i)) in place, one thread per request (the chain is
//                inherently serial per request; both mixers run here so the streaming kernel
//                stays far below the integer-issue ceiling)
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
__global__ void __launch_bounds__(1024) k_scan_partials(i64* __restrict__ partial, i64 n) {
    __shared__ i64 sm[34];
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

__global__ void __launch_bounds__(SCAN_THREADS) k_nb_apply(const i64* __restrict__ tok_off, i64 N,
                                                          const i64* __restrict__ partial,
                                                          i64* __restrict__ blk_off) {
    __shared__ i64 sm[34];
    // thread t owns SCAN_ITEMS consecutive requests so the scan is a plain blocked scan
    i64 r0 = (i64)blockIdx.x * SCAN_CHUNK + (i64)threadIdx.x * SCAN_ITEMS;
    i64 nb[SCAN_ITEMS];
    i64 s = 0;
#pragma unroll
    for (int it = 0; it < SCAN_ITEMS; ++it) {
        i64 r = r0 + it;
        nb[it] = r < N ? (tok_off[r + 1] - tok_off[r]) / B16 : 0;
        s += nb[it];
    }
    i64 tot;
    i64 ex = block_exscan_i64(s, sm, &tot) + partial[blockIdx.x];
    if (blockIdx.x == 0 && threadIdx.x == 0) blk_off[0] = 0;
#pragma unroll
    for (int it = 0; it < SCAN_ITEMS; ++it) {
        i64 r = r0 + it;
        ex += nb[it];
        if (r < N) blk_off[r + 1] = ex;
    }
}

// ---- content ---------------------------------------------------------------------------
static constexpr int HB_THREADS = 256;
static constexpr int TILE_BLOCKS = 128;  // token blocks per warp tile (8 KB of tokens)
static constexpr int UNROLL = 4;         // warp steps (8 blocks each) in flight

// 4 tokens of this lane's quarter-block, from up to two 16-byte aligned vectors
__device__ __forceinline__ void pick4(const int4& v, const int4& n, int a, u32 t[4]) {
    if (a == 0) { t[0] = v.x; t[1] = v.y; t[2] = v.z; t[3] = v.w; }
    else if (a == 1) { t[0] = v.y; t[1] = v.z; t[2] = v.w; t[3] = n.x; }
    else if (a == 2) { t[0] = v.z; t[1] = v.w; t[2] = n.x; t[3] = n.y; }
    else { t[0] = v.w; t[1] = n.x; t[2] = n.y; t[3] = n.z; }
}

__global__ void __launch_bounds__(HB_THREADS) k_block_content(const i32* __restrict__ tokens,
                                                             const i64* __restrict__ tok_off,
                                                             const i64* __restrict__ blk_off, i64 N,
                                                             u64* __restrict__ hashes, i64 cap) {
    const int lane = threadIdx.x & 31;
    const int quad = lane >> 2, p = lane & 3;
    const i64 NB = blk_off[N];
    const i64 warp = ((i64)blockIdx.x * HB_THREADS + threadIdx.x) >> 5;
    i64 x = warp * TILE_BLOCKS;
    if (x >= NB) return;
    const i64 x_end = min(x + TILE_BLOCKS, NB);
    const u64 m0 = c_M[4 * p], m1 = c_M[4 * p + 1], m2 = c_M[4 * p + 2], m3 = c_M[4 * p + 3];

    // request holding global block x: largest r with blk_off[r] <= x (warp-uniform search)
    i64 lo = 0, hi = N;  // invariant blk_off[lo] <= x < blk_off[hi]
    while (hi - lo > 1) {
        i64 mid = (lo + hi) >> 1;
        if (blk_off[mid] <= x) lo = mid; else hi = mid;
    }
    i64 r = lo;
    while (x < x_end) {
        i64 rb = blk_off[r], re = blk_off[r + 1];
        while (re <= x) { ++r; rb = re; re = blk_off[r + 1]; }  // skip requests with no blocks left
        const i64 cnt = min(re, x_end) - x;                       // blocks of request r in this tile
        const i32* src = tokens + tok_off[r] + (x - rb) * B16;   // first token of block x
        const int a = (int)(((uintptr_t)src >> 2) & 3);          // misalignment in tokens
        const int4* vbase = (const int4*)(src - a);              // 16-byte aligned
        for (i64 s0 = 0; s0 < cnt; s0 += 8 * UNROLL) {
            int4 v[UNROLL], n[UNROLL];
#pragma unroll
            for (int u = 0; u < UNROLL; ++u) {
                i64 b = s0 + u * 8 + quad;  // block within the run
                bool act = b < cnt;
                v[u] = make_int4(0, 0, 0, 0);
                n[u] = make_int4(0, 0, 0, 0);
                if (act) v[u] = ld_stream_v4(vbase + b * 4 + p);
            }
            if (a != 0) {
#pragma unroll
                for (int u = 0; u < UNROLL; ++u) {
                    i64 b = s0 + u * 8 + quad;
                    bool act = b < cnt;
                    n[u].x = __shfl_down_sync(0xffffffffu, v[u].x, 1);
                    n[u].y = __shfl_down_sync(0xffffffffu, v[u].y, 1);
                    n[u].z = __shfl_down_sync(0xffffffffu, v[u].z, 1);
                    bool nxt_act = (s0 + u * 8 + ((lane + 1) >> 2)) < cnt;
                    if (act && (lane == 31 || !nxt_act)) {
                        int4 e = ld_stream_v4(vbase + b * 4 + p + 1);
                        n[u].x = e.x; n[u].y = e.y; n[u].z = e.z;
                    }
                }
            }
#pragma unroll
            for (int u = 0; u < UNROLL; ++u) {
                i64 b = s0 + u * 8 + quad;
                u32 t[4];
                pick4(v[u], n[u], a, t);
                u64 s = (u64)t[0] * m0 + (u64)t[1] * m1 + (u64)t[2] * m2 + (u64)t[3] * m3;
                s += __shfl_xor_sync(0xffffffffu, s, 1);
                s += __shfl_xor_sync(0xffffffffu, s, 2);
                if (p == 0 && b < cnt && x + b < cap) hashes[x + b] = s + SUM_M;
            }
        }
        x += cnt;
    }
}

// ---- chain -----------------------------------------------------------------------------
__global__ void __launch_bounds__(128) k_block_chain(const i64* __restrict__ blk_off, i64 N, u64 seed,
                                                    u64* __restrict__ hashes, i64 cap) {
    i64 r = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= N) return;
    i64 b = blk_off[r], e = min(blk_off[r + 1], cap);
    u64 k = seed;
    for (; b + 4 <= e; b += 4) {
        u64 s0 = hashes[b], s1 = hashes[b + 1], s2 = hashes[b + 2], s3 = hashes[b + 3];
        u64 c0 = mix64(s0), c1 = mix64(s1), c2 = mix64(s2), c3 = mix64(s3);
        k = mix64(k ^ c0); if (k == PEEK_EMPTY) k = PEEK_EMPTY - 1; hashes[b] = k;
        k = mix64(k ^ c1); if (k == PEEK_EMPTY) k = PEEK_EMPTY - 1; hashes[b + 1] = k;
        k = mix64(k ^ c2); if (k == PEEK_EMPTY) k = PEEK_EMPTY - 1; hashes[b + 2] = k;
        k = mix64(k ^ c3); if (k == PEEK_EMPTY) k = PEEK_EMPTY - 1; hashes[b + 3] = k;
    }
    for (; b < e; ++b) {
        k = mix64(k ^ mix64(hashes[b]));
        if (k == PEEK_EMPTY) k = PEEK_EMPTY - 1;
        hashes[b] = k;
    }
}

i64 block_hash_ws_bytes(i64 N) {
    Arena a(nullptr);
    a.take<i64>((N + SCAN_CHUNK - 1) / SCAN_CHUNK + 1);
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
    if (!ws || ((uintptr_t)ws & 255) || ws_bytes < block_hash_ws_bytes(N)) {
        set_error("peek_block_hash: workspace NULL, misaligned or too small");
        return PEEK_ERR_WORKSPACE;
    }
    cudaStream_t st = (cudaStream_t)stream;
    Arena a(ws);
    i64 nchunks = (N + SCAN_CHUNK - 1) / SCAN_CHUNK;
    i64* partial = a.take<i64>(nchunks + 1);
    {
        Prof pr(PROF_HASH_SCAN, st, 3);
        k_nb_partial<<<(unsigned)nchunks, SCAN_THREADS, 0, st>>>(tok_off, N, partial);
        k_scan_partials<<<1, 1024, 0, st>>>(partial, nchunks);
        k_nb_apply<<<(unsigned)nchunks, SCAN_THREADS, 0, st>>>(tok_off, N, partial, blk_off);
    }
    if (hashes_capacity > 0) {
        // NB is only known on the device; the grid is sized for the caller's capacity (>= NB).
        i64 warps = (hashes_capacity + TILE_BLOCKS - 1) / TILE_BLOCKS;
        i64 ctas = (warps * 32 + HB_THREADS - 1) / HB_THREADS;
        {
            Prof pr(PROF_HASH_CONTENT, st, 1);
            k_block_content<<<(unsigned)ctas, HB_THREADS, 0, st>>>(tokens, tok_off, blk_off, N, hashes,
                                                                  hashes_capacity);
        }
        {
            Prof pr(PROF_HASH_CHAIN, st, 1);
            k_block_chain<<<(unsigned)((N + 127) / 128), 128, 0, st>>>(blk_off, N, seed, hashes,
                                                                      hashes_capacity);
        }
    }
    PEEK_CUDA(cudaGetLastError());
    return PEEK_OK;
}
