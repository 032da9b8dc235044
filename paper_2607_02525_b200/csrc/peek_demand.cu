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
#include "peek_sort.cuh"

namespace peek {

// ---- demand -----------------------------------------------------------------------------

__device__ __forceinline__ i64 table_slot_from(const u64* __restrict__ t_keys, u64 mask, u64 key, u64 p,
                                              u64 tk) {  // tk = t_keys[p] already loaded
    for (;;) {
        if (tk == key) return (i64)p;
        if (tk == PEEK_EMPTY) return -1;
        p = (p + 1) & mask;
        tk = ld_u64_keep(t_keys + p);
    }
}

// A warp owns 32 consecutive sorted positions.  Lane q describes position j0 + q: its chain, the
// range [l0, nb) of blocks that first appear there, and the first step of the next-smaller-value
// walk (blocks [lo1, l1) are shared with positions j+1 .. t1-1, pending_count cnt1 = t1 - j).  The
// new blocks of the 32 positions are then flattened and handed out 32 x DM_UNROLL at a time, one
// block per lane: hash load -> table probe -> atomicAdd(pending_count), coalesced along each chain.
// Blocks below lo1 (tries nested deeper than one level under this position) take a per-lane search.
static constexpr int DM_THREADS = 256, DM_WARPS = DM_THREADS / 32, DM_UNROLL = 2;

struct DemandMeta {
    i64 b0[32];
    i32 l0[32], l1[32], lo1[32], cnt1[32], t1[32];
};

template <bool TAGS>
__global__ void __launch_bounds__(DM_THREADS) k_demand(const u64* __restrict__ hashes,
                                                      const i64* __restrict__ blk_off, i64 N,
                                                      const i32* __restrict__ order,
                                                      const i32* __restrict__ lcp, MinTree mt,
                                                      const u64* __restrict__ t_keys, u64 mask,
                                                      const unsigned char* __restrict__ tags,
                                                      i32* __restrict__ demand, int ppw) {
    // ppw = positions per warp (1..32): few long chains (small N) spread over more warps
    __shared__ DemandMeta sm[DM_WARPS];
    const unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const i64 j0 = (((i64)blockIdx.x * DM_THREADS + threadIdx.x) >> 5) * ppw;
    if (j0 >= N) return;
    DemandMeta& M = sm[w];
    const i64 j = j0 + lane;
    i32 n_new = 0;
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
        }
        i32 lo1 = l1, cnt1 = 1, t1 = (i32)(j + 1);
        if (valid && l1 > l0) {
            const i64 t = nsv_next_less(mt, j + 1, l1);  // first later position sharing < l1 blocks
            const i32 lt = mt.val(0, t);
            lo1 = lt > l0 ? lt : l0;
            cnt1 = (i32)(t - j);
            t1 = (i32)t;
        }
        M.b0[lane] = b0; M.l0[lane] = l0; M.l1[lane] = l1; M.lo1[lane] = lo1; M.cnt1[lane] = cnt1; M.t1[lane] = t1;
    }
    i32 pre = n_new;  // inclusive prefix of the new-block counts over the warp's positions
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const i32 t = __shfl_up_sync(FULL, pre, o);
        if (lane >= o) pre += t;
    }
    const i32 total = __shfl_sync(FULL, pre, 31);
    const i32 excl = pre - n_new;
    __syncwarp();
    for (i32 base = 0; base < total; base += 32 * DM_UNROLL) {
        u64 key[DM_UNROLL], slot0[DM_UNROLL], tk[DM_UNROLL];
        i32 cnt[DM_UNROLL];
        bool act[DM_UNROLL];
#pragma unroll
        for (int u = 0; u < DM_UNROLL; ++u) {
            const i32 it = base + u * 32 + lane;
            act[u] = it < total;
            const i32 itc = act[u] ? it : total - 1;
            int lo = 0, hi = 31;  // first position q with pre[q] > itc
#pragma unroll
            for (int s = 0; s < 5; ++s) {
                const int mid = (lo + hi) >> 1;
                const i32 v = __shfl_sync(FULL, pre, mid);
                if (v > itc) hi = mid; else lo = mid + 1;
            }
            const int q = lo;
            const i32 i = M.l0[q] + (itc - __shfl_sync(FULL, excl, q));
            key[u] = ld_u64_once(hashes + M.b0[q] + i);
            i32 c = 1;
            if (i < M.l1[q]) {
                if (i >= M.lo1[q]) c = M.cnt1[q];
                else c = (i32)(nsv_next_less(mt, (i64)M.t1[q], i + 1) - (j0 + q));
            }
            cnt[u] = c;
        }
#pragma unroll
        for (int u = 0; u < DM_UNROLL; ++u) {
            slot0[u] = key[u] & mask;
            tk[u] = TAGS ? ld_tagword(tags + (slot0[u] & ~7ull)) : ld_u64_keep(t_keys + slot0[u]);
        }
#pragma unroll
        for (int u = 0; u < DM_UNROLL; ++u) {
            if (act[u]) {
                const i64 p = TAGS ? table_slot_tagged(t_keys, tags, mask, key[u], slot0[u], tk[u])
                                   : table_slot_from(t_keys, mask, key[u], slot0[u], tk[u]);
                if (p >= 0) atomicAdd(demand + p, cnt[u]);
            }
        }
    }
}

// ---- cLPM order ---------------------------------------------------------------------------
// Order-preserving u32 images of the three key parts: th, tc descending (signed), ta ascending.
// One pass finds their ranges; the parts are packed, range-compressed, into one u64 key when they
// fit (they do for every BASELINE config: e.g. 15 + 5 + 20 bits in config 5) and the pairs
// (key, request index) go through ONE stable LSD sort whose passes cover only the varying bits.
// If they do not fit: a first sort by arrival, then a stable sort by (hit, cluster size).
struct RankCtl {
    u32 bar;
    u32 mx[3];  // max of th, tc, ta
    u32 mn[3];  // max of ~th, ~tc, ~ta  (i.e. ~min)
    u32 pad;
    unsigned long long vary[2];
};

struct RankArgs {
    const i32 *hit, *csize, *arrival;
    i64 N;
    i32* out;
    RankCtl* ctl;
    GsBufs bufs;
};

__device__ __forceinline__ u32 img_desc(i32 v) { return ~((u32)v ^ 0x80000000u); }
__device__ __forceinline__ u32 img_asc(i32 v) { return (u32)v ^ 0x80000000u; }

// Queues of at most RANK_SMALL_MAX requests (the paper's own queues hold 60-200): one
// CTA, thread r ranks request r by counting the requests that precede it under the same total order
// (hit desc, cluster size desc, arrival asc, index) - N broadcast shared-memory reads per thread
// instead of range pass + packed keys + radix passes through global memory.
static constexpr int RANK_SMALL_MAX = 512;
__global__ void __launch_bounds__(RANK_SMALL_MAX) k_clpm_rank_small(RankArgs A) {
    __shared__ u64 s_hc[RANK_SMALL_MAX], s_ai[RANK_SMALL_MAX];
    const int r = threadIdx.x, N = (int)A.N;
    u64 hc = 0, ai = 0;
    if (r < N) {
        hc = ((u64)img_desc(__ldg(A.hit + r)) << 32) | (u64)img_desc(__ldg(A.csize + r));
        ai = ((u64)(A.arrival ? img_asc(__ldg(A.arrival + r)) : (u32)r) << 32) | (u64)(u32)r;
        s_hc[r] = hc;
        s_ai[r] = ai;
    }
    __syncthreads();
    if (r >= N) return;
    int rank = 0;
#pragma unroll 4
    for (int j = 0; j < N; ++j) {
        const u64 h = s_hc[j], a = s_ai[j];
        rank += (h < hc || (h == hc && a < ai)) ? 1 : 0;
    }
    A.out[rank] = r;
}

__global__ void __launch_bounds__(GS_THREADS, 1) k_clpm_sort(RankArgs A) {
    extern __shared__ __align__(16) unsigned char dyn_smem[];
    __shared__ GsSmem ssm;
    const GsStage stg = gs_stage(dyn_smem);
    const i64 N = A.N;
    const i64 gtid = (i64)blockIdx.x * GS_THREADS + threadIdx.x, gsize = (i64)gridDim.x * GS_THREADS;
    Grid g{&A.ctl->bar, 0};
    PEEK_MARK(1);
    if (gridDim.x == 1) {  // one CTA: the control block and the sort's accumulators are cleared here, not by a memset node
        for (int i = threadIdx.x; i < (int)(sizeof(RankCtl) / 4); i += GS_THREADS) ((u32*)A.ctl)[i] = 0;
        for (int i = threadIdx.x; i < (int)gs_hist_words(1); i += GS_THREADS) A.bufs.hist[i] = 0;
        __syncthreads();
    }
    const i32* __restrict__ hit = A.hit;
    const i32* __restrict__ cs = A.csize;
    const i32* __restrict__ arr = A.arrival;
    {   // ranges of the three key images; RK_U x 3 loads in flight per thread
        constexpr int RK_U = 8;
        u32 mx[3] = {0, 0, 0}, mn[3] = {0, 0, 0};
        for (i64 r0 = gtid; r0 < N; r0 += gsize * RK_U) {
            u32 v[RK_U][3];
#pragma unroll
            for (int u = 0; u < RK_U; ++u) {
                const i64 r = r0 + u * gsize;
                const bool in = r < N;
                v[u][0] = in ? img_desc(__ldg(hit + r)) : 0;
                v[u][1] = in ? img_desc(__ldg(cs + r)) : 0;
                v[u][2] = in ? (arr ? img_asc(__ldg(arr + r)) : (u32)r) : 0;
            }
#pragma unroll
            for (int u = 0; u < RK_U; ++u) {
                if (r0 + u * gsize < N) {
#pragma unroll
                    for (int q = 0; q < 3; ++q) { mx[q] = max(mx[q], v[u][q]); mn[q] = max(mn[q], ~v[u][q]); }
                }
            }
        }
        // CTA-level max through shared memory, then six atomics per CTA
        __shared__ u32 s_mm[6];
        if (threadIdx.x < 6) s_mm[threadIdx.x] = 0;
        __syncthreads();
#pragma unroll
        for (int q = 0; q < 3; ++q) {
            const u32 a = __reduce_max_sync(0xffffffffu, mx[q]), b = __reduce_max_sync(0xffffffffu, mn[q]);
            if ((threadIdx.x & 31) == 0) { atomicMax(&s_mm[q], a); atomicMax(&s_mm[3 + q], b); }
        }
        __syncthreads();
        if (threadIdx.x < 3) atomicMax(&A.ctl->mx[threadIdx.x], s_mm[threadIdx.x]);
        else if (threadIdx.x < 6) atomicMax(&A.ctl->mn[threadIdx.x - 3], s_mm[threadIdx.x]);
    }
    g.sync();
    PEEK_MARK(2);
    u32 lo[3];
    int bits[3];
#pragma unroll
    for (int q = 0; q < 3; ++q) {
        lo[q] = ~__ldcg(&A.ctl->mn[q]);
        bits[q] = bits_for((u64)(__ldcg(&A.ctl->mx[q]) - lo[q]));
    }
    const int bca = bits[1] + bits[2], ball = bits[0] + bca;
    const bool one = ball <= 64;
    auto key_a = [&](u32 r) -> u64 { return (u64)((arr ? img_asc(__ldg(arr + r)) : r) - lo[2]); };
    auto key_hc = [&](u32 r) -> u64 {
        return ((u64)(img_desc(__ldg(hit + r)) - lo[0]) << bits[1]) | (u64)(img_desc(__ldg(cs + r)) - lo[1]);
    };
    auto mask_of = [](int nb) -> u64 { return nb >= 64 ? ~0ull : ((1ull << nb) - 1ull); };
    int src;
    if (one) {  // one packed key: [hit | cluster size | arrival], request index breaks ties (stable)
        src = grid_sort_pairs_gen(A.bufs, N, mask_of(ball), g, ssm, stg, [&](i64 i, u64& k, u32& v) {
            v = (u32)i;
            k = (key_hc((u32)i) << bits[2]) | key_a((u32)i);  // bits[2] <= 32 here: no shift overflow
        });
    } else {    // arrival first, then a stable sort by (hit, cluster size)
        src = grid_sort_pairs_gen(A.bufs, N, mask_of(bits[2]), g, ssm, stg, [&](i64 i, u64& k, u32& v) {
            v = (u32)i;
            k = key_a((u32)i);
        });
        for (i64 j = gtid; j < N; j += gsize) A.bufs.key[src][j] = key_hc(__ldcg(&A.bufs.val[src][j]));
        g.sync();
        src = grid_sort_pairs(A.bufs, N, mask_of(bits[0] + bits[1]), g, ssm, stg, src);
    }
    PEEK_MARK(3);
    const u32* res = A.bufs.val[src];
    for (i64 j = gtid; j < N; j += gsize) A.out[j] = (i32)__ldcg(res + j);
    PEEK_MARK(4);
}

// ---- the full Eq. 1 key: (section, -h, -score, -|cluster|, arrival), index last ----
// Five parts, least significant first: arrival, cluster size, score, hit, section.  Their ranges
// are measured, consecutive parts are packed greedily into 64-bit keys, and every pack is one
// stable pair sort on top of the previous order (config 5: 20 + 5 + 35 bits, then 15 + 2 bits).
struct FullCtl {
    u32 bar, pad;
    unsigned long long mx[5], mn[5];  // max of the image, max of its complement (= ~min)
};
struct FullArgs {
    const i32 *section, *hit, *csize, *arrival;
    const i64* score;
    i64 N;
    i32* out;
    FullCtl* ctl;
    GsBufs bufs;
    int nparts;       // key parts in use, least significant first
    int part[5];      // which: 0 arrival asc, 1 cluster size desc, 2 score desc, 3 hit desc, 4 section asc
};
__device__ __forceinline__ u64 full_part(const FullArgs& A, int q, u32 r) {
    switch (A.part[q]) {
        case 0: return A.arrival ? (u64)img_asc(__ldg(A.arrival + r)) : (u64)r;
        case 1: return (u64)img_desc(__ldg(A.csize + r));
        case 2: return ~((u64)__ldg(A.score + r) ^ 0x8000000000000000ull);
        case 3: return (u64)img_desc(__ldg(A.hit + r));
        default: return (u64)img_asc(__ldg(A.section + r));
    }
}

__global__ void __launch_bounds__(GS_THREADS, 1) k_clpm_sort_full(FullArgs A) {
    extern __shared__ __align__(16) unsigned char dyn_smem[];
    __shared__ GsSmem ssm;
    __shared__ unsigned long long s_mm[10];
    const GsStage stg = gs_stage(dyn_smem);
    const i64 N = A.N;
    const i64 gtid = (i64)blockIdx.x * GS_THREADS + threadIdx.x, gsize = (i64)gridDim.x * GS_THREADS;
    Grid g{&A.ctl->bar, 0};
    {
        u64 mx[5] = {0, 0, 0, 0, 0}, mn[5] = {0, 0, 0, 0, 0};
        for (i64 r = gtid; r < N; r += gsize) {
#pragma unroll
            for (int q = 0; q < 5; ++q) {
                if (q < A.nparts) {
                    const u64 v = full_part(A, q, (u32)r);
                    mx[q] = v > mx[q] ? v : mx[q];
                    mn[q] = ~v > mn[q] ? ~v : mn[q];
                }
            }
        }
        if (threadIdx.x < 10) s_mm[threadIdx.x] = 0;
        __syncthreads();
#pragma unroll
        for (int q = 0; q < 5; ++q) {
            atomicMax(&s_mm[q], (unsigned long long)mx[q]);
            atomicMax(&s_mm[5 + q], (unsigned long long)mn[q]);
        }
        __syncthreads();
        if (threadIdx.x < 5) atomicMax(&A.ctl->mx[threadIdx.x], s_mm[threadIdx.x]);
        else if (threadIdx.x < 10) atomicMax(&A.ctl->mn[threadIdx.x - 5], s_mm[threadIdx.x]);
    }
    g.sync();
    u64 lo[5];
    int bits[5];
#pragma unroll
    for (int q = 0; q < 5; ++q) {
        lo[q] = ~__ldcg(&A.ctl->mn[q]);
        const u64 span = __ldcg(&A.ctl->mx[q]) - lo[q];
        bits[q] = (span == 0 || q >= A.nparts) ? 0 : bits_for(span);  // a constant part takes no key bits
    }
    int src = -1;  // buffer holding the current order; -1: the identity
    int q0 = 0;
    const int NP = A.nparts;
    while (q0 < NP) {
        int q1 = q0, total = 0;
        while (q1 < NP && total + bits[q1] <= 64) { total += bits[q1]; ++q1; }
        // parts q0 .. q1-1 form this sort's key, part q0 in the low bits
        auto make_key = [&](u32 r) -> u64 {
            u64 key = 0;
            int sh = 0;
            for (int q = q0; q < q1; ++q) {
                if (bits[q]) { key |= (full_part(A, q, r) - lo[q]) << sh; sh += bits[q]; }
            }
            return key;
        };
        const u64 vary = total >= 64 ? ~0ull : ((1ull << total) - 1ull);
        if (src < 0) {
            src = grid_sort_pairs_gen(A.bufs, N, vary, g, ssm, stg, [&](i64 i, u64& k, u32& v) {
                v = (u32)i;
                k = make_key((u32)i);
            });
        } else if (vary) {
            for (i64 j = gtid; j < N; j += gsize) A.bufs.key[src][j] = make_key(__ldcg(&A.bufs.val[src][j]));
            g.sync();
            src = grid_sort_pairs(A.bufs, N, vary, g, ssm, stg, src);
            g.sync();
        }
        q0 = q1;
    }
    const u32* res = A.bufs.val[src];
    for (i64 j = gtid; j < N; j += gsize) A.out[j] = (i32)__ldcg(res + j);
}

static void full_layout(Arena& a, i64 N, int grid, FullArgs& A) {
    A.ctl = a.take<FullCtl>(1);
    A.bufs.hist = a.take<u32>(gs_hist_words(grid));  // directly after ctl: one memset clears both
    A.bufs.key[0] = a.take<u64>(N);
    A.bufs.key[1] = a.take<u64>(N);
    A.bufs.val[0] = a.take<u32>(N);
    A.bufs.val[1] = a.take<u32>(N);
}

static void rank_layout(Arena& a, i64 N, int grid, RankArgs& A) {
    A.ctl = a.take<RankCtl>(1);
    A.bufs.hist = a.take<u32>(gs_hist_words(grid));  // directly after ctl: one memset clears both
    A.bufs.key[0] = a.take<u64>(N);
    A.bufs.key[1] = a.take<u64>(N);
    A.bufs.val[0] = a.take<u32>(N);
    A.bufs.val[1] = a.take<u32>(N);
}

static constexpr int RANK_MAX_GRID = 1024;  // workspace sizing bound on the cooperative grid

// ---- group-major admission (R24) -----------------------------------------
// order by (lane position of the cluster's first member, own lane position).  The first member is
// an atomicMin per cluster through an open-addressed table keyed by cluster_id (clusters nested
// on the same leftmost leaf differ in depth, so the id, not the leaf, is the key); then one pair sort.
struct GmCtl { u32 bar, pad; };
struct GmArgs {
    const i32* lane;
    const i64* cluster_id;
    i64 N;
    i32* out;
    GmCtl* ctl;
    GsBufs bufs;
    unsigned long long* tkeys;  // H slots, all-ones = empty
    u32* tfirst;                // H slots
    u32* slot;                  // N: table slot of the cluster of the request at lane position p
    u64 hmask;
};

__global__ void __launch_bounds__(GS_THREADS, 1) k_group_major(GmArgs A) {
    extern __shared__ __align__(16) unsigned char dyn_smem[];
    __shared__ GsSmem ssm;
    const GsStage stg = gs_stage(dyn_smem);
    const i64 N = A.N;
    const i64 gtid = (i64)blockIdx.x * GS_THREADS + threadIdx.x, gsize = (i64)gridDim.x * GS_THREADS;
    Grid g{&A.ctl->bar, 0};
    for (i64 p = gtid; p < N; p += gsize) {
        const u32 r = (u32)__ldg(A.lane + p);
        const unsigned long long cid = (unsigned long long)__ldg(A.cluster_id + r);
        u64 h = mix64(cid) & A.hmask;
        for (;;) {
            const unsigned long long prev = atomicCAS(A.tkeys + h, ~0ull, cid);
            if (prev == ~0ull || prev == cid) break;
            h = (h + 1) & A.hmask;
        }
        atomicMin(A.tfirst + h, (u32)p);
        A.slot[p] = (u32)h;
    }
    g.sync();
    const int nbits = bits_for((u64)(N > 1 ? N - 1 : 1));
    const int src = grid_sort_pairs_gen(A.bufs, N, nbits >= 32 ? ~0ull : ((1ull << (2 * nbits)) - 1ull), g, ssm, stg,
                                        [&](i64 p, u64& k, u32& v) {
        v = (u32)__ldg(A.lane + p);
        k = ((u64)__ldcg(A.tfirst + __ldcg(A.slot + p)) << nbits) | (u64)p;
    });
    const u32* res = A.bufs.val[src];
    for (i64 j = gtid; j < N; j += gsize) A.out[j] = (i32)__ldcg(res + j);
}

static i64 gm_table_slots(i64 N) {
    i64 h = 64;
    while (h < 2 * N) h <<= 1;
    return h;
}
static void gm_layout(Arena& a, i64 N, int grid, GmArgs& A) {
    A.ctl = a.take<GmCtl>(1);
    A.bufs.hist = a.take<u32>(gs_hist_words(grid));  // directly after ctl: one memset clears both
    A.bufs.key[0] = a.take<u64>(N);
    A.bufs.key[1] = a.take<u64>(N);
    A.bufs.val[0] = a.take<u32>(N);
    A.bufs.val[1] = a.take<u32>(N);
    const i64 H = gm_table_slots(N);
    A.tkeys = a.take<unsigned long long>(H);
    A.tfirst = a.take<u32>(H);  // directly after tkeys: one 0xff memset covers both
    A.slot = a.take<u32>(N);
    A.hmask = (u64)(H - 1);
}
i64 group_major_ws_bytes(i64 N) {
    Arena a(nullptr);
    GmArgs A;
    gm_layout(a, N, 1024, A);
    return a.used;
}

i64 clpm_order_full_ws_bytes(i64 N) {
    Arena a(nullptr);
    FullArgs A;
    full_layout(a, N, 1024, A);
    return a.used;
}

i64 demand_rank_ws_bytes(i64 N, i64 S) {
    Arena a(nullptr);
    RankArgs A;
    rank_layout(a, N, RANK_MAX_GRID, A);
    a.take<i32>(mintree_words(N));
    if (S >= TAGS_MIN_S) a.take<unsigned char>(S);
    return a.used;
}


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
    if (N > 0 && (demand || clpm_order) &&
        (!ws || ((uintptr_t)ws & 255) || ws_bytes < demand_rank_ws_bytes(N, table ? table->S : 0))) {
        set_error("peek_demand_rank: workspace NULL, misaligned or too small");
        return PEEK_ERR_WORKSPACE;
    }
    // every argument is checked: from here on work is enqueued
    // (the tag pass reads the keys and clears the counters with 16-byte accesses)
    const bool tagged = demand && N > 0 && table->S >= TAGS_MIN_S && (((uintptr_t)table->t_keys | (uintptr_t)demand) & 15) == 0;
    if (demand && !tagged) PEEK_CUDA(cudaMemsetAsync(demand, 0, sizeof(i32) * (size_t)table->S, st));  // else k_table_tags clears it
    if (N == 0 || (!demand && !clpm_order)) return PEEK_OK;
    Arena a(ws);
    RankArgs A;
    rank_layout(a, N, RANK_MAX_GRID, A);
    i32* mt_buf = a.take<i32>(mintree_words(N));
    unsigned char* tags = (table && table->S >= TAGS_MIN_S) ? a.take<unsigned char>(table->S) : nullptr;
    a.arm(st);
    if (demand) {
        MinTree mt;
        mintree_layout(mt, lcp, N, mt_buf);
        Prof pr(PROF_DEMAND, st, mintree_launches(mt) + 1 + (tagged ? 1 : 0));
        if (tagged) k_table_tags<<<(unsigned)((table->S / 8 + 255) / 256), 256, 0, st>>>(table->t_keys, table->S, tags, demand);
        mintree_build(mt, st);
        int ppw = 32;  // at least ~16 K warps when the queue is small
        while (ppw > 1 && N / ppw < 16384) ppw >>= 1;
        const i64 warps = (N + ppw - 1) / ppw;
        unsigned grid = (unsigned)((warps * 32 + DM_THREADS - 1) / DM_THREADS);
        if (tagged) k_demand<true><<<grid, DM_THREADS, 0, st>>>(hashes, blk_off, N, order, lcp, mt, table->t_keys,
                                                                (u64)(table->S - 1), tags, demand, ppw);
        else k_demand<false><<<grid, DM_THREADS, 0, st>>>(hashes, blk_off, N, order, lcp, mt, table->t_keys,
                                                          (u64)(table->S - 1), nullptr, demand, ppw);
    }
    if (clpm_order) {
        A.hit = hit; A.csize = cluster_size; A.arrival = arrival; A.N = N; A.out = clpm_order;
        int grid = persistent_ctas();  // one CTA of GS_THREADS per SM (co-resident: cooperative launch)
        if (grid > RANK_MAX_GRID) grid = RANK_MAX_GRID;
        i64 want = (N + GS_THREADS - 1) / GS_THREADS;
        if (want < grid) grid = (int)(want < 1 ? 1 : want);
        if (grid > 1) {
            PEEK_CUDA(cudaMemsetAsync(A.ctl, 0, (size_t)((char*)(A.bufs.hist + gs_hist_words(RANK_MAX_GRID)) - (char*)A.ctl), st));
            a.arm(st);  // the memset spans a canary
        }
        void* params[] = {&A};
        Prof pr(PROF_RANK, st, 1);
        if (N <= RANK_SMALL_MAX && !grid_limited()) {  // PEEK_OPT_GRID_LIMIT (test hook) keeps the general path
            k_clpm_rank_small<<<1, RANK_SMALL_MAX, 0, st>>>(A);
            PEEK_CUDA(cudaGetLastError());
            return PEEK_OK;
        }
        PEEK_CUDA(func_smem_optin((const void*)k_clpm_sort, GS_STAGE_BYTES));
        if (grid == 1) k_clpm_sort<<<1, GS_THREADS, GS_STAGE_BYTES, st>>>(A);  // one CTA: no co-residency to ask for
        else PEEK_CUDA(cudaLaunchCooperativeKernel((const void*)k_clpm_sort, dim3(grid), dim3(GS_THREADS), params,
                                                   GS_STAGE_BYTES, st));
    }
    PEEK_CUDA(cudaGetLastError());
    return PEEK_OK;
}

static peek_status launch_sort_full(FullArgs& A, i64 N, void* ws, cudaStream_t st) {
    Arena a(ws);
    full_layout(a, N, 1024, A);
    int grid = persistent_ctas();
    if (grid > 1024) grid = 1024;
    i64 want = (N + GS_THREADS - 1) / GS_THREADS;
    if (want < grid) grid = (int)(want < 1 ? 1 : want);
    PEEK_CUDA(cudaMemsetAsync(A.ctl, 0, (size_t)((char*)(A.bufs.hist + gs_hist_words(1024)) - (char*)A.ctl), st));
    a.arm(st);
    PEEK_CUDA(func_smem_optin((const void*)k_clpm_sort_full, GS_STAGE_BYTES));
    void* params[] = {&A};
    Prof pr(PROF_RANK_FULL, st, 1);
    PEEK_CUDA(cudaLaunchCooperativeKernel((const void*)k_clpm_sort_full, dim3(grid), dim3(GS_THREADS), params,
                                          GS_STAGE_BYTES, st));
    return PEEK_OK;
}

extern "C" peek_status peek_clpm_order_full(const int32_t* section, const int32_t* hit, const int64_t* score,
                                            const int32_t* cluster_size, const int32_t* arrival, int64_t N,
                                            int32_t* clpm_order, void* ws, int64_t ws_bytes, void* stream) {
    if (N < 0 || N >= 0x7fffffffLL) { set_error("peek_clpm_order_full: N out of range"); return PEEK_ERR_INVALID_ARG; }
    if (N == 0) return PEEK_OK;
    if (!section || !hit || !score || !cluster_size || !clpm_order) {
        set_error("peek_clpm_order_full: NULL argument");
        return PEEK_ERR_INVALID_ARG;
    }
    if (!ws || ((uintptr_t)ws & 255) || ws_bytes < clpm_order_full_ws_bytes(N)) {
        set_error("peek_clpm_order_full: workspace NULL, misaligned or too small");
        return PEEK_ERR_WORKSPACE;
    }
    FullArgs A;
    A.section = section; A.hit = hit; A.score = score; A.csize = cluster_size; A.arrival = arrival;
    A.N = N; A.out = clpm_order;
    A.nparts = 5;
    for (int q = 0; q < 5; ++q) A.part[q] = q;  // arrival, cluster, score, hit, section
    return launch_sort_full(A, N, ws, (cudaStream_t)stream);
}

// fairness lane of Alg. 2 line 18: (section, arrival, -h), index last
extern "C" peek_status peek_clpm_lane_b(const int32_t* section, const int32_t* hit, const int32_t* arrival,
                                        int64_t N, int32_t* lane_b_order, void* ws, int64_t ws_bytes, void* stream) {
    if (N < 0 || N >= 0x7fffffffLL) { set_error("peek_clpm_lane_b: N out of range"); return PEEK_ERR_INVALID_ARG; }
    if (N == 0) return PEEK_OK;
    if (!section || !hit || !lane_b_order) { set_error("peek_clpm_lane_b: NULL argument"); return PEEK_ERR_INVALID_ARG; }
    if (!ws || ((uintptr_t)ws & 255) || ws_bytes < clpm_order_full_ws_bytes(N)) {
        set_error("peek_clpm_lane_b: workspace NULL, misaligned or too small");
        return PEEK_ERR_WORKSPACE;
    }
    FullArgs A;
    A.section = section; A.hit = hit; A.score = nullptr; A.csize = nullptr; A.arrival = arrival;
    A.N = N; A.out = lane_b_order;
    A.nparts = 3;
    A.part[0] = 3; A.part[1] = 0; A.part[2] = 4; A.part[3] = A.part[4] = 0;  // hit desc, arrival, section
    return launch_sort_full(A, N, ws, (cudaStream_t)stream);
}

// ---- dynamic-lane controller (Alg. 2 line 20; R27) ---------------------
__global__ void __launch_bounds__(256) k_count_singletons(const i32* __restrict__ cs, i64 N, unsigned long long* cnt) {
    u32 c = 0;
    for (i64 r = (i64)blockIdx.x * 256 + threadIdx.x; r < N; r += (i64)gridDim.x * 256) c += cs[r] == 1;
    c = __reduce_add_sync(0xffffffffu, c);
    if ((threadIdx.x & 31) == 0 && c) atomicAdd(cnt, (unsigned long long)c);
}
__global__ void k_dynamic_lane(const unsigned long long* cnt, i64 N, double age, double prev, double* out) {
    // every product and sum rounded once (no fused multiply-add), as the plain definition does
    const double sf = N ? __ddiv_rn((double)*cnt, (double)N) : 0.0;
    double x = __dadd_rn(__dadd_rn(0.15, __dmul_rn(0.5, sf)), __dmul_rn(0.3, age));
    if (x < 0.10) x = 0.10;
    if (x > 0.60) x = 0.60;
    out[0] = __dadd_rn(__dmul_rn(0.3, x), __dmul_rn(0.7, prev));
    out[1] = sf;
}
extern "C" peek_status peek_dynamic_lane(const int32_t* cluster_size, int64_t N, double age_pressure,
                                         double prev_fair_share, double* out, void* ws, int64_t ws_bytes,
                                         void* stream) {
    if (N < 0 || !out || (N > 0 && !cluster_size)) { set_error("peek_dynamic_lane: bad argument"); return PEEK_ERR_INVALID_ARG; }
    if (!ws || ((uintptr_t)ws & 255) || ws_bytes < 256) { set_error("peek_dynamic_lane: workspace"); return PEEK_ERR_WORKSPACE; }
    cudaStream_t st = (cudaStream_t)stream;
    unsigned long long* cnt = (unsigned long long*)ws;
    PEEK_CUDA(cudaMemsetAsync(cnt, 0, sizeof(unsigned long long), st));
    Prof pr(PROF_RANK_FULL, st, 2);
    if (N > 0) {
        unsigned grid = (unsigned)((N + 255) / 256);
        if (grid > 148u * 8u) grid = 148u * 8u;
        k_count_singletons<<<grid, 256, 0, st>>>(cluster_size, N, cnt);
    }
    k_dynamic_lane<<<1, 1, 0, st>>>(cnt, N, age_pressure, prev_fair_share, out);
    PEEK_CUDA(cudaGetLastError());
    return PEEK_OK;
}

extern "C" peek_status peek_clpm_group_major(const int32_t* lane_order, const int64_t* cluster_id, int64_t N,
                                             int32_t* gm_order, void* ws, int64_t ws_bytes, void* stream) {
    if (N < 0 || N >= 0x7fffffffLL) { set_error("peek_clpm_group_major: N out of range"); return PEEK_ERR_INVALID_ARG; }
    if (N == 0) return PEEK_OK;
    if (!lane_order || !cluster_id || !gm_order) {
        set_error("peek_clpm_group_major: NULL argument");
        return PEEK_ERR_INVALID_ARG;
    }
    if (!ws || ((uintptr_t)ws & 255) || ws_bytes < group_major_ws_bytes(N)) {
        set_error("peek_clpm_group_major: workspace NULL, misaligned or too small");
        return PEEK_ERR_WORKSPACE;
    }
    cudaStream_t st = (cudaStream_t)stream;
    Arena a(ws);
    GmArgs A;
    gm_layout(a, N, 1024, A);
    A.lane = lane_order; A.cluster_id = cluster_id; A.N = N; A.out = gm_order;
    int grid = persistent_ctas();
    if (grid > 1024) grid = 1024;
    i64 want = (N + GS_THREADS - 1) / GS_THREADS;
    if (want < grid) grid = (int)(want < 1 ? 1 : want);
    PEEK_CUDA(cudaMemsetAsync(A.ctl, 0, (size_t)((char*)(A.bufs.hist + gs_hist_words(1024)) - (char*)A.ctl), st));
    PEEK_CUDA(cudaMemsetAsync(A.tkeys, 0xff, (size_t)((char*)(A.tfirst + (A.hmask + 1)) - (char*)A.tkeys), st));
    a.arm(st);
    PEEK_CUDA(func_smem_optin((const void*)k_group_major, GS_STAGE_BYTES));
    void* params[] = {&A};
    Prof pr(PROF_RANK_FULL, st, 1);
    PEEK_CUDA(cudaLaunchCooperativeKernel((const void*)k_group_major, dim3(grid), dim3(GS_THREADS), params,
                                          GS_STAGE_BYTES, st));
    return PEEK_OK;
}

PEEK_TRACE_EXPORT(peek_trace_read_rank)

using namespace peek;

