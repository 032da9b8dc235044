// peek_tree.cu — a2-a4 peek_pending_tree: the pending radix tree built as
// a batch: lexicographic order of the requests' hash chains (= DFS order of the compressed trie),
// adjacent LCP (= its branching depths), flat groups and per-request clusters.
//
// ONE persistent cooperative kernel (a CTA per SM slot, grid barriers between phases), because
// the number of refinement rounds is data dependent and the call may not synchronise with the host.
//
// Sort = path-peeling refinement.  Every unresolved segment (a run of sorted positions whose
// chains share a prefix) picks its LONGEST chain as head h.  A member r is classified by its
// LCP with h in units of w-bit digits (a 64-bit hash word = D digits, most significant first):
//     r proper prefix of h            -> before h, by ascending LCP, "ended" (identical chains)
//     r's digit < h's at the LCP      -> before h, by ascending LCP, then digit
//     r identical to h                -> with h
//     r's digit > h's at the LCP      -> after h, by DESCENDING LCP, then digit
// One stable LSD radix sort by key = [segment start | class+LCP | digit] splits the segment along
// the whole root-to-leaf path of h at once, so rounds ~ 3 on the paper's workloads (shared
// prompt / conversation / turn) instead of one per trie level.  LCPs use the chain property
// (k_i equal => all earlier words equal, R15) to binary-search the first differing word.
#include "peek_sort.cuh"

namespace peek {

struct TreeCtl {      // device control block (zeroed by the host before launch)
    u32 bar;          // grid barrier word
    u32 unres[3];     // unresolved-position counters, rotating
    u32 maxnb;        // max chain length in blocks
    u32 pad[3];
    unsigned long long kor[2], kand[2];  // OR / AND of the round's keys (rotating): varying bits
};

struct TreeArgs {
    const u64* hashes;
    const i64* blk_off;
    i64 N;
    i32 *order, *lcp, *group_id, *group_size, *cluster_depth, *cluster_size;
    i64* cluster_id;
    i32* n_groups;
    // workspace
    TreeCtl* ctl;
    GsBufs bufs;      // (sort key, request) by position, ping-pong
    u32* seg;         // N   by position: segment start | unresolved << 31
    u64* seghead;     // N   by segment start: (nb << 32) | ~position of the longest chain
    i32* segdepth;    // N   by segment start: blocks all members are known to share
    i64* agg;         // gridDim scratch for grid scans
    i32* gsz;         // N   group size by group id
    i32* mt_buf;      // min hierarchy
};

// number of leading equal hash words of chains a[0..na), b[0..nb), given the first `lo` are equal
__device__ __forceinline__ i64 chain_lcp(const u64* __restrict__ a, i64 na, const u64* __restrict__ b, i64 nb,
                                         i64 lo) {
    i64 m = na < nb ? na : nb;
    if (m <= lo) return m;
    if (__ldg(a + m - 1) == __ldg(b + m - 1)) return m;
    if (__ldg(a + lo) != __ldg(b + lo)) return lo;
    i64 L = lo, R = m - 1;  // equal at L, differ at R
    while (R - L > 1) {
        i64 mid = (L + R) >> 1;
        if (__ldg(a + mid) == __ldg(b + mid)) L = mid; else R = mid;
    }
    return R;
}

struct KeyLayout {
    int w, D, lbits, sbits, total;
    u64 LDmax;
    __device__ __forceinline__ u64 f_before(u64 ld, bool ended) const { return 2 * ld + (ended ? 0 : 1); }
    __device__ __forceinline__ u64 f_head() const { return 2 * LDmax + 2; }
    __device__ __forceinline__ u64 f_after(u64 ld) const { return 2 * LDmax + 3 + (LDmax - ld); }
    __device__ __forceinline__ bool is_branch(u64 F) const {
        return (F <= 2 * LDmax + 1) ? (F & 1) : (F >= 2 * LDmax + 3);
    }
    __device__ __forceinline__ u64 ld_of(u64 F) const {  // digit LCP of a branch class
        return (F <= 2 * LDmax + 1) ? (F >> 1) : (LDmax - (F - (2 * LDmax + 3)));
    }
    __device__ __forceinline__ u64 pack(u64 seg, u64 F, u64 dig) const {
        return (seg << (lbits + w)) | (F << w) | dig;
    }
    __device__ __forceinline__ u64 F_of(u64 key) const { return (key >> w) & ((1ull << lbits) - 1); }
};

__device__ __forceinline__ KeyLayout make_layout(i64 N, u64 maxnb) {
    KeyLayout kl;
    kl.sbits = bits_for((u64)(N > 1 ? N - 1 : 1));
    for (int w = 32; w >= 1; --w) {
        int D = (64 + w - 1) / w;
        u64 LDmax = (u64)D * maxnb + D;
        int lbits = bits_for(3 * LDmax + 4);
        kl.w = w; kl.D = D; kl.LDmax = LDmax; kl.lbits = lbits;
        if (kl.sbits + lbits + w <= 64) break;
    }
    kl.total = kl.sbits + kl.lbits + kl.w;
    return kl;
}

__global__ void __launch_bounds__(GS_THREADS, 1) k_pending_tree(TreeArgs A) {
    __shared__ GsSmem ssm;
    __shared__ i64 s64[GS_WARPS + 2];
    const int lane = threadIdx.x & 31;
    const i64 N = A.N;
    const i64 gtid = (i64)blockIdx.x * GS_THREADS + threadIdx.x, gsize = (i64)gridDim.x * GS_THREADS;
    const i64 gwarp = gtid >> 5, nwarps = gsize >> 5;
    Grid g{&A.ctl->bar, 0};
    const u64* __restrict__ H = A.hashes;
    const i64* __restrict__ BO = A.blk_off;
    PEEK_MARK(1);

    // ---- phase 0: max chain length, initial state (one segment, everything "branch at 0") ----
    {
        u32 mx = 0;
        for (i64 r = gtid; r < N; r += gsize) {
            i64 nb = BO[r + 1] - BO[r];
            mx = max(mx, (u32)nb);
            A.bufs.val[0][r] = (u32)r;
        }
        mx = __reduce_max_sync(0xffffffffu, mx);
        if (lane == 0 && mx) atomicMax(&A.ctl->maxnb, mx);
        if (gtid == 0) { A.ctl->kand[0] = ~0ull; A.ctl->kand[1] = ~0ull; }
    }
    g.sync();
    const KeyLayout kl = make_layout(N, __ldcg(&A.ctl->maxnb));
    for (i64 r = gtid; r < N; r += gsize) A.bufs.key[0][r] = kl.pack(0, kl.f_before(0, false), 0);
    int cb = 0;  // buffer that holds the current (key, request) pairs by position

    for (int round = 0;; ++round) {
        // ---- R1: segment boundaries from equal keys, max-scan of segment starts, heads ----
        g.sync();  // keys / order of the previous phase visible
        PEEK_MARK(10);
        const u64* K = A.bufs.key[cb];
        const u32* cur = A.bufs.val[cb];
        u32* cnt = &A.ctl->unres[round % 3];
        if (gtid == 0) {
            A.ctl->unres[(round + 1) % 3] = 0;
            A.ctl->kor[(round + 1) & 1] = 0;
            A.ctl->kand[(round + 1) & 1] = ~0ull;
        }
        for (i64 j = gtid; j < N; j += gsize) {
            u64 kj = __ldcg(K + j);
            bool start = j == 0 || __ldcg(K + j - 1) != kj;
            if (start) {
                A.seghead[j] = 0;
                u64 F = kl.F_of(kj);
                A.segdepth[j] = kl.is_branch(F) ? (i32)(kl.ld_of(F) / kl.D) : 0;
            }
        }
        {
            auto load = [&](i64 j) -> i64 {
                bool start = j == 0 || __ldcg(K + j - 1) != __ldcg(K + j);
                return start ? j : 0;
            };
            auto store = [&](i64 j, i64 s) {
                u64 kj = __ldcg(K + j);
                bool start = j == 0 || __ldcg(K + j - 1) != kj;
                bool last = j == N - 1 || __ldcg(K + j + 1) != kj;
                bool unres = kl.is_branch(kl.F_of(kj)) && !(start && last);
                A.seg[j] = (u32)s | (unres ? 0x80000000u : 0u);
                // head = longest chain of the segment (lowest position on ties); one atomic per
                // warp when the whole warp sits in one unresolved segment (the common case)
                const unsigned act = __activemask();
                unsigned any = __ballot_sync(act, unres);
                u32 nb = 0;
                if (unres) {
                    u32 r = __ldcg(cur + j);
                    nb = (u32)(BO[r + 1] - BO[r]);
                }
                int same = 0;
                __match_all_sync(act, (u32)s, &same);
                if (same && any == act) {
                    u32 mnb = __reduce_max_sync(act, nb);
                    u32 mj = __reduce_max_sync(act, nb == mnb ? 0xffffffffu - (u32)j : 0u);
                    if (lane == (__ffs(act) - 1)) {
                        atomicAdd(cnt, (u32)__popc(any));
                        atomicMax((unsigned long long*)&A.seghead[s], ((u64)mnb << 32) | (u64)mj);
                    }
                } else if (unres) {
                    if (lane == (__ffs(any) - 1)) atomicAdd(cnt, (u32)__popc(any));
                    atomicMax((unsigned long long*)&A.seghead[s], ((u64)nb << 32) | (u64)(0xffffffffu - (u32)j));
                }
            };
            grid_inscan<i64>(N, load, store, [](i64 a, i64 b) { return a > b ? a : b; }, (i64)0, A.agg, s64, g);
        }
        PEEK_MARK(11);
        if (__ldcg(cnt) == 0) break;  // grid-uniform: read after the scan's final barrier

        // ---- R2: classify every unresolved position against its segment head (keys in place) ----
        {
            u64* Kw = A.bufs.key[cb];
            u64 orv = 0, andv = ~0ull;
            for (i64 j = gtid; j < N; j += gsize) {
                u32 sg = A.seg[j];
                u32 s = sg & 0x7fffffffu;
                u64 nk;
                if (!(sg >> 31)) {
                    nk = kl.pack(s, 0, 0);
                } else {
                    u32 r = __ldcg(cur + j);
                    u64 hv = __ldcg(A.seghead + s);
                    u32 hp = 0xffffffffu - (u32)hv;
                    i64 nbh = (i64)(hv >> 32);
                    u32 h = __ldcg(cur + hp);
                    i64 nbr = BO[r + 1] - BO[r];
                    const u64* cr = H + BO[r];
                    const u64* ch = H + BO[h];
                    i64 l = (r == h) ? nbr : chain_lcp(cr, nbr, ch, nbh, A.segdepth[s]);
                    u64 F, dig = 0;
                    if (l == nbr && l == nbh) F = kl.f_head();
                    else if (l == nbr) F = kl.f_before((u64)kl.D * l, true);
                    else {  // l < nbr <= nbh: the words at l differ
                        u64 a = __ldg(cr + l), b = __ldg(ch + l);
                        int jd = __clzll((long long)(a ^ b)) / kl.w;
                        u64 ld = (u64)kl.D * l + jd;
                        u64 da = (a << (jd * kl.w)) >> (64 - kl.w), db = (b << (jd * kl.w)) >> (64 - kl.w);
                        dig = da;
                        F = da < db ? kl.f_before(ld, false) : kl.f_after(ld);
                    }
                    nk = kl.pack(s, F, dig);
                }
                Kw[j] = nk;
                orv |= nk;
                andv &= nk;
            }
            const u32 olo = __reduce_or_sync(0xffffffffu, (u32)orv), ohi = __reduce_or_sync(0xffffffffu, (u32)(orv >> 32));
            const u32 alo = __reduce_and_sync(0xffffffffu, (u32)andv), ahi = __reduce_and_sync(0xffffffffu, (u32)(andv >> 32));
            if (lane == 0) {
                atomicOr(&A.ctl->kor[round & 1], ((unsigned long long)ohi << 32) | olo);
                atomicAnd(&A.ctl->kand[round & 1], ((unsigned long long)ahi << 32) | alo);
            }
        }
        g.sync();
        PEEK_MARK(12);

        // ---- R3: stable LSD radix sort of the pairs over the bits that vary ----
        const u64 vary = __ldcg(&A.ctl->kor[round & 1]) & ~__ldcg(&A.ctl->kand[round & 1]);
        cb = grid_sort_pairs(A.bufs, N, vary, g, ssm, cb);
        PEEK_MARK(13);
    }
    const u32* cur = A.bufs.val[cb];

    // ---- F1: final order into `order`, adjacent LCP ----
    for (i64 j = gtid; j < N; j += gsize) A.order[j] = (i32)cur[j];
    for (i64 j = gtid; j < N; j += gsize) {
        i32 l = 0;
        if (j > 0) {
            u32 a = cur[j - 1], b = cur[j];
            l = (i32)chain_lcp(H + BO[a], BO[a + 1] - BO[a], H + BO[b], BO[b + 1] - BO[b], 0);
        }
        A.lcp[j] = l;
    }
    PEEK_MARK(20);
    const bool want_groups = A.group_id || A.group_size || A.n_groups;
    const bool want_clusters = A.cluster_depth || A.cluster_size || A.cluster_id;
    if (!want_groups && !want_clusters) return;
    g.sync();

    // ---- F3: groups: sum-scan of (lcp == 0) flags and max-scan of their positions, packed ----
    if (want_groups) {
        auto op = [](i64 a, i64 b) -> i64 {
            i64 hs = (a >> 32) + (b >> 32);
            u32 la = (u32)a, lb = (u32)b;
            return (hs << 32) | (i64)(la > lb ? la : lb);
        };
        auto load = [&](i64 j) -> i64 { return __ldcg(A.lcp + j) == 0 ? (((i64)1 << 32) | j) : 0; };
        auto store = [&](i64 j, i64 v) {
            i32 gid = (i32)(v >> 32) - 1;
            i64 gstart = (u32)v;
            A.seg[j] = (u32)gid;
            bool last = j == N - 1 || __ldcg(A.lcp + j + 1) == 0;
            if (last) {
                A.gsz[gid] = (i32)(j - gstart + 1);
                if (j == N - 1 && A.n_groups) *A.n_groups = gid + 1;
            }
        };
        grid_inscan<i64>(N, load, store, op, (i64)0, A.agg, s64, g);
        for (i64 j = gtid; j < N; j += gsize) {
            u32 r = (u32)A.order[j];
            i32 gid = (i32)A.seg[j];
            if (A.group_id) A.group_id[r] = gid;
            if (A.group_size) A.group_size[r] = __ldcg(A.gsz + gid);
        }
    }
    PEEK_MARK(21);
    if (!want_clusters) return;

    // ---- F4: clusters by nearest-smaller-value searches on the LCP array ----
    MinTree mt;
    mintree_layout(mt, A.lcp, N, A.mt_buf);
    for (int k = 1; k < mt.levels; ++k) {
        mintree_build_level(mt, k, gwarp, nwarps, lane);
        g.sync();
    }
    for (i64 j = gtid; j < N; j += gsize) {
        u32 r = (u32)A.order[j];
        i32 l0 = A.lcp[j], l1 = j + 1 < N ? A.lcp[j + 1] : 0;
        i32 cd = l0 > l1 ? l0 : l1;
        i32 cs = 1;
        i64 cid = (i64)((u64)j << 32);
        if (cd > 0) {
            i64 a = nsv_prev_less(mt, j, cd);
            i64 b = nsv_next_less(mt, j + 1, cd) - 1;
            cs = (i32)(b - a + 1);
            cid = (i64)(((u64)a << 32) | (u64)(u32)cd);
        }
        if (A.cluster_depth) A.cluster_depth[r] = cd;
        if (A.cluster_size) A.cluster_size[r] = cs;
        if (A.cluster_id) A.cluster_id[r] = cid;
    }
    PEEK_MARK(22);
}


static void tree_layout(Arena& a, i64 N, int grid, TreeArgs& A) {
    A.ctl = a.take<TreeCtl>(1);
    A.bufs.key[0] = a.take<u64>(N);
    A.bufs.key[1] = a.take<u64>(N);
    A.bufs.val[0] = a.take<u32>(N);
    A.bufs.val[1] = a.take<u32>(N);
    A.bufs.hist = a.take<u32>(256 * (i64)grid);
    A.seg = a.take<u32>(N);
    A.seghead = a.take<u64>(N);
    A.segdepth = a.take<i32>(N);
    A.agg = a.take<i64>(grid);
    A.gsz = a.take<i32>(N);
    A.mt_buf = a.take<i32>(mintree_words(N));
}

static constexpr int MAX_GRID = 1024;  // upper bound on the cooperative grid (workspace sizing)

i64 pending_tree_ws_bytes(i64 N) {
    Arena a(nullptr);
    TreeArgs A;
    tree_layout(a, N, MAX_GRID, A);
    return a.used;
}

}  // namespace peek

using namespace peek;

extern "C" peek_status peek_pending_tree(const uint64_t* hashes, const int64_t* blk_off, int64_t N,
                                         int32_t* order, int32_t* lcp, int32_t* group_id,
                                         int32_t* group_size, int32_t* cluster_depth,
                                         int32_t* cluster_size, int64_t* cluster_id, int32_t* n_groups,
                                         void* ws, int64_t ws_bytes, void* stream) {
    if (N < 0 || N >= 0x7fffffffLL) { set_error("peek_pending_tree: N out of range"); return PEEK_ERR_INVALID_ARG; }
    if (N == 0) return PEEK_OK;
    if (!blk_off || !order || !lcp) { set_error("peek_pending_tree: NULL argument"); return PEEK_ERR_INVALID_ARG; }
    if (!ws || ((uintptr_t)ws & 255) || ws_bytes < pending_tree_ws_bytes(N)) {
        set_error("peek_pending_tree: workspace NULL, misaligned or too small");
        return PEEK_ERR_WORKSPACE;
    }
    cudaStream_t st = (cudaStream_t)stream;
    int grid = sm_count();  // one CTA of GS_THREADS per SM, all co-resident (cooperative launch)
    if (grid > MAX_GRID) grid = MAX_GRID;
    i64 want = (N + GS_THREADS - 1) / GS_THREADS;  // no point in more CTAs than work
    if (want < grid) grid = (int)(want < 1 ? 1 : want);
    Arena a(ws);
    TreeArgs A;
    A.hashes = hashes; A.blk_off = blk_off; A.N = N;
    A.order = order; A.lcp = lcp; A.group_id = group_id; A.group_size = group_size;
    A.cluster_depth = cluster_depth; A.cluster_size = cluster_size; A.cluster_id = cluster_id;
    A.n_groups = n_groups;
    tree_layout(a, N, MAX_GRID, A);
    PEEK_CUDA(cudaMemsetAsync(A.ctl, 0, sizeof(TreeCtl), st));
    void* params[] = {&A};
    Prof pr(PROF_TREE, st, 1);
    PEEK_CUDA(cudaLaunchCooperativeKernel((const void*)k_pending_tree, dim3(grid), dim3(GS_THREADS), params, 0, st));
    return PEEK_OK;
}

PEEK_TRACE_EXPORT(peek_trace_read_tree)
