// peek_tree.cu — a2-a4 peek_pending_tree: the pending radix tree built as
// a batch: lexicographic order of the requests' hash chains (= DFS order of the compressed trie),
// adjacent LCP (= its branching depths), flat groups and per-request clusters.
//
// ONE persistent cooperative kernel (one CTA of GS_THREADS per SM, grid barriers between phases),
// because the number of refinement rounds is data dependent and the call may not synchronise with
// the host.  The pairs (sort key, request) are kept BY POSITION and go through peek_sort.cuh's
// key/value sort; every phase walks the CTA's own chunk of positions in register tiles.
//
// Sort = path-peeling refinement.  Every unresolved segment (a run of sorted positions whose
// chains share a prefix) picks its LONGEST chain as head h.  A member r is classified by its
// LCP with h in units of w-bit digits (a 64-bit hash word = D digits, most significant first):
//     r proper prefix of h            -> before h, by ascending LCP, "ended" (identical chains)
//     r's digit < h's at the LCP      -> before h, by ascending LCP, then digit
//     r identical to h                -> with h
//     r's digit > h's at the LCP      -> after h, by DESCENDING LCP, then digit
// One stable LSD radix sort by key = [segment rank | class+LCP | digit] splits the segment along
// the whole root-to-leaf path of h at once, so rounds ~ 3 on the paper's workloads (shared
// prompt / conversation / turn) instead of one per trie level; only the key bits that vary are
// sorted on.  LCPs with the head use the chain property (k_i equal => all earlier words equal,
// DESIGN.md R15) to bisect for the first differing word; the probes are random 32-byte sectors of
// the hash array (the phase is HBM-transaction bound), so a warp row lets one lane bisect and the
// others verify its answer with one probe pair (lcp_lockstep).
// The ADJACENT LCP (output `lcp`) costs no chain reads at all: when a sort splits two neighbours
// that came from one segment, they leave the old head's path at known digit depths, and
// min(depths) / D is exactly their LCP (R1a); neighbours never split have identical chains.
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
    int signals_only;  // order and lcp are given: only groups and clusters are computed
    // workspace
    TreeCtl* ctl;
    GsBufs bufs;      // (sort key, request) by position, ping-pong
    u32* seg;         // N   by position: segment start | unresolved << 31
    u32* srank;       // N   by position: dense rank of the segment (the sort key's leading field)
    u64* lasth;       // N   by request: last word of its chain (read once; every round's first probe)
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
    __device__ __forceinline__ u64 seg_of(u64 key) const { return key >> (lbits + w); }
    // digits a member of class F shares with its segment head (the head itself: everything)
    __device__ __forceinline__ u64 ldv(u64 F) const {
        return (F <= 2 * LDmax + 1) ? (F >> 1) : (F == 2 * LDmax + 2 ? 2 * LDmax : LDmax - (F - (2 * LDmax + 3)));
    }
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

// ---- staged tile processing ---------------------------------------------------------------------
// Every phase walks the CTA's chunk of positions (the sort engine's ownership: CTA c owns
// [c0, c1), element (t, k) of thread (w, lane) is c0 + t*GS_TILE + w*32*GS_KPT + k*32 + lane) with
// GS_KPT elements per thread held in registers, and is written stage by stage: all loads of a
// stage are issued for the GS_KPT elements before any is used, so a phase costs (dependent stages)
// x (one memory round trip) instead of (elements per thread) x (stages) round trips.
#define ELEMS(k) _Pragma("unroll") for (int k = 0; k < GS_KPT; ++k)
// the register-hungry phases (lock-step searches) take the tile in sub-batches of SB elements
#ifndef PEEK_SB
#define PEEK_SB 1
#endif
static constexpr int SB = PEEK_SB;
#define SUBS(k) _Pragma("unroll") for (int k = 0; k < SB; ++k)

struct TreeSmem {
    i32 wv[GS_WARPS + 1];   // per-warp values of the carry chains
    i64 wv64[GS_WARPS + 1];
    i64 carry64;
    i32 carry;
    i32 lvl_hi[2048 + 64 + 8];  // per-CTA copy of the min-hierarchy levels >= 3
};

// LCP of K pairs of chains in lock step: chains H[ao..ao+na), H[bo..bo+nb), first lo words known
// equal (chain property R15: equal at a depth => equal above it, so the first difference is found
// by bisection).  act[k] selects the pairs to do; others keep res[k].
// Probes are random 32-byte sectors of a multi-GB array (the phase is bound by HBM transactions,
// not latency), so the search is organised to need few of them: (1) the last common word (one chain
// prefixes the other: done); (2) per warp row, ONE lane bisects and its answer g is the guess of
// the others (neighbours in sorted order mostly branch off their head at the same depth), who
// probe words g-1 and g - usually one sector - and (3) bisect on only if that did not settle it.
// HINT = false skips (2).  Must be called by full warps (uses warp collectives).
template <int K, bool HINT>
__device__ __forceinline__ void lcp_lockstep(const u64* __restrict__ H, const i64 (&ao)[K], const i32 (&na)[K],
                                             const i64 (&bo)[K], const i32 (&nb)[K], const i32 (&lo)[K],
                                             const bool (&act)[K], i32 (&res)[K], bool probe_lo,
                                             const u64 (&alast)[K]) {  // alast[k] = H[ao[k] + na[k] - 1]
    const unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    i32 L[K], R[K];  // while go: equal below/at L (L = lo - 1: nothing known), differ at R
    bool go[K];
    u64 x[K], y[K];
#pragma unroll
    for (int k = 0; k < K; ++k) {
        const i32 m = na[k] < nb[k] ? na[k] : nb[k];
        go[k] = act[k] && m > lo[k];
        if (act[k] && !go[k]) res[k] = m;
        L[k] = lo[k] - 1;
        R[k] = m - 1;
    }
    {   // first round trip: the last common word and - if the caller expects branches right at
        // lo (first round) - the first unknown word with it
        u64 x2[K], y2[K];
#pragma unroll
        for (int k = 0; k < K; ++k) {
            if (go[k]) {
                x[k] = R[k] == na[k] - 1 ? alast[k] : __ldg(H + ao[k] + R[k]);
                y[k] = __ldg(H + bo[k] + R[k]);
                if (probe_lo) { x2[k] = __ldg(H + ao[k] + lo[k]); y2[k] = __ldg(H + bo[k] + lo[k]); }
            }
        }
#pragma unroll
        for (int k = 0; k < K; ++k) {
            if (go[k]) {
                if (x[k] == y[k]) { res[k] = R[k] + 1; go[k] = false; }
                else if (probe_lo) {
                    if (x2[k] != y2[k]) { res[k] = lo[k]; go[k] = false; }
                    else L[k] = lo[k];
                }
                if (go[k] && R[k] - L[k] <= 1) { res[k] = R[k]; go[k] = false; }
            }
        }
    }
    // one bisection step for the elements selected by sel[k]; returns whether any is still going
    auto step = [&](const bool (&sel)[K]) -> bool {
#pragma unroll
        for (int k = 0; k < K; ++k) {
            if (go[k] && sel[k]) {
                const i32 p = (L[k] + R[k]) >> 1;
                x[k] = __ldg(H + ao[k] + p); y[k] = __ldg(H + bo[k] + p);
            }
        }
        bool any = false;
#pragma unroll
        for (int k = 0; k < K; ++k) {
            if (go[k] && sel[k]) {
                const i32 p = (L[k] + R[k]) >> 1;
                if (x[k] == y[k]) L[k] = p; else R[k] = p;
                if (R[k] - L[k] <= 1) { res[k] = R[k]; go[k] = false; }
                any |= go[k];
            }
        }
        return any;
    };
    bool all_sel[K];
#pragma unroll
    for (int k = 0; k < K; ++k) all_sel[k] = true;
    bool pending = false;
#pragma unroll
    for (int k = 0; k < K; ++k) pending |= go[k];
    if (HINT && __any_sync(FULL, pending)) {
        bool lead[K];
        int leader[K];
#pragma unroll
        for (int k = 0; k < K; ++k) {
            const unsigned bal = __ballot_sync(FULL, go[k]);
            leader[k] = bal ? __ffs(bal) - 1 : -1;
            lead[k] = lane == leader[k];
        }
        bool any = true;
        while (__any_sync(FULL, any)) any = step(lead);
        // the others probe around the leader's answer
#pragma unroll
        for (int k = 0; k < K; ++k) {
            const i32 gk = __shfl_sync(FULL, res[k], leader[k] < 0 ? 0 : leader[k]);
            const bool pr = go[k] && leader[k] >= 0;
            const bool p1 = pr && gk - 1 > L[k] && gk - 1 < R[k], p2 = pr && gk > L[k] && gk < R[k];
            if (p1) { x[k] = __ldg(H + ao[k] + gk - 1); y[k] = __ldg(H + bo[k] + gk - 1); }
            u64 x2 = 0, y2 = 0;
            if (p2) { x2 = __ldg(H + ao[k] + gk); y2 = __ldg(H + bo[k] + gk); }
            if (p1) { if (x[k] == y[k]) L[k] = gk - 1; else R[k] = gk - 1; }
            if (p2 && gk < R[k]) { if (x2 == y2) L[k] = gk; else R[k] = gk; }
            if (go[k] && R[k] - L[k] <= 1) { res[k] = R[k]; go[k] = false; }
        }
    }
    bool any = true;
    while (any) any = step(all_sel);
}

__global__ void __launch_bounds__(GS_THREADS, 1) k_pending_tree(TreeArgs A) {
    extern __shared__ __align__(16) unsigned char dyn_smem[];
    __shared__ GsSmem ssm;
    __shared__ TreeSmem tsm;
    const GsStage stg = gs_stage(dyn_smem);
    const unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const unsigned le_mask = 0xffffffffu >> (31 - lane);  // lanes <= this one
    const i64 N = A.N;
    const int G = gridDim.x, me = blockIdx.x;
    const i64 gtid = (i64)me * GS_THREADS + threadIdx.x;
    Grid g{&A.ctl->bar, 0};
    const u64* __restrict__ H = A.hashes;
    const i64* __restrict__ BO = A.blk_off;
    const i64 C = (N + G - 1) / G;
    const i64 c0 = min((i64)me * C, N), c1 = min(c0 + C, N);
    const int ntiles = (int)((C + GS_TILE - 1) / GS_TILE);
    auto IDX = [&](int t, int k) -> i64 { return c0 + (i64)t * GS_TILE + w * (32 * GS_KPT) + k * 32 + lane; };
    PEEK_MARK(1);

    if (!A.signals_only) {  // build order + lcp; otherwise they are inputs (peek_pending_tree_update)
    // ---- phase 0: max chain length, identity order ----
    {
        u32 mx = 0;
        for (int t = 0; t < ntiles; ++t) {
            i64 b0[GS_KPT], b1[GS_KPT];
            ELEMS(k) {
                const i64 i = IDX(t, k);
                b0[k] = b1[k] = 0;
                if (i < c1) { b0[k] = __ldg(BO + i); b1[k] = __ldg(BO + i + 1); A.bufs.val[0][i] = (u32)i; }
            }
            ELEMS(k) mx = max(mx, (u32)(b1[k] - b0[k]));
            // the last word of every chain, gathered once: a member's chain is never longer than
            // its head's, so the "does one chain prefix the other" probe of every round reads it
            u64 lw[GS_KPT];
            ELEMS(k) lw[k] = b1[k] > b0[k] ? __ldg(H + b1[k] - 1) : 0ull;
            ELEMS(k) { const i64 i = IDX(t, k); if (i < c1) A.lasth[i] = lw[k]; }
        }
        mx = __reduce_max_sync(FULL, mx);
        if (lane == 0 && mx) atomicMax(&A.ctl->maxnb, mx);
        if (gtid == 0) { A.ctl->kand[0] = ~0ull; A.ctl->kand[1] = ~0ull; }
    }
    g.sync();
    const KeyLayout kl = make_layout(N, __ldcg(&A.ctl->maxnb));
    {
        const u64 k_init = kl.pack(0, kl.f_before(0, false), 0);
        for (int t = 0; t < ntiles; ++t)
            ELEMS(k) { const i64 i = IDX(t, k); if (i < c1) A.bufs.key[0][i] = k_init; }
    }
    int cb = 0;  // buffer that holds the current (key, request) pairs by position

    for (int round = 0;; ++round) {
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
        // ---- R1a: segment starts (key differs from the left neighbour); last start per CTA ----
        {
            i32 cta_last = -1;
            u32 cta_cnt = 0;  // segment starts seen by this warp
            for (int t = 0; t < ntiles; ++t)
            for (int hb = 0; hb < GS_KPT / SB; ++hb) {
                u64 k0[SB], km[SB];
                SUBS(k) {
                    const i64 i = IDX(t, hb * SB + k);
                    k0[k] = km[k] = 0;
                    if (i < c1) { k0[k] = __ldcg(K + i); if (i > 0) km[k] = __ldcg(K + i - 1); }
                }
                SUBS(k) {
                    const i64 i = IDX(t, hb * SB + k);
                    const bool start = i < c1 && (i == 0 || km[k] != k0[k]);
                    const unsigned bal = __ballot_sync(FULL, start);
                    if (bal) cta_last = (i32)(i - lane) + 31 - __clz(bal);
                    cta_cnt += __popc(bal);
                    if (start) {
                        A.seghead[i] = 0;
                        const u64 F = kl.F_of(k0[k]);
                        A.segdepth[i] = kl.is_branch(F) ? (i32)(kl.ld_of(F) / kl.D) : 0;
                        // a boundary made by the last sort (both sides come from one segment): the
                        // two chains leave their old head's path at ldv digits, so they share
                        // exactly min(ldv) digits - the final adjacent LCP, no chain reads needed
                        if (i == 0) A.lcp[0] = 0;
                        else if (round > 0 && kl.seg_of(km[k]) == kl.seg_of(k0[k])) {
                            const u64 la = kl.ldv(kl.F_of(km[k])), lb = kl.ldv(F);
                            A.lcp[i] = (i32)((la < lb ? la : lb) / kl.D);
                        }
                    }
                }
            }
            if (lane == 0) tsm.wv64[w] = ((i64)cta_cnt << 32) | (u32)(cta_last + 1);
            __syncthreads();
            if (w == 0) {
                const i64 v = lane < GS_WARPS ? tsm.wv64[lane] : 0;
                const u32 cs = __reduce_add_sync(FULL, (u32)(v >> 32)), ls = __reduce_max_sync(FULL, (u32)v);
                if (lane == 0) A.agg[me] = ((i64)cs << 32) | ls;
            }
        }
        g.sync();
        // ---- R1b: segment start of every position, unresolved flag, head = longest chain ----
        {
            if (w == 0) {  // segment starts in the chunks before mine: how many, and the last one
                u32 cs = 0, ls = 0;
                for (int cbase = 0; cbase < me; cbase += 32 * 5) {
                    i64 x[5];
#pragma unroll
                    for (int q = 0; q < 5; ++q) { const int c = cbase + q * 32 + lane; x[q] = c < me ? __ldcg(A.agg + c) : 0; }
#pragma unroll
                    for (int q = 0; q < 5; ++q) { cs += (u32)(x[q] >> 32); ls = max(ls, (u32)x[q]); }
                }
                cs = __reduce_add_sync(FULL, cs);
                ls = __reduce_max_sync(FULL, ls);
                if (lane == 0) tsm.carry64 = ((i64)cs << 32) | ls;
            }
            __syncthreads();
            u32 n_unres = 0;
            u64 carry_v = 0;  // head candidate of the segment the warp's last full rows lay in
            i32 carry_s = 0;
            for (int t = 0; t < ntiles; ++t) {
                unsigned bal[GS_KPT];
                u32 fl[GS_KPT];  // bit 0 start, bit 1 last, bit 2 branch class
                u32 wl = 0, wc = 0;  // this warp's last segment start + 1, and how many it has
#pragma unroll
                for (int hb = 0; hb < GS_KPT / SB; ++hb) {
                    u64 k0[SB], km[SB], kp[SB];
                    SUBS(k) {
                        const i64 i = IDX(t, hb * SB + k);
                        k0[k] = km[k] = kp[k] = 0;
                        if (i < c1) {
                            k0[k] = __ldcg(K + i);
                            if (i > 0) km[k] = __ldcg(K + i - 1);
                            if (i + 1 < N) kp[k] = __ldcg(K + i + 1);
                        }
                    }
                    SUBS(k) {
                        const i64 i = IDX(t, hb * SB + k);
                        const bool valid = i < c1;
                        const bool start = valid && (i == 0 || km[k] != k0[k]);
                        const bool last = valid && (i == N - 1 || kp[k] != k0[k]);
                        const bool br = valid && kl.is_branch(kl.F_of(k0[k]));
                        const unsigned bl = __ballot_sync(FULL, start);
                        if (bl) wl = (u32)((i - lane) + 31 - __clz(bl)) + 1u;
                        wc += __popc(bl);
                        bal[hb * SB + k] = bl;
                        fl[hb * SB + k] = (start ? 1u : 0u) | (last ? 2u : 0u) | (br ? 4u : 0u);
                    }
                }
                if (lane == 0) tsm.wv64[w] = ((i64)wc << 32) | wl;
                __syncthreads();
                if (w == 0) {  // exclusive (sum, max) scan over the warps, seeded with the carry
                    const i64 own = lane < GS_WARPS ? tsm.wv64[lane] : 0;
                    u32 ic = (u32)(own >> 32), il = (u32)own;
#pragma unroll
                    for (int o = 1; o < 32; o <<= 1) {
                        const u32 xc = __shfl_up_sync(FULL, ic, o), xl = __shfl_up_sync(FULL, il, o);
                        if (lane >= o) { ic += xc; il = max(il, xl); }
                    }
                    u32 ec = __shfl_up_sync(FULL, ic, 1), el = __shfl_up_sync(FULL, il, 1);
                    if (lane == 0) { ec = 0; el = 0; }
                    const i64 cin = tsm.carry64;
                    if (lane < GS_WARPS) tsm.wv64[lane] = ((i64)(ec + (u32)(cin >> 32)) << 32) | max(el, (u32)cin);
                    if (lane == 31) tsm.carry64 = ((i64)(ic + (u32)(cin >> 32)) << 32) | max(il, (u32)cin);
                }
                __syncthreads();
                i32 c = (i32)(u32)tsm.wv64[w] - 1;     // last segment start before this warp's rows
                u32 cc = (u32)(tsm.wv64[w] >> 32);     // segment starts before this warp's rows
#pragma unroll
                for (int hb = 0; hb < GS_KPT / SB; ++hb) {
                    i32 sarr[SB];
                    bool un[SB];
                    u32 r[SB];
                    SUBS(k) {
                        const int kk = hb * SB + k;
                        const i64 i = IDX(t, kk);
                        const bool valid = i < c1;
                        const unsigned m = bal[kk] & le_mask;
                        const i32 s = m ? (i32)(i - lane) + 31 - __clz(m) : c;
                        if (bal[kk]) c = (i32)(i - lane) + 31 - __clz(bal[kk]);
                        const u32 rank = cc + __popc(m) - 1u;
                        cc += __popc(bal[kk]);
                        un[k] = valid && (fl[kk] & 4u) && (fl[kk] & 3u) != 3u;
                        sarr[k] = s;
                        if (valid) { A.seg[i] = (u32)s | (un[k] ? 0x80000000u : 0u); A.srank[i] = rank; }
                        r[k] = un[k] ? __ldcg(cur + i) : 0u;
                    }
                    i64 b0[SB], b1[SB];
                    SUBS(k) { b0[k] = b1[k] = 0; if (un[k]) { b0[k] = __ldg(BO + r[k]); b1[k] = __ldg(BO + r[k] + 1); } }
                    SUBS(k) {
                        // head = longest chain of the segment, lowest position on ties: segmented
                        // max over the row's runs of equal s, one atomic per run
                        const i64 i = IDX(t, hb * SB + k);
                        u64 v = un[k] ? (((u64)(u32)(b1[k] - b0[k]) << 32) | (u64)(0xffffffffu - (u32)i)) : 0ull;
                        const i32 s = sarr[k];
#pragma unroll
                        for (int o = 1; o < 32; o <<= 1) {
                            const u64 x = __shfl_up_sync(FULL, v, o);
                            const i32 sx = __shfl_up_sync(FULL, s, o);
                            if (lane >= o && sx == s && x > v) v = x;
                        }
                        const i32 s0 = __shfl_sync(FULL, s, 0), s31 = __shfl_sync(FULL, s, 31);
                        if (s0 == s31) {  // the whole row lies in one segment: keep its maximum in the
                                          // warp and post one atomic when the segment changes
                            const u64 v31 = __shfl_sync(FULL, v, 31);
                            if (carry_v && carry_s != s0) {
                                if (lane == 0) atomicMax((unsigned long long*)&A.seghead[carry_s], carry_v);
                                carry_v = 0;
                            }
                            carry_s = s0;
                            if (v31 > carry_v) carry_v = v31;
                        } else {
                            if (carry_v) {
                                if (lane == 0) atomicMax((unsigned long long*)&A.seghead[carry_s], carry_v);
                                carry_v = 0;
                            }
                            const i32 sn = __shfl_down_sync(FULL, s, 1);
                            if (v && (lane == 31 || sn != s)) atomicMax((unsigned long long*)&A.seghead[s], v);
                        }
                        n_unres += __popc(__ballot_sync(FULL, un[k]));
                    }
                }
                __syncthreads();  // tsm.wv is reused by the next tile
            }
            if (lane == 0 && carry_v) atomicMax((unsigned long long*)&A.seghead[carry_s], carry_v);
            if (lane == 0 && n_unres) atomicAdd(cnt, n_unres);
        }
        g.sync();
        PEEK_MARK(11);
        if (__ldcg(cnt) == 0) break;  // grid-uniform: read after the barrier

        // ---- R2: classify every unresolved position against its segment head (keys in place) ----
        {
            u64* Kw = A.bufs.key[cb];
            u64 orv = 0, andv = ~0ull;
            for (int t = 0; t < ntiles; ++t)
            for (int hb = 0; hb < GS_KPT / SB; ++hb) {
                u32 sg[SB], r[SB], h[SB], rk[SB];
                bool un[SB], cmp[SB];
                SUBS(k) {
                    const i64 i = IDX(t, hb * SB + k);
                    sg[k] = 0; r[k] = 0; rk[k] = 0;
                    if (i < c1) { sg[k] = A.seg[i]; r[k] = __ldcg(cur + i); rk[k] = A.srank[i]; }
                    un[k] = (sg[k] >> 31) != 0;
                }
                u64 hv[SB];
                i64 ao[SB], bo[SB];
                i32 na[SB], nb[SB], lo[SB], l[SB];
                SUBS(k) {
                    hv[k] = 0; ao[k] = 0; na[k] = 0; lo[k] = 0;
                    if (un[k]) {
                        const u32 s = sg[k] & 0x7fffffffu;
                        hv[k] = __ldcg(A.seghead + s);
                        lo[k] = __ldcg(A.segdepth + s);
                        ao[k] = __ldg(BO + r[k]);
                        na[k] = (i32)(__ldg(BO + r[k] + 1) - ao[k]);
                    }
                }
                SUBS(k) { h[k] = un[k] ? __ldcg(cur + (0xffffffffu - (u32)hv[k])) : 0u; nb[k] = (i32)(hv[k] >> 32); }
                SUBS(k) {
                    bo[k] = un[k] ? __ldg(BO + h[k]) : 0;
                    cmp[k] = un[k] && r[k] != h[k];
                    l[k] = na[k];  // r == h: the head itself
                }
                u64 al[SB];
                SUBS(k) al[k] = un[k] ? __ldcg(A.lasth + r[k]) : 0ull;
                lcp_lockstep<SB, true>(H, ao, na, bo, nb, lo, cmp, l, round == 0, al);
                u64 wa[SB], wb[SB];
                SUBS(k) {
                    wa[k] = wb[k] = 0;
                    if (un[k] && l[k] < na[k]) { wa[k] = __ldg(H + ao[k] + l[k]); wb[k] = __ldg(H + bo[k] + l[k]); }
                }
                SUBS(k) {
                    const i64 i = IDX(t, hb * SB + k);
                    if (i < c1) {
                        const u32 s = rk[k];  // dense segment rank: few leading key bits vary
                        u64 nk;
                        if (!un[k]) {
                            nk = kl.pack(s, 0, 0);
                        } else {
                            u64 F, dig = 0;
                            if (l[k] == na[k] && l[k] == nb[k]) F = kl.f_head();
                            else if (l[k] == na[k]) F = kl.f_before((u64)kl.D * l[k], true);
                            else {  // l < na <= nb: the words at l differ
                                const u64 a = wa[k], b = wb[k];
                                const int jd = __clzll((long long)(a ^ b)) / kl.w;
                                const u64 ld = (u64)kl.D * l[k] + jd;
                                const u64 da = (a << (jd * kl.w)) >> (64 - kl.w), db = (b << (jd * kl.w)) >> (64 - kl.w);
                                dig = da;
                                F = da < db ? kl.f_before(ld, false) : kl.f_after(ld);
                            }
                            nk = kl.pack(s, F, dig);
                        }
                        Kw[i] = nk;
                        orv |= nk;
                        andv &= nk;
                    }
                }
            }
            const u32 olo = __reduce_or_sync(FULL, (u32)orv), ohi = __reduce_or_sync(FULL, (u32)(orv >> 32));
            const u32 alo = __reduce_and_sync(FULL, (u32)andv), ahi = __reduce_and_sync(FULL, (u32)(andv >> 32));
            if (lane == 0) {
                atomicOr(&A.ctl->kor[round & 1], ((unsigned long long)ohi << 32) | olo);
                atomicAnd(&A.ctl->kand[round & 1], ((unsigned long long)ahi << 32) | alo);
            }
        }
        g.sync();
        PEEK_MARK(12);

        // ---- R3: stable LSD radix sort of the pairs over the bits that vary ----
        const u64 vary = __ldcg(&A.ctl->kor[round & 1]) & ~__ldcg(&A.ctl->kand[round & 1]);
        cb = grid_sort_pairs(A.bufs, N, vary, g, ssm, stg, cb);
        PEEK_MARK(13);
    }
    const u32* cur = A.bufs.val[cb];

    // ---- F1: final order.  The adjacent LCP of every segment boundary was written when the
    // boundary appeared (R1a); positions inside a final segment repeat their neighbour's chain ----
    {
        const u64* K = A.bufs.key[cb];
        for (int t = 0; t < ntiles; ++t) {
            u32 r[GS_KPT];
            bool same[GS_KPT];
            ELEMS(k) {
                const i64 i = IDX(t, k);
                r[k] = 0; same[k] = false;
                if (i < c1) {
                    r[k] = __ldcg(cur + i);
                    if (i > 0) same[k] = __ldcg(K + i) == __ldcg(K + i - 1);
                }
            }
            ELEMS(k) {
                const i64 i = IDX(t, k);
                if (i < c1) {
                    A.order[i] = (i32)r[k];
                    if (same[k]) A.lcp[i] = (i32)(__ldg(BO + r[k] + 1) - __ldg(BO + r[k]));
                }
            }
        }
    }
    }  // !signals_only
    PEEK_MARK(20);
    const bool want_groups = A.group_id || A.group_size || A.n_groups;
    const bool want_clusters = A.cluster_depth || A.cluster_size || A.cluster_id;
    if (!want_groups && !want_clusters) return;
    g.sync();
    MinTree mt;
    mintree_layout(mt, A.lcp, N, A.mt_buf);
    const i64 gwarp = gtid >> 5, nwarps = ((i64)G * GS_THREADS) >> 5;

    // ---- G1: per-CTA count of group starts (lcp == 0) and the last one; min-hierarchy level 1 ----
    {
        u32 cntw = 0;
        i32 lastw = -1;
        for (int t = 0; t < ntiles; ++t) {
            i32 lv[GS_KPT];
            ELEMS(k) { const i64 i = IDX(t, k); lv[k] = i < c1 ? __ldcg(A.lcp + i) : 1; }
            ELEMS(k) {
                const i64 i = IDX(t, k);
                const unsigned bal = __ballot_sync(FULL, lv[k] == 0);
                cntw += __popc(bal);
                if (bal) lastw = (i32)(i - lane) + 31 - __clz(bal);
            }
        }
        if (lane == 0) tsm.wv64[w] = ((i64)cntw << 32) | (u32)(lastw + 1);
        __syncthreads();
        if (w == 0) {
            const i64 v = lane < GS_WARPS ? tsm.wv64[lane] : 0;
            const u32 cs = __reduce_add_sync(FULL, (u32)(v >> 32)), ls = __reduce_max_sync(FULL, (u32)v);
            if (lane == 0) A.agg[me] = ((i64)cs << 32) | ls;
        }
        if (want_clusters && mt.levels > 1) mintree_build_level(mt, 1, gwarp, nwarps, lane);
    }
    g.sync();
    // ---- G2: group id / start of every position, group sizes; min-hierarchy level 2 ----
    {
        if (w == 0) {
            u32 cs = 0, ls = 0;
            for (int cbase = 0; cbase < me; cbase += 32 * 5) {
                i64 x[5];
#pragma unroll
                for (int q = 0; q < 5; ++q) { const int c = cbase + q * 32 + lane; x[q] = c < me ? __ldcg(A.agg + c) : 0; }
#pragma unroll
                for (int q = 0; q < 5; ++q) { cs += (u32)(x[q] >> 32); ls = max(ls, (u32)x[q]); }
            }
            cs = __reduce_add_sync(FULL, cs);
            ls = __reduce_max_sync(FULL, ls);
            if (lane == 0) tsm.carry64 = ((i64)cs << 32) | ls;
        }
        __syncthreads();
        for (int t = 0; t < ntiles; ++t) {
            i32 lv[GS_KPT], ln[GS_KPT];
            unsigned bal[GS_KPT];
            ELEMS(k) {
                const i64 i = IDX(t, k);
                lv[k] = 1; ln[k] = 0;
                if (i < c1) { lv[k] = __ldcg(A.lcp + i); if (i + 1 < N) ln[k] = __ldcg(A.lcp + i + 1); }
            }
            u32 cntw = 0, lastw = 0;
            ELEMS(k) {
                const i64 i = IDX(t, k);
                bal[k] = __ballot_sync(FULL, lv[k] == 0);
                cntw += __popc(bal[k]);
                if (bal[k]) lastw = (u32)((i - lane) + 31 - __clz(bal[k])) + 1u;
            }
            if (lane == 0) tsm.wv64[w] = ((i64)cntw << 32) | lastw;
            __syncthreads();
            if (w == 0) {  // exclusive (sum, max) scan over the warps, seeded with the carry
                const i64 own = lane < GS_WARPS ? tsm.wv64[lane] : 0;
                u32 ic = (u32)(own >> 32), il = (u32)own;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const u32 xc = __shfl_up_sync(FULL, ic, o), xl = __shfl_up_sync(FULL, il, o);
                    if (lane >= o) { ic += xc; il = max(il, xl); }
                }
                u32 ec = __shfl_up_sync(FULL, ic, 1), el = __shfl_up_sync(FULL, il, 1);
                if (lane == 0) { ec = 0; el = 0; }
                const i64 cin = tsm.carry64;
                if (lane < GS_WARPS) tsm.wv64[lane] = ((i64)(ec + (u32)(cin >> 32)) << 32) | max(el, (u32)cin);
                if (lane == 31) tsm.carry64 = ((i64)(ic + (u32)(cin >> 32)) << 32) | max(il, (u32)cin);
            }
            __syncthreads();
            u32 cc = (u32)(tsm.wv64[w] >> 32), cl = (u32)tsm.wv64[w];
            ELEMS(k) {
                const i64 i = IDX(t, k);
                const unsigned m = bal[k] & le_mask;
                const i32 gid = (i32)(cc + __popc(m)) - 1;
                const i64 gstart = m ? (i - lane) + 31 - __clz(m) : (i64)cl - 1;
                cc += __popc(bal[k]);
                if (bal[k]) cl = (u32)((i - lane) + 31 - __clz(bal[k])) + 1u;
                if (i < c1) {
                    A.seg[i] = (u32)gid;
                    if (i == N - 1 || ln[k] == 0) {
                        A.gsz[gid] = (i32)(i - gstart + 1);
                        if (i == N - 1 && A.n_groups) *A.n_groups = gid + 1;
                    }
                }
            }
            __syncthreads();
        }
        if (want_clusters && mt.levels > 2) mintree_build_level(mt, 2, gwarp, nwarps, lane);
    }
    g.sync();
    // ---- min-hierarchy levels >= 3: a private copy per CTA in shared memory when they fit ----
    if (want_clusters && mt.levels > 3) {
        if (mt.n[3] <= 2048) {
            int off = 0;
            for (int k = 3; k < mt.levels; ++k) {
                mt.lvl[k] = tsm.lvl_hi + off;
                off += k == 3 ? 2048 : (k == 4 ? 64 : 2);
            }
            for (int k = 3; k < mt.levels; ++k) {
                mintree_build_level(mt, k, (i64)w, (i64)GS_WARPS, lane);
                __syncthreads();
            }
        } else {
            for (int k = 3; k < mt.levels; ++k) {
                mintree_build_level(mt, k, gwarp, nwarps, lane);
                g.sync();
            }
        }
    }
    PEEK_MARK(21);
    // ---- G3: group outputs; clusters by nearest-smaller-value walks on the LCP array, in lock step ----
    for (int t = 0; t < ntiles; ++t)
    for (int hb = 0; hb < GS_KPT / SB; ++hb) {
        u32 r[SB];
        i32 gid[SB], l0[SB], l1[SB];
        SUBS(k) {
            const i64 i = IDX(t, hb * SB + k);
            r[k] = 0; gid[k] = 0; l0[k] = 0; l1[k] = 0;
            if (i < c1) {
                r[k] = (u32)A.order[i];
                if (want_groups) gid[k] = (i32)A.seg[i];
                l0[k] = __ldcg(A.lcp + i);
                if (i + 1 < N) l1[k] = __ldcg(A.lcp + i + 1);
            }
        }
        if (want_groups) {
            i32 gs[SB];
            SUBS(k) { const i64 i = IDX(t, hb * SB + k); gs[k] = i < c1 ? __ldcg(A.gsz + gid[k]) : 0; }
            SUBS(k) {
                const i64 i = IDX(t, hb * SB + k);
                if (i < c1) {
                    if (A.group_id) A.group_id[r[k]] = gid[k];
                    if (A.group_size) A.group_size[r[k]] = gs[k];
                }
            }
        }
        if (!want_clusters) continue;
        i32 cd[SB];
        i64 pa[SB], pb[SB];
        int lv[SB];
        bool go[SB];
        // a = largest p <= i with L0x[p] < cd
        bool any = false;
        SUBS(k) {
            const i64 i = IDX(t, hb * SB + k);
            cd[k] = l0[k] > l1[k] ? l0[k] : l1[k];
            go[k] = i < c1 && cd[k] > 0;
            pa[k] = i; lv[k] = 0;
            if (go[k] && l0[k] < cd[k]) go[k] = false;  // the position itself (value already at hand)
            else if (go[k]) { if ((i & 31) == 0) { pa[k] = (i >> 5) - 1; lv[k] = 1; } else pa[k] = i - 1; }
            any |= go[k];
        }
        // Most runs are short: the 32 positions of this warp row, the row before and the row after
        // sit in three registers per lane, and a lane scans its neighbours with shuffles; only
        // the searches that leave that window fall through to the walk on the min hierarchy.
        i32 w_prev = 0, w_cur = 0, w_next = 0;
        if (SB == 1) {
            const i64 i = IDX(t, hb * SB);
            w_cur = i < N ? __ldcg(A.lcp + i) : 0;
            w_next = i + 32 < N ? __ldcg(A.lcp + i + 32) : 0;
            w_prev = i >= 32 ? __ldcg(A.lcp + i - 32) : 0;
            bool g0 = go[0];
            for (int d = 1; d < 64 && __any_sync(FULL, g0); ++d) {
                const int idx = lane - d;
                const i32 x0 = __shfl_sync(FULL, w_cur, idx & 31), xu = __shfl_sync(FULL, w_prev, idx & 31);
                if (g0 && idx >= -32 && (idx >= 0 ? x0 : xu) < cd[0]) { pa[0] = (i - lane) + idx; g0 = false; }
            }
            if (go[0] && g0) { pa[0] = (i - lane) - 33; lv[0] = 0; }  // left the window (index >= 0 then)
            go[0] = g0;
            any = g0;
        }
        while (any) {
            i32 v[SB];
            SUBS(k) v[k] = go[k] ? mt.val(lv[k], pa[k]) : 0;
            any = false;
            SUBS(k) {
                if (go[k]) {
                    if (v[k] < cd[k]) {
                        if (lv[k] == 0) go[k] = false;
                        else { --lv[k]; pa[k] = min(pa[k] * 32 + 31, mt.n[lv[k]] - 1); }
                    } else if ((pa[k] & 31) == 0) { pa[k] = (pa[k] >> 5) - 1; ++lv[k]; }
                    else --pa[k];
                }
                any |= go[k];
            }
        }
        // b + 1 = smallest q >= i + 1 with L0x[q] < cd
        any = false;
        SUBS(k) {
            const i64 i = IDX(t, hb * SB + k);
            go[k] = i < c1 && cd[k] > 0;
            pb[k] = i + 1; lv[k] = 0;
            if (go[k] && l1[k] < cd[k]) go[k] = false;  // position i + 1 itself
            else if (go[k]) {
                if (((i + 1) & 31) == 31 || i + 1 == mt.n[0] - 1) { pb[k] = ((i + 1) >> 5) + 1; lv[k] = 1; } else pb[k] = i + 2;
            }
            any |= go[k];
        }
        if (SB == 1) {
            const i64 i = IDX(t, hb * SB);
            bool g0 = go[0];
            for (int d = 1; d < 64 && __any_sync(FULL, g0); ++d) {
                const int idx = lane + d;
                const i32 x0 = __shfl_sync(FULL, w_cur, idx & 31), xn = __shfl_sync(FULL, w_next, idx & 31);
                if (g0 && idx < 64 && (idx < 32 ? x0 : xn) < cd[0]) { pb[0] = (i - lane) + idx; g0 = false; }
            }
            if (go[0] && g0) { pb[0] = (i - lane) + 64; lv[0] = 0; }  // left the window (index <= N then)
            go[0] = g0;
            any = g0;
        }
        while (any) {
            i32 v[SB];
            SUBS(k) v[k] = go[k] ? mt.val(lv[k], pb[k]) : 0;
            any = false;
            SUBS(k) {
                if (go[k]) {
                    if (v[k] < cd[k]) {
                        if (lv[k] == 0) go[k] = false;
                        else { --lv[k]; pb[k] = pb[k] * 32; }
                    } else if ((pb[k] & 31) == 31 || pb[k] == mt.n[lv[k]] - 1) { pb[k] = (pb[k] >> 5) + 1; ++lv[k]; }
                    else ++pb[k];
                }
                any |= go[k];
            }
        }
        SUBS(k) {
            const i64 i = IDX(t, hb * SB + k);
            if (i < c1) {
                i32 cs = 1;
                i64 cid = (i64)((u64)i << 32);
                if (cd[k] > 0) {
                    cs = (i32)(pb[k] - pa[k]);
                    cid = (i64)(((u64)pa[k] << 32) | (u64)(u32)cd[k]);
                }
                if (A.cluster_depth) A.cluster_depth[r[k]] = cd[k];
                if (A.cluster_size) A.cluster_size[r[k]] = cs;
                if (A.cluster_id) A.cluster_id[r[k]] = cid;
            }
        }
    }
    PEEK_MARK(22);
}

static void tree_layout(Arena& a, i64 N, int grid, TreeArgs& A) {
    A.ctl = a.take<TreeCtl>(1);
    A.bufs.hist = a.take<u32>(gs_hist_words(grid));  // directly after ctl: one memset clears both
    A.bufs.key[0] = a.take<u64>(N);
    A.bufs.key[1] = a.take<u64>(N);
    A.bufs.val[0] = a.take<u32>(N);
    A.bufs.val[1] = a.take<u32>(N);
    A.seg = a.take<u32>(N);
    A.srank = a.take<u32>(N);
    A.lasth = a.take<u64>(N);
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

// enqueue k_pending_tree (build, or signals only on a given order + lcp); ws holds pending_tree_ws_bytes(N)
static peek_status tree_launch(const u64* hashes, const i64* blk_off, i64 N, i32* order, i32* lcp,
                               i32* group_id, i32* group_size, i32* cluster_depth, i32* cluster_size,
                               i64* cluster_id, i32* n_groups, int signals_only, void* ws, cudaStream_t st) {
    int grid = persistent_ctas();  // one CTA of GS_THREADS per SM, all co-resident (cooperative launch)
    if (grid > MAX_GRID) grid = MAX_GRID;
    i64 want = (N + GS_THREADS - 1) / GS_THREADS;  // no point in more CTAs than work
    if (want < grid) grid = (int)(want < 1 ? 1 : want);
    Arena a(ws);
    TreeArgs A;
    A.hashes = hashes; A.blk_off = blk_off; A.N = N;
    A.order = order; A.lcp = lcp; A.group_id = group_id; A.group_size = group_size;
    A.cluster_depth = cluster_depth; A.cluster_size = cluster_size; A.cluster_id = cluster_id;
    A.n_groups = n_groups;
    A.signals_only = signals_only;
    tree_layout(a, N, MAX_GRID, A);
    PEEK_CUDA(cudaMemsetAsync(A.ctl, 0, (size_t)((char*)(A.bufs.hist + gs_hist_words(MAX_GRID)) - (char*)A.ctl), st));
    void* params[] = {&A};
    Prof pr(PROF_TREE, st, 1);
    static bool attr_set = false;
    if (!attr_set) {
        PEEK_CUDA(cudaFuncSetAttribute(k_pending_tree, cudaFuncAttributeMaxDynamicSharedMemorySize, GS_STAGE_BYTES));
        attr_set = true;
    }
    PEEK_CUDA(cudaLaunchCooperativeKernel((const void*)k_pending_tree, dim3(grid), dim3(GS_THREADS), params,
                                          GS_STAGE_BYTES, st));
    return PEEK_OK;
}

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
    return tree_launch(hashes, blk_off, N, order, lcp, group_id, group_size, cluster_depth, cluster_size,
                       cluster_id, n_groups, 0, ws, (cudaStream_t)stream);
}

// ---- a13 peek_pending_tree_update: incremental maintenance -----------------
// the paper keeps its pending tree incrementally (insert / remove O(D) per
// request) instead of rebuilding it every cycle.  Here the tree is (order, lcp); a cycle's delta -
// some requests admitted (removed), M arrivals appended - is applied without sorting the survivors:
//   1  compaction: the survivors keep their relative order; the LCP across a run of removed
//      positions is the minimum over the run (an ordered segmented-min scan)
//   2  the M arrivals are sorted among themselves by the batch build (k_pending_tree on M requests)
//   3  merge: every arrival bisects for its place among the survivors (chain comparisons by the
//      depth bisection of chain_lcp) and learns its LCP with both neighbours
//   4  placement: a prefix sum of the insertion counts shifts the survivors; every adjacent LCP
//      of the merged order is one of: the compacted LCP, a batch LCP, or a neighbour LCP from 3
//   5  groups and clusters from the merged (order, lcp): k_pending_tree in signals-only mode
// The result is by construction what peek_pending_tree returns on the new queue (the parity tests
// compare it with the oracle's rebuild).
namespace peek {

struct UpdCtl { u32 bar, pad; i64 S; };
struct UpdArgs {
    const u64* hashes;
    const i64* blk_off;
    i64 N_old, N_new, M;
    const i32 *old_order, *old_lcp, *remap;
    i32 *order, *lcp;
    UpdCtl* ctl;
    i32 *s_order, *s_lcp;        // survivors, compacted (<= N_old)
    const i32 *b_order, *b_lcp;  // the arrivals' own tree (M), local indices
    i32 *ins, *lcpL, *lcpR;      // per arrival: survivors before it, LCP with the survivor on either side
    i64* hist;                   // N_old + 1: arrivals inserted directly before survivor p (p = S: at the end)
    i32* rfix;                   // N_old + 1: LCP of survivor p with the arrival directly before it
    u64* agg;                    // gridDim scratch of the grid scans
};

// ordered grid-wide inclusive scan (associative op, NOT necessarily commutative)
template <typename T, typename Op, typename Load, typename Store>
__device__ void grid_inscan_ordered(i64 n, Load load, Store store, Op op, T ident, T* agg, T* smem, Grid& g) {
    const i64 chunk = (((n + gridDim.x - 1) / gridDim.x) + blockDim.x - 1) / blockDim.x * blockDim.x;
    const i64 c0 = min((i64)blockIdx.x * chunk, n), c1 = min(c0 + chunk, n);
    T carry = ident;
    for (i64 b = c0; b < c1; b += blockDim.x) {
        const i64 i = b + threadIdx.x;
        T tt;
        block_inscan(i < c1 ? load(i) : ident, op, ident, smem, &tt);
        carry = op(carry, tt);
    }
    if (threadIdx.x == 0) agg[blockIdx.x] = carry;
    g.sync();
    {   // what the chunks before mine add up to, in order: a contiguous slice of them per thread
        const int per = ((int)blockIdx.x + (int)blockDim.x - 1) / (int)blockDim.x;
        T acc = ident;
        for (int c = (int)threadIdx.x * per; c < min(((int)threadIdx.x + 1) * per, (int)blockIdx.x); ++c) acc = op(acc, agg[c]);
        block_inscan(acc, op, ident, smem, &carry);
    }
    for (i64 b = c0; b < c1; b += blockDim.x) {
        const i64 i = b + threadIdx.x;
        T tt;
        const T inc = block_inscan(i < c1 ? load(i) : ident, op, ident, smem, &tt);
        if (i < c1) store(i, op(carry, inc));
        carry = op(carry, tt);
    }
    g.sync();
}

// survivors kept so far | min LCP since the last kept position | "a segment starts here" flag
__device__ __forceinline__ u64 upd_pack(u32 cnt, u32 mn, u32 flag) { return ((u64)cnt << 32) | ((u64)mn << 1) | flag; }
__device__ __forceinline__ u64 upd_op(u64 a, u64 b) {
    const u32 cnt = (u32)(a >> 32) + (u32)(b >> 32);
    const u32 am = (u32)(a & 0xffffffffu) >> 1, bm = (u32)(b & 0xffffffffu) >> 1;
    if (b & 1) return ((u64)cnt << 32) | ((u64)bm << 1) | 1u;
    return ((u64)cnt << 32) | ((u64)(am < bm ? am : bm) << 1) | (a & 1);
}

// order of an arrival x against a survivor y: -1 x first, +1 y first (ties: the survivor, whose
// request index is smaller); *l = their LCP in blocks
__device__ __forceinline__ int upd_cmp(const u64* __restrict__ H, const i64* __restrict__ BO, i64 x, i64 y, i32* l) {
    const i64 bx = BO[x], nx = BO[x + 1] - bx, by = BO[y], ny = BO[y + 1] - by;
    const i64 m = chain_lcp(H + bx, nx, H + by, ny, 0);
    *l = (i32)m;
    if (m == ny) return 1;   // y is a prefix of x, or equal
    if (m == nx) return -1;  // x is a proper prefix of y
    return __ldg(H + bx + m) < __ldg(H + by + m) ? -1 : 1;
}

static constexpr int UP_THREADS = 512;

__global__ void __launch_bounds__(UP_THREADS) k_tree_update(UpdArgs A) {
    __shared__ u64 s64[UP_THREADS / 32 + 2];
    Grid g{&A.ctl->bar, 0};
    const i64 gtid = (i64)blockIdx.x * UP_THREADS + threadIdx.x, gsize = (i64)gridDim.x * UP_THREADS;
    const u64* __restrict__ H = A.hashes;
    const i64* __restrict__ BO = A.blk_off;
    // ---- 1: compaction of the survivors ----
    for (i64 p = gtid; p <= A.N_old; p += gsize) { A.hist[p] = 0; A.rfix[p] = -1; }
    if (gtid == 0) A.ctl->S = 0;
    {
        auto keep = [&](i64 j) -> bool { return __ldg(A.remap + __ldg(A.old_order + j)) >= 0; };
        auto load = [&](i64 j) -> u64 {
            return upd_pack(keep(j) ? 1u : 0u, (u32)__ldg(A.old_lcp + j), (j == 0 || keep(j - 1)) ? 1u : 0u);
        };
        auto store = [&](i64 j, u64 v) {
            if (keep(j)) {
                const i64 ps = (i64)(v >> 32) - 1;
                A.s_order[ps] = __ldg(A.remap + __ldg(A.old_order + j));
                A.s_lcp[ps] = (i32)((u32)(v & 0xffffffffu) >> 1);
            }
            if (j == A.N_old - 1) A.ctl->S = (i64)(v >> 32);
        };
        grid_inscan_ordered<u64>(A.N_old, load, store, [](u64 a, u64 b) { return upd_op(a, b); },
                                 upd_pack(0, 0x7fffffffu, 0), A.agg, s64, g);
    }
    const i64 S = A.N_old > 0 ? __ldcg(&A.ctl->S) : 0;
    // ---- 3: every arrival bisects for its place among the survivors ----
    const i64 first_new = A.N_new - A.M;
    for (i64 q = gtid; q < A.M; q += gsize) {
        const i64 x = first_new + __ldg(A.b_order + q);
        i64 lo = 0, hi = S;
        while (lo < hi) {  // survivors before lo sort at or before x, from hi on after x
            const i64 mid = (lo + hi) >> 1;
            i32 l;
            if (upd_cmp(H, BO, x, __ldcg(A.s_order + mid), &l) > 0) lo = mid + 1; else hi = mid;
        }
        i32 lL = 0, lR = 0;
        if (lo > 0) upd_cmp(H, BO, x, __ldcg(A.s_order + lo - 1), &lL);
        if (lo < S) upd_cmp(H, BO, x, __ldcg(A.s_order + lo), &lR);
        A.ins[q] = (i32)lo; A.lcpL[q] = lL; A.lcpR[q] = lR;
        atomicAdd((unsigned long long*)(A.hist + lo), 1ull);
    }
    g.sync();
    // ---- 4: placement ----
    for (i64 q = gtid; q < A.M; q += gsize) {
        const i32 in = A.ins[q];
        const i64 pos = (i64)in + q;
        A.order[pos] = (i32)(first_new + __ldg(A.b_order + q));
        A.lcp[pos] = (q > 0 && A.ins[q - 1] == in) ? __ldg(A.b_lcp + q) : A.lcpL[q];
        if (q == A.M - 1 || A.ins[q + 1] != in) A.rfix[in] = A.lcpR[q];  // the arrival right before survivor `in`
    }
    {
        auto load = [&](i64 p) -> u64 { return (u64)__ldcg(A.hist + p); };
        auto store = [&](i64 p, u64 inc) {
            if (p < S) {
                const i64 pos = p + (i64)inc;
                A.order[pos] = __ldcg(A.s_order + p);
                const i32 fix = __ldcg(A.rfix + p);
                A.lcp[pos] = fix >= 0 ? fix : __ldcg(A.s_lcp + p);
            }
        };
        grid_inscan_ordered<u64>(S + 1, load, store, [](u64 a, u64 b) { return a + b; }, (u64)0, A.agg, s64, g);
    }
}

struct UpdWs { UpdArgs A; i32 *b_order, *b_lcp; void* tree_ws; };
static void update_layout(Arena& a, i64 N_old, i64 N_new, i64 M, UpdWs& W) {
    UpdArgs& A = W.A;
    A.ctl = a.take<UpdCtl>(1);
    A.s_order = a.take<i32>(N_old); A.s_lcp = a.take<i32>(N_old);
    W.b_order = a.take<i32>(M); W.b_lcp = a.take<i32>(M);
    A.ins = a.take<i32>(M); A.lcpL = a.take<i32>(M); A.lcpR = a.take<i32>(M);
    A.hist = a.take<i64>(N_old + 1);
    A.rfix = a.take<i32>(N_old + 1);
    A.agg = a.take<u64>(MAX_GRID);
    W.tree_ws = a.take<char>(pending_tree_ws_bytes(N_new > M ? N_new : M));
}
i64 pending_tree_update_ws_bytes(i64 N_old, i64 N_new, i64 M) {
    Arena a(nullptr);
    UpdWs W;
    update_layout(a, N_old, N_new, M, W);
    return a.used;
}

}  // namespace peek

using namespace peek;

extern "C" peek_status peek_pending_tree_update(const uint64_t* hashes, const int64_t* blk_off, int64_t N_new,
                                                int64_t M, const int32_t* old_order, const int32_t* old_lcp,
                                                int64_t N_old, const int32_t* remap, int32_t* order,
                                                int32_t* lcp, int32_t* group_id, int32_t* group_size,
                                                int32_t* cluster_depth, int32_t* cluster_size,
                                                int64_t* cluster_id, int32_t* n_groups, void* ws,
                                                int64_t ws_bytes, void* stream) {
    if (N_new < 0 || N_new >= 0x7fffffffLL || N_old < 0 || N_old >= 0x7fffffffLL || M < 0 || M > N_new) {
        set_error("peek_pending_tree_update: sizes out of range");
        return PEEK_ERR_INVALID_ARG;
    }
    if (N_new == 0) return PEEK_OK;
    if (!blk_off || !order || !lcp || (N_old > 0 && (!old_order || !old_lcp || !remap))) {
        set_error("peek_pending_tree_update: NULL argument");
        return PEEK_ERR_INVALID_ARG;
    }
    if (!ws || ((uintptr_t)ws & 255) || ws_bytes < pending_tree_update_ws_bytes(N_old, N_new, M)) {
        set_error("peek_pending_tree_update: workspace NULL, misaligned or too small");
        return PEEK_ERR_WORKSPACE;
    }
    cudaStream_t st = (cudaStream_t)stream;
    Arena a(ws);
    UpdWs W;
    update_layout(a, N_old, N_new, M, W);
    if (M > 0) {  // the arrivals' own tree: their chains are requests N_new - M .. N_new - 1
        peek_status rc = tree_launch(hashes, blk_off + (N_new - M), M, W.b_order, W.b_lcp, nullptr, nullptr,
                                     nullptr, nullptr, nullptr, nullptr, 0, W.tree_ws, st);
        if (rc != PEEK_OK) return rc;
    }
    UpdArgs& A = W.A;
    A.hashes = hashes; A.blk_off = blk_off; A.N_old = N_old; A.N_new = N_new; A.M = M;
    A.old_order = old_order; A.old_lcp = old_lcp; A.remap = remap; A.order = order; A.lcp = lcp;
    A.b_order = W.b_order; A.b_lcp = W.b_lcp;
    PEEK_CUDA(cudaMemsetAsync(A.ctl, 0, sizeof(UpdCtl), st));
    int grid = persistent_ctas();
    if (grid > MAX_GRID) grid = MAX_GRID;
    i64 want = ((N_old > M ? N_old : M) + UP_THREADS - 1) / UP_THREADS;
    if (want < grid) grid = (int)(want < 1 ? 1 : want);
    {
        void* params[] = {&A};
        Prof pr(PROF_TREE, st, 1);
        PEEK_CUDA(cudaLaunchCooperativeKernel((const void*)k_tree_update, dim3(grid), dim3(UP_THREADS), params, 0, st));
    }
    if (group_id || group_size || n_groups || cluster_depth || cluster_size || cluster_id)
        return tree_launch(hashes, blk_off, N_new, order, lcp, group_id, group_size, cluster_depth, cluster_size,
                           cluster_id, n_groups, 1, W.tree_ws, st);
    return PEEK_OK;
}

PEEK_TRACE_EXPORT(peek_trace_read_tree)
