// peek_tree.cu — a2-a4 peek_pending_tree: the pending radix tree built as
// a batch: lexicographic order of the requests' hash chains (= DFS order of the compressed trie),
// adjacent LCP (= its branching depths), flat groups and per-request clusters.
//
// Two stages, three kernels on one stream (k_tree_global -> k_tree_local -> k_tree_signals):
//   GLOBAL stage (cooperative, one CTA of GS_THREADS per SM) - grid-wide partition.  Round 0 sorts the
//     requests by the leading bits of their first hash word (stable LSD pair sort of
//     peek_sort.cuh); further grid-wide rounds of the refinement below run only while some
//     unresolved segment is larger than what one CTA should finish alone (cap_seg positions).
//   LOCAL stage (persistent, no CTA waits for another) - every unresolved segment (a run of sorted
//     positions whose chains share a prefix and are not ordered yet) is finished by ONE CTA out of
//     shared memory: all further refinement rounds, their sorts and their scans cost CTA barriers
//     instead of grid barriers, and segments are independent, so the tail of one does not hold up
//     the others.  Work items are handed out through two atomic queues (the segments above the
//     quantum first, then fixed quanta of positions holding the small ones); which CTA takes
//     which item never changes a result.  A work item occupies one SM, so cap_seg and the quantum
//     scale with the queue (tree_launch): mid-size queues get enough items to fill the GPU.
//   SIGNALS (cooperative) - groups and clusters from (order, lcp).
//   Queues of at most TREE_SMALL_MAX requests (the paper's hold 60-200) run in one CTA
//   and one launch from the first step on (k_tree_small) and see no grid barrier at all.
//
// Refinement = path peeling.  Every unresolved segment picks its LONGEST chain as head h.  A member
// r is classified by its LCP with h in units of w-bit digits (a 64-bit hash word = D digits, most
// significant first):
//     r proper prefix of h            -> before h, by ascending LCP, "ended" (identical chains)
//     r's digit < h's at the LCP      -> before h, by ascending LCP, then digit
//     r identical to h                -> with h
//     r's digit > h's at the LCP      -> after h, by DESCENDING LCP, then digit
// One stable LSD radix sort by key = [segment rank | class+LCP | digit] splits the segment along
// the whole root-to-leaf path of h at once, so rounds ~ 3 on the paper's workloads (shared
// prompt / conversation / turn) instead of one per trie level; only the key bits that vary are
// sorted on.  Round 0 is the same thing against a virtual head that is smaller than every chain
// (class "after, LCP 0", digit = leading bits of the first word): no head, no probes.
// LCPs with the head use the chain property (k_i equal => all earlier words equal, R15)
// to bisect for the first differing word; the probes are random 32-byte sectors of the hash
// array, so a lane first tries the answer of its previous element, then one lane per warp row
// bisects and the others verify its answer with one probe pair (lcp_lockstep).
// The ADJACENT LCP (output `lcp`) costs no chain reads at all: when a sort splits two neighbours
// that came from one segment, they leave the old head's path at known digit depths, and
// min(depths) / D is exactly their LCP; neighbours never split have identical chains.
#include "peek_sort.cuh"

namespace peek {

#ifndef PEEK_LOC_K
#define PEEK_LOC_K 11
#endif
static constexpr int LOC_K = PEEK_LOC_K;              // positions per thread of a local work item
static constexpr int LOC_CAP = GS_THREADS * LOC_K;    // positions one CTA refines out of shared memory
static constexpr int TREE_DYN_SMEM = LOC_CAP * 18;    // u64 key + u32 request + 3 x u16 per position
static_assert(TREE_DYN_SMEM >= GS_STAGE_BYTES, "the grid sort stages its tiles in the same buffer");
static_assert(LOC_CAP <= 32768, "local positions are kept in 15 bits of a u16");
static constexpr int W0_BITS = 16;                    // round 0: leading bits of the first hash word
static constexpr int LOC_W = 24;                      // digit width of the local stage's keys

struct TreeCtl {      // device control block (zeroed by the host before launch)
    u32 bar;          // grid barrier word
    u32 unres[3];     // unresolved-position counters, rotating
    u32 maxnb;        // max chain length in blocks
    u32 flags;        // bit 0: some chain is empty (no full block)
    u32 maxseg[3];    // size of the largest unresolved segment, rotating
    u32 nbig[3];      // entries of the big-segment list, rotating
    u32 next_big, next_q;  // work queues of the local stage
    u32 bar2;              // grid barrier word of the signals kernel
    u32 fin_cb, fin_round; // where the grid-wide stage stopped: pair buffer, round (counter index)
    u32 pad[2];
    unsigned long long kor[2], kand[2];  // OR / AND of the round's keys (rotating): varying bits
};

// per-request record, one 32-byte sector: everything a refinement round wants to know about a chain
// without touching the hash array (gathered by request id, so it is packed to cost ONE sector)
struct __align__(32) ReqRec {
    i64 ao;     // blk_off[r]
    u32 na;     // chain length in blocks
    u32 pad;
    u64 lasth;  // last word of the chain (0 for an empty chain): "does one chain prefix the other"
    u64 k0;     // first word (0 for an empty chain): the first unknown word of a segment at depth 0
};
// the whole record in one 256-bit load that asks L2 to keep the line (the records are gathered again
// every round; the hash-array probes below are marked evict-first instead)
__device__ __forceinline__ void rec_load(const ReqRec* __restrict__ rec, u32 r, i64& ao, i32& na, u64& lasth, u64& k0) {
    u64 a, b;
    asm volatile("ld.global.nc.L2::evict_last.v4.b64 {%0,%1,%2,%3}, [%4];"
                 : "=l"(a), "=l"(b), "=l"(lasth), "=l"(k0) : "l"(rec + r));
    ao = (i64)a; na = (i32)(u32)b;
}
// a word of the hash array: read-once random sector, first in line for eviction from L2
__device__ __forceinline__ u64 ldh(const u64* p) {
    u64 pol, v;
    asm("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    asm volatile("ld.global.nc.L2::cache_hint.u64 %0, [%1], %2;" : "=l"(v) : "l"(p), "l"(pol));
    return v;
}

// per-segment record of the local stage, by segment start: what every member needs for its
// classification, in one sector
struct __align__(32) SegRec {
    unsigned long long head;  // (nb << 32) | ~position of the longest chain (atomicMax)
    u64 bo;                   // the head's blk_off
    u64 k0b;                  // the head's first word
    u32 depth;                // blocks all members are known to share
    u32 rank;                 // dense rank of the segment inside the work item
};

struct TreeArgs {
    const u64* hashes;
    const i64* blk_off;
    i64 N;
    i32 *order, *lcp, *group_id, *group_size, *cluster_depth, *cluster_size;
    i64* cluster_id;
    i32* n_groups;
    int signals_only;  // order and lcp are given: only groups and clusters are computed
    int cap_seg;       // an unresolved segment of at most this many positions goes to the local stage
    int quantum;       // positions per small-segment work item; segments above it are items of their own
    // workspace
    TreeCtl* ctl;
    GsBufs bufs;      // (sort key, request) by position, ping-pong
    u32* seg;         // N   by position: segment start | unresolved << 31
    u32* srank;       // N   by position (global rounds) / by segment start (local): dense segment rank
    ReqRec* rec;      // N   by request (phase 0)
    u64* seghead;     // N   by segment start: (nb << 32) | ~position of the longest chain
    i32* segdepth;    // N   by segment start: blocks all members are known to share
    i64* agg;         // gridDim scratch for grid scans
    i32* gsz;         // N   unresolved segment size by segment start; later group size by group id
    u64* biglist;     // segments above the quantum: start | size << 32
    SegRec* segrec;   // N   by segment start (local stage)
    unsigned short* posna;  // N by position: chain length of an unresolved position (0xffff: see the record)
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

// wmax caps the digit width (the local stage sorts on narrower digits)
__device__ __forceinline__ KeyLayout make_layout(i64 N, u64 maxnb, int wmax) {
    KeyLayout kl;
    kl.sbits = bits_for((u64)(N > 1 ? N - 1 : 1));
    for (int w = wmax; w >= 1; --w) {
        int D = (64 + w - 1) / w;
        u64 LDmax = (u64)D * maxnb + D;
        int lbits = bits_for(3 * LDmax + 4);
        kl.w = w; kl.D = D; kl.LDmax = LDmax; kl.lbits = lbits;
        if (kl.sbits + lbits + w <= 64) break;
    }
    kl.total = kl.sbits + kl.lbits + kl.w;
    if (kl.total > 64) __trap();  // no layout fits (a chain of >= 2^24 blocks): fail loudly, never sort truncated keys
    return kl;
}
// The narrowest layout (w = 1: D = 64, LDmax = 64 maxnb + 64, lbits <= bits(192 maxnb + 196)) needs
// sbits + lbits + 1 <= 64; with N < 2^31 (sbits <= 31) that holds for every maxnb < 2^24, i.e.
// chains of up to 2.6e8 tokens.  The entry point rejects longer chains (PEEK_ERR_UNSUPPORTED is
// reported through the status word; see tree_launch).

// Digit width of the grid-wide rounds.  A sort pass there costs two grid barriers whatever the queue
// holds, so queues of at most 65 536 requests take 16-bit digits (two passes fewer per round): 16 bits
// already tell that many branches apart, and the few that collide are finished by the local stage.
__device__ __forceinline__ int global_wmax(i64 N) { return N <= 65536 ? 16 : 32; }

// round-0 key of a request: d0 = (leading W0_BITS of its first word) | 1 << 31, or 0 for an empty chain
__device__ __forceinline__ u64 round0_key(const KeyLayout& kl, u32 d0) {
    const int w0 = kl.w < W0_BITS ? kl.w : W0_BITS;
    return (d0 >> 31) ? kl.pack(0, kl.f_after(0), (u64)((d0 & 0xffffu) >> (W0_BITS - w0)))
                      : kl.pack(0, kl.f_before(0, true), 0);
}
__device__ __forceinline__ u64 round0_vary(const KeyLayout& kl, u32 flags) {
    const int w0 = kl.w < W0_BITS ? kl.w : W0_BITS;
    u64 v = (1ull << w0) - 1;
    if (flags & 1u) v |= (kl.f_after(0) ^ kl.f_before(0, true)) << kl.w;
    return v;
}

// ---- staged tile processing ---------------------------------------------------------------------
// Every grid-wide phase walks the CTA's chunk of positions (the sort engine's ownership: CTA c owns
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
#ifndef PEEK_LSB
#define PEEK_LSB 1
#endif
static constexpr int LSB = PEEK_LSB;  // sub-batch of the local stage's classification
static_assert(LOC_K % LSB == 0, "LOC_K must be a multiple of LSB");
#define LSUBS(k) _Pragma("unroll") for (int k = 0; k < LSB; ++k)

struct TreeSmem {
    i32 wv[GS_WARPS + 1];   // per-warp values of the carry chains
    i64 wv64[GS_WARPS + 1];
    i64 carry64;
    i32 carry;
    u32 cnt, item, red;
    unsigned long long orv, andv;
};
static constexpr int LVL_HI_WORDS = 2048 + 64 + 8;  // per-CTA copy of the min-hierarchy levels >= 3

// LCP of K pairs of chains in lock step: chains H[ao..ao+na), H[bo..bo+nb), first lo words known
// equal (chain property R15: equal at a depth => equal above it, so the first difference is found
// by bisection).  act[k] selects the pairs to do; others keep res[k].
// Probes are random 32-byte sectors of a multi-GB array and the phase is bound by how many of them
// the memory system serves, so the search spends as few as it can:
//   (1) the last common word - one chain prefixes the other: done (the member's side comes from
//       its record, the head's chain is shared by the segment);
//   (2) the first unknown word (at depth 0 both first words are in the records: no read) together
//       with `hint`, the answer of this lane's previous element - neighbours in sorted order mostly
//       branch off their head at the same depth: one probe pair settles them;
//   (3) per warp row, ONE lane bisects and its answer g is the guess of the others, who probe
//       words g-1 and g; (4) whoever is still open bisects on.
// Must be called by full warps.
template <int K>
__device__ __forceinline__ void lcp_lockstep(const u64* __restrict__ H, const i64 (&ao)[K], const i32 (&na)[K],
                                             const i64 (&bo)[K], const i32 (&nb)[K], const i32 (&lo)[K],
                                             const bool (&act)[K], i32 (&res)[K],
                                             const u64 (&alast)[K],  // alast[k] = H[ao[k] + na[k] - 1]
                                             const u64 (&k0a)[K], const u64 (&k0b)[K],  // first words
                                             u64 (&wx)[K], u64 (&wy)[K],  // out: the two words at res when the chains branch
                                             i32& hint,              // in/out, < 0: none
                                             int& mode) {            // in/out: 1 = try the hint before (1)
    const unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    // while go: equal below/at L (L = lo - 1: nothing known); differ at R - known once R < Rm or the
    // last common word has been compared (lastdone)
    i32 L[K], R[K], Rm[K];
    bool go[K], lastdone[K];
    u64 x[K], y[K];
#pragma unroll
    for (int k = 0; k < K; ++k) {
        const i32 m = na[k] < nb[k] ? na[k] : nb[k];
        go[k] = act[k] && m > lo[k];
        if (act[k] && !go[k]) res[k] = m;
        L[k] = lo[k] - 1;
        R[k] = Rm[k] = m - 1;
        lastdone[k] = false;
        wx[k] = wy[k] = 0;
    }
    // (1) the last common word, for the pairs selected by sel[k] that can still be prefixes
    auto probe_last = [&](const bool (&sel)[K]) {
#pragma unroll
        for (int k = 0; k < K; ++k) {
            if (go[k] && sel[k] && R[k] == Rm[k]) {
                x[k] = R[k] == na[k] - 1 ? alast[k] : ldh(H + ao[k] + R[k]);
                y[k] = ldh(H + bo[k] + R[k]);
            }
        }
#pragma unroll
        for (int k = 0; k < K; ++k) {
            if (go[k] && sel[k] && R[k] == Rm[k]) {
                lastdone[k] = true;
                if (x[k] == y[k]) { res[k] = R[k] + 1; go[k] = false; }
                else { wx[k] = x[k]; wy[k] = y[k]; }
                if (go[k] && R[k] - L[k] <= 1) { res[k] = R[k]; go[k] = false; }
            }
        }
    };
    // probe words g - 1 and g of the pairs selected by pr[k] (one round trip): settles the pair when
    // g is the answer.  first = also probe word lo (the first unknown word) in the same round trip.
    auto probe_around = [&](const i32 (&gk)[K], const bool (&pr)[K], bool first, const bool (&fsel)[K]) {
        u64 x2[K], y2[K], x3[K], y3[K];
        bool p0[K], p1[K], p2[K];
#pragma unroll
        for (int k = 0; k < K; ++k) {
            p0[k] = first && go[k] && fsel[k];
            p1[k] = pr[k] && gk[k] - 1 > L[k] + (first ? 1 : 0) && gk[k] - 1 < R[k];
            p2[k] = pr[k] && gk[k] > L[k] + (first ? 1 : 0) && gk[k] < R[k];
            x3[k] = y3[k] = 0;
            if (p0[k]) {
                if (lo[k] == 0) { x3[k] = k0a[k]; y3[k] = k0b[k]; }
                else { x3[k] = ldh(H + ao[k] + lo[k]); y3[k] = ldh(H + bo[k] + lo[k]); }
            }
            if (p1[k]) { x[k] = ldh(H + ao[k] + gk[k] - 1); y[k] = ldh(H + bo[k] + gk[k] - 1); }
            if (p2[k]) { x2[k] = ldh(H + ao[k] + gk[k]); y2[k] = ldh(H + bo[k] + gk[k]); }
        }
#pragma unroll
        for (int k = 0; k < K; ++k) {
            if (p0[k]) {
                if (x3[k] != y3[k]) { res[k] = lo[k]; go[k] = false; p1[k] = p2[k] = false; wx[k] = x3[k]; wy[k] = y3[k]; }
                else L[k] = lo[k];
            }
            if (p1[k]) { if (x[k] == y[k]) L[k] = gk[k] - 1; else { R[k] = gk[k] - 1; wx[k] = x[k]; wy[k] = y[k]; } }
            if (p2[k] && gk[k] < R[k]) { if (x2[k] == y2[k]) L[k] = gk[k]; else { R[k] = gk[k]; wx[k] = x2[k]; wy[k] = y2[k]; } }
            if (go[k] && (p0[k] || pr[k]) && R[k] - L[k] <= 1 && (R[k] < Rm[k] || lastdone[k])) { res[k] = R[k]; go[k] = false; }
        }
    };
    // one bisection step for the elements selected by sel[k]; returns whether any is still going
    auto step = [&](const bool (&sel)[K]) -> bool {
#pragma unroll
        for (int k = 0; k < K; ++k) {
            if (go[k] && sel[k]) {
                const i32 p = (L[k] + R[k]) >> 1;
                x[k] = ldh(H + ao[k] + p); y[k] = ldh(H + bo[k] + p);
            }
        }
        bool any = false;
#pragma unroll
        for (int k = 0; k < K; ++k) {
            if (go[k] && sel[k]) {
                const i32 p = (L[k] + R[k]) >> 1;
                if (x[k] == y[k]) L[k] = p; else { R[k] = p; wx[k] = x[k]; wy[k] = y[k]; }
                if (R[k] - L[k] <= 1) { res[k] = R[k]; go[k] = false; }
                any |= go[k];
            }
        }
        return any;
    };
    bool all_sel[K], doneB[K];
#pragma unroll
    for (int k = 0; k < K; ++k) { all_sel[k] = true; doneB[k] = false; }
    // (2) the first unknown word and this lane's previous answer
    auto probe_hint = [&](const bool (&sel)[K]) {
        i32 gk[K];
        bool pr[K];
#pragma unroll
        for (int k = 0; k < K; ++k) { gk[k] = hint; pr[k] = go[k] && sel[k] && hint >= 0; }
        probe_around(gk, pr, true, sel);
#pragma unroll
        for (int k = 0; k < K; ++k) doneB[k] |= sel[k];
    };
    {   // lanes whose previous element branched try that depth first: it usually settles the pair
        // and then the last common word is never read
        bool early[K];
        bool e = false;
#pragma unroll
        for (int k = 0; k < K; ++k) { early[k] = go[k] && mode == 1 && hint >= 0; e |= early[k]; }
        if (__any_sync(FULL, e)) probe_hint(early);
    }
    bool pending = false;
#pragma unroll
    for (int k = 0; k < K; ++k) pending |= go[k];
    if (__any_sync(FULL, pending)) probe_last(all_sel);
    pending = false;
#pragma unroll
    for (int k = 0; k < K; ++k) pending |= go[k];
    if (__any_sync(FULL, pending)) {
        {
            bool late[K];
            bool e = false;
#pragma unroll
            for (int k = 0; k < K; ++k) { late[k] = go[k] && !doneB[k]; e |= late[k]; }
            if (__any_sync(FULL, e)) probe_hint(late);
            pending = false;
#pragma unroll
            for (int k = 0; k < K; ++k) pending |= go[k];
        }
        if (__any_sync(FULL, pending)) {  // (3) one lane per row bisects, the others verify
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
            i32 gk[K];
            bool pr[K];
#pragma unroll
            for (int k = 0; k < K; ++k) {
                gk[k] = __shfl_sync(FULL, res[k], leader[k] < 0 ? 0 : leader[k]);
                pr[k] = go[k] && leader[k] >= 0;
            }
            probe_around(gk, pr, false, all_sel);
        }
    }
    bool any = true;
    while (any) any = step(all_sel);  // (4)
#pragma unroll
    for (int k = 0; k < K; ++k) {
        if (act[k]) {
            const bool branched = res[k] <= Rm[k];  // not a prefix relation
            mode = branched ? 1 : 0;
            if (branched) hint = res[k];
        }
    }
}

// new sort key of a classified member (l = LCP with the head in words; wa / wb = the two words at l)
__device__ __forceinline__ u64 class_key(const KeyLayout& kl, u32 rank, i32 l, i32 na, i32 nb, u64 wa, u64 wb) {
    u64 F, dig = 0;
    if (l == na && l == nb) F = kl.f_head();
    else if (l == na) F = kl.f_before((u64)kl.D * l, true);
    else {  // l < na <= nb: the words at l differ
        const int jd = __clzll((long long)(wa ^ wb)) / kl.w;
        const u64 ld = (u64)kl.D * l + jd;
        const u64 da = (wa << (jd * kl.w)) >> (64 - kl.w), db = (wb << (jd * kl.w)) >> (64 - kl.w);
        dig = da;
        F = da < db ? kl.f_before(ld, false) : kl.f_after(ld);
    }
    return kl.pack(rank, F, dig);
}

// ---- local stage ----------------------------------------------------------------------------------
// A work item lives in shared memory.  Its elements (sort key, request, chain length saturated to
// 16 bits - the head of a segment is its longest chain, found without a gather) never move: the
// sorted order is a permutation `idx` of element numbers (u16), so a sort pass moves two bytes per
// element and nothing is held in registers across a barrier.  The second index buffer doubles as
// the per-position scratch between sorts (segment start + unresolved flag).
struct LocalBufs {
    u64* key;             // by element
    u32* val;             // by element: request
    unsigned short* na;   // by element: chain length, 0xffff = look it up in the record
    unsigned short* idx;  // by position: element (current order)
    unsigned short* aux;  // by position: the other index buffer / segment start | unresolved << 15
};
__device__ __forceinline__ LocalBufs local_bufs(unsigned char* dyn_smem) {
    return LocalBufs{(u64*)dyn_smem, (u32*)(dyn_smem + (size_t)LOC_CAP * 8),
                     (unsigned short*)(dyn_smem + (size_t)LOC_CAP * 12),
                     (unsigned short*)(dyn_smem + (size_t)LOC_CAP * 14),
                     (unsigned short*)(dyn_smem + (size_t)LOC_CAP * 16)};
}

static constexpr int LOC_COUNT_MAX = 512;  // items up to this size rank by counting (quadratic: 21 us at 1024, 5 us at 512)
// Stable LSD sort of the item's n <= LOC_CAP positions by the key bits set in `vary` (8-bit
// digits): permutes lb.idx (ping-pong with lb.aux; the roles are swapped in place).  Warp w owns
// positions [w*32*Kp, (w+1)*32*Kp), Kp = ceil(n / GS_THREADS) rows.
__device__ __forceinline__ void local_sort(LocalBufs& lb, int n, u64 vary, GsSmem& sm) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int Kp = (n + GS_THREADS - 1) / GS_THREADS;
    const int wbase = w * 32 * Kp;
    if (n <= LOC_COUNT_MAX) {
        // Small items (one position per thread; the paper's queues hold 60-200 requests,
        // PAPER.md:364): no passes at all - every position counts the positions that sort before it
        // (smaller key, or equal key and earlier) against the keys staged by position, and its
        // element goes straight to that rank.
        if (!vary) return;
        static_assert(sizeof(sm.wcnt) >= GS_THREADS * sizeof(u64), "staging area of the counting sort");
        u64* kp = (u64*)&sm.wcnt[0][0];
        const int t = threadIdx.x;
        unsigned short e = 0;
        u64 key = ~0ull;
        if (t < n) { e = lb.idx[t]; key = lb.key[e]; kp[t] = key; }
        __syncthreads();
        if (t < n) {
            u32 rank = 0;
#pragma unroll 8
            for (int j = 0; j < n; ++j) {
                const u64 kj = kp[j];
                rank += (kj < key || (kj == key && j < t)) ? 1u : 0u;
            }
            lb.aux[rank] = e;
        }
        __syncthreads();
        unsigned short* tt = lb.idx; lb.idx = lb.aux; lb.aux = tt;
        return;
    }
    while (vary) {
        const int sh = __ffsll((long long)vary) - 1;
        vary &= ~(0xffull << sh);
        u32 meta[LOC_K];
        unsigned short el[LOC_K];
#pragma unroll
        for (int k = 0; k < LOC_K; ++k) {
            const int i = wbase + k * 32 + lane;
            const bool valid = k < Kp && i < n;
            el[k] = valid ? lb.idx[i] : (unsigned short)0;
            meta[k] = valid ? (u32)(lb.key[el[k]] >> sh) & 255u : (0x100u | lane);
        }
        gs_rank_tile<LOC_K>(meta, sm);
#pragma unroll
        for (int k = 0; k < LOC_K; ++k) {
            const int i = wbase + k * 32 + lane;
            if (k < Kp && i < n) {
                const u32 d = meta[k] & 0xffffu;
                lb.aux[sm.dstart[d] + sm.wcnt[w][d] + (meta[k] >> 16)] = el[k];
            }
        }
        __syncthreads();
        unsigned short* t = lb.idx; lb.idx = lb.aux; lb.aux = t;
    }
}

enum { LOCAL_FROM_GLOBAL = 0, LOCAL_WHOLE_QUEUE = 1 };

// One CTA finishes positions [p0, p0 + n), n <= LOC_CAP, which hold whole segments: all remaining
// refinement rounds, then the final order and the adjacent LCPs of the range.
//   LOCAL_FROM_GLOBAL  the pairs are Kg / Vg as the global stage left them (keys in layout kg); the
//                      LCP at every boundary of the range as it stands is already written
//   LOCAL_WHOLE_QUEUE  p0 = 0, n = N: round 0 runs here too (A.srank holds the round-0 digits)
// Keys made here use the layout kl (narrower digits than the grid-wide rounds: fewer sort passes;
// a digit collision only keeps two branches together for one more round).
__device__ __forceinline__ void tree_local(const TreeArgs& A, const KeyLayout& kg, const KeyLayout& kl,
                                           const u64* __restrict__ Kg, const u32* __restrict__ Vg, i64 p0, int n,
                                           int mode, GsSmem& ssm, TreeSmem& tsm, LocalBufs lb) {
    const unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const unsigned le_mask = 0xffffffffu >> (31 - lane);
    const u64* __restrict__ H = A.hashes;
    const ReqRec* __restrict__ rec = A.rec;
    const int Kp = (n + GS_THREADS - 1) / GS_THREADS;
    const int wbase = w * 32 * Kp;
    PEEK_MARK(30);
    for (int i = threadIdx.x; i < n; i += GS_THREADS) {
        u32 r;
        if (mode == LOCAL_FROM_GLOBAL) { lb.key[i] = __ldcg(Kg + p0 + i); r = __ldcg(Vg + p0 + i); }
        else { lb.key[i] = round0_key(kl, __ldcg(A.srank + i)); r = (u32)i; }
        PEEK_CHECK((i64)r < A.N, "request id of a sorted pair out of range");
        lb.val[i] = r;
        lb.idx[i] = (unsigned short)i;
        if (mode == LOCAL_FROM_GLOBAL) lb.na[i] = __ldcg(A.posna + p0 + i);
        else { const u32 na = __ldg(&rec[r].na); lb.na[i] = (unsigned short)(na < 0xffffu ? na : 0xffffu); }
    }
    __syncthreads();
    i32 hint = -1;
    int hmode = 0;
    u64 vary = mode == LOCAL_WHOLE_QUEUE ? round0_vary(kl, __ldcg(&A.ctl->flags)) : 0;
    for (int lr = mode == LOCAL_WHOLE_QUEUE ? 1 : 0;; ++lr) {
        // stable sort of the range by the keys of the last classification (round 0: the first words)
        PEEK_MARK(31);
        if (lr > 0) local_sort(lb, n, vary, ssm);
        PEEK_MARK(32);
        const KeyLayout& kc = lr == 0 ? kg : kl;  // layout of the keys as they stand
        // key of position i, of its left and of its right neighbour (shuffles inside the row)
        auto keys3 = [&](int i, bool valid, u64& key, u64& prev, u64& next) {
            key = valid ? lb.key[lb.idx[i]] : 0;
            prev = __shfl_up_sync(FULL, key, 1);
            next = __shfl_down_sync(FULL, key, 1);
            if (lane == 0) prev = (valid && i > 0) ? lb.key[lb.idx[i - 1]] : 0;
            if (lane == 31 || !(i + 1 < n)) next = (valid && i + 1 < n) ? lb.key[lb.idx[i + 1]] : 0;
        };
        // ---- L1a: segment starts per warp ----
        {
            u32 wc = 0, wl = 0;
#pragma unroll
            for (int k = 0; k < LOC_K; ++k) {
                if (k < Kp) {
                    const int i = wbase + k * 32 + lane;
                    const bool valid = i < n;
                    u64 key, prev, next;
                    keys3(i, valid, key, prev, next);
                    const bool start = valid && (i == 0 || prev != key);
                    if (start) A.segrec[p0 + i].head = 0;  // reset before L1b's maxima (a CTA barrier apart)
                    const unsigned bal = __ballot_sync(FULL, start);
                    wc += __popc(bal);
                    if (bal) wl = (u32)((i - lane) + 31 - __clz(bal)) + 1u;
                }
            }
            if (lane == 0) tsm.wv64[w] = ((i64)wc << 32) | wl;
            if (threadIdx.x == 0) { tsm.cnt = 0; tsm.orv = 0; tsm.andv = ~0ull; }
            __syncthreads();
            if (w == 0) {  // exclusive (sum, max) scan over the warps
                const i64 own = lane < GS_WARPS ? tsm.wv64[lane] : 0;
                u32 ic = (u32)(own >> 32), il = (u32)own;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const u32 xc = __shfl_up_sync(FULL, ic, o), xl = __shfl_up_sync(FULL, il, o);
                    if (lane >= o) { ic += xc; il = max(il, xl); }
                }
                u32 ec = __shfl_up_sync(FULL, ic, 1), el = __shfl_up_sync(FULL, il, 1);
                if (lane == 0) { ec = 0; el = 0; }
                if (lane < GS_WARPS) tsm.wv64[lane] = ((i64)ec << 32) | el;
            }
            __syncthreads();
        }
        // ---- L1b: segment start and rank of every position, adjacent LCP of the boundaries the
        // last sort made, unresolved flag, head = longest chain of every unresolved segment ----
        {
            i32 c = (i32)(u32)tsm.wv64[w] - 1;  // last segment start before this warp's rows
            u32 cc = (u32)(tsm.wv64[w] >> 32);  // segment starts before this warp's rows
            u32 n_unres = 0;
#pragma unroll
            for (int k = 0; k < LOC_K; ++k) {
                if (k < Kp) {
                    const int i = wbase + k * 32 + lane;
                    const bool valid = i < n;
                    u64 key, prev, next;
                    keys3(i, valid, key, prev, next);
                    const bool start = valid && (i == 0 || prev != key);
                    const bool last = valid && (i == n - 1 || next != key);
                    const u64 F = kc.F_of(key);
                    const bool br = valid && kc.is_branch(F);
                    const unsigned bal = __ballot_sync(FULL, start);
                    const unsigned m = bal & le_mask;
                    const i32 s = m ? (i32)(i - lane) + 31 - __clz(m) : c;
                    if (bal) c = (i32)(i - lane) + 31 - __clz(bal);
                    const u32 rank = cc + __popc(m) - 1u;
                    cc += __popc(bal);
                    const bool un = br && !(start && last);
                    if (valid) lb.aux[i] = (unsigned short)(s | (un ? 0x8000 : 0));
                    if (start) {
                        A.segrec[p0 + i].rank = rank;
                        A.segrec[p0 + i].depth = br ? (u32)(kc.ld_of(F) / kc.D) : 0u;
                        if (p0 + i == 0) A.lcp[0] = 0;
                        else if (i > 0 && lr > 0 && kc.seg_of(prev) == kc.seg_of(key)) {
                            const u64 la = kc.ldv(kc.F_of(prev)), lb2 = kc.ldv(F);
                            A.lcp[p0 + i] = (i32)((la < lb2 ? la : lb2) / kc.D);
                        }
                    }
                    const unsigned ub = __ballot_sync(FULL, un);
                    n_unres += __popc(ub);
                    if (ub) {  // warp-uniform
                        const int e = valid ? lb.idx[i] : 0;
                        u32 nbv = un ? (u32)lb.na[e] : 0u;
                        if (nbv == 0xffffu) nbv = __ldg(&rec[lb.val[e]].na);  // saturated: the record has it
                        u64 v = un ? (((u64)nbv << 32) | (u64)(0xffffffffu - (u32)i)) : 0ull;
#pragma unroll
                        for (int o = 1; o < 32; o <<= 1) {
                            const u64 x = __shfl_up_sync(FULL, v, o);
                            const i32 sx = __shfl_up_sync(FULL, s, o);
                            if (lane >= o && sx == s && x > v) v = x;
                        }
                        const i32 sn = __shfl_down_sync(FULL, s, 1);
                        if (v && (lane == 31 || sn != s)) atomicMax(&A.segrec[p0 + s].head, v);
                    }
                }
            }
            if (lane == 0 && n_unres) atomicAdd(&tsm.cnt, n_unres);
            __syncthreads();
        }
        PEEK_MARK(33);
        if (tsm.cnt == 0) break;
        // ---- L1c: the head's chain offset and first word into every unresolved segment's record ----
#pragma unroll
        for (int k = 0; k < LOC_K; ++k) {
            if (k < Kp) {
                const int i = wbase + k * 32 + lane;
                if (i < n) {
                    const u32 a = lb.aux[i];
                    if (a == (0x8000u | (u32)i)) {  // an unresolved segment starts here
                        const unsigned long long hv = __ldcg(&A.segrec[p0 + i].head);
                        PEEK_CHECK(0xffffffffu - (u32)hv < (u32)n, "segment head position outside the work item");
                        const u32 h = lb.val[lb.idx[0xffffffffu - (u32)hv]];
                        i64 bo; i32 nh; u64 lh, k0b;
                        rec_load(rec, h, bo, nh, lh, k0b);
                        A.segrec[p0 + i].bo = (u64)bo;
                        A.segrec[p0 + i].k0b = k0b;
                    }
                }
            }
        }
        __syncthreads();
        // ---- L2: classify every unresolved position against its segment head.  The new key
        // replaces the element's old one in place: this phase reads no neighbour's key ----
        {
            u64 orv = 0, andv = ~0ull;
            for (int hb = 0; hb * LSB < Kp; ++hb) {
                u32 sg[LSB], r[LSB], rk[LSB], h[LSB], el[LSB];
                bool val_[LSB], un[LSB], cmp[LSB];
                u64 hv[LSB], al[LSB], k0a[LSB], k0b[LSB];
                i64 ao[LSB], bo[LSB];
                i32 na[LSB], nb[LSB], lo[LSB], l[LSB];
                LSUBS(k) {
                    const int kk = hb * LSB + k;
                    const int i = wbase + kk * 32 + lane;
                    val_[k] = kk < Kp && i < n;
                    sg[k] = 0; r[k] = 0; un[k] = false; el[k] = 0;
                    if (val_[k]) {
                        const u32 a = lb.aux[i];
                        sg[k] = a & 0x7fffu;
                        un[k] = (a >> 15) != 0;
                        el[k] = lb.idx[i];
                        r[k] = lb.val[el[k]];
                    }
                }
                LSUBS(k) {
                    rk[k] = 0; hv[k] = 0; ao[k] = 0; na[k] = 0; lo[k] = 0; al[k] = 0; k0a[k] = 0; bo[k] = 0; k0b[k] = 0;
                    if (val_[k]) {
                        PEEK_CHECK((int)sg[k] < n && p0 + sg[k] < A.N, "segment start outside the work item");
                        const ulonglong2* sp = (const ulonglong2*)(A.segrec + p0 + sg[k]);
                        const ulonglong2 s0 = __ldcg(sp), s1 = __ldcg(sp + 1);
                        hv[k] = s0.x; bo[k] = (i64)s0.y; k0b[k] = s1.x;
                        lo[k] = (i32)(u32)s1.y; rk[k] = (u32)(s1.y >> 32);
                    }
                    if (un[k]) rec_load(rec, r[k], ao[k], na[k], al[k], k0a[k]);
                }
                LSUBS(k) {
                    nb[k] = (i32)(hv[k] >> 32);
                    const int kk = hb * LSB + k;
                    cmp[k] = un[k] && (u32)(wbase + kk * 32 + lane) != 0xffffffffu - (u32)hv[k];  // not the head itself
                    l[k] = na[k];
                }
                PEEK_MARK(40 + hb);
                u64 wa[LSB], wb[LSB];
                lcp_lockstep<LSB>(H, ao, na, bo, nb, lo, cmp, l, al, k0a, k0b, wa, wb, hint, hmode);
                PEEK_MARK(60 + hb);
                LSUBS(k) {
                    if (val_[k]) {
                        const u64 nk = un[k] ? class_key(kl, rk[k], l[k], na[k], nb[k], wa[k], wb[k])
                                             : kl.pack(rk[k], 0, 0);
                        lb.key[el[k]] = nk;
                        orv |= nk;
                        andv &= nk;
                    }
                }
            }
            const u32 olo = __reduce_or_sync(FULL, (u32)orv), ohi = __reduce_or_sync(FULL, (u32)(orv >> 32));
            const u32 alo = __reduce_and_sync(FULL, (u32)andv), ahi = __reduce_and_sync(FULL, (u32)(andv >> 32));
            if (lane == 0) {
                atomicOr(&tsm.orv, ((unsigned long long)ohi << 32) | olo);
                atomicAnd(&tsm.andv, ((unsigned long long)ahi << 32) | alo);
            }
            __syncthreads();
        }
        vary = tsm.orv & ~tsm.andv;  // sorted on at the top of the next round
        __syncthreads();             // tsm.orv is reset by the next round's L1a
    }
    // ---- final order of the range; positions inside a final segment repeat their neighbour's
    // chain (the LCP of every boundary was written when the boundary appeared) ----
    PEEK_MARK(35);
#pragma unroll
    for (int k = 0; k < LOC_K; ++k) {
        if (k < Kp) {
            const int i = wbase + k * 32 + lane;
            if (i < n) {
                const int e = lb.idx[i];
                const u32 r = lb.val[e];
                A.order[p0 + i] = (i32)r;
                if (i > 0 && lb.key[e] == lb.key[lb.idx[i - 1]]) {
                    u32 nbv = lb.na[e];
                    if (nbv == 0xffffu) nbv = __ldg(&rec[r].na);
                    A.lcp[p0 + i] = (i32)nbv;
                }
            }
        }
    }
    __syncthreads();  // the shared buffers are reused by the next work item
}

// final order and LCP of positions [x, y) that the global stage left resolved: written straight
// from the global pairs (a non-start position of a resolved segment repeats its neighbour's chain)
__device__ __forceinline__ void tree_direct_output(const TreeArgs& A, const u32* __restrict__ Vg, i64 x, i64 y) {
    for (i64 j = x + threadIdx.x; j < y; j += GS_THREADS) {
        const u32 r = __ldcg(Vg + j);
        A.order[j] = (i32)r;
        if ((i64)(__ldcg(A.seg + j) & 0x7fffffffu) != j) A.lcp[j] = (i32)__ldg(&A.rec[r].na);
    }
}

// ---- the stages as device functions; the kernels below string them together ---------------------

// phase 0: chain lengths, last words, round-0 digits.  Ends with a grid barrier.
__device__ __forceinline__ void tree_phase0(const TreeArgs& A, Grid& g) {
    const unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const unsigned le_mask = 0xffffffffu >> (31 - lane);  // lanes <= this one
    const i64 N = A.N;
    const int G = gridDim.x, me = blockIdx.x;
    const i64 gtid = (i64)me * GS_THREADS + threadIdx.x;
    const u64* __restrict__ H = A.hashes;
    const i64* __restrict__ BO = A.blk_off;
    const i64 C = (N + G - 1) / G;
    const i64 c0 = min((i64)me * C, N), c1 = min(c0 + C, N);
    const int ntiles = (int)((C + GS_TILE - 1) / GS_TILE);
    // rows per warp: a chunk of less than a tile is spread over all warps of the CTA (rows beyond KP
    // are out of range), so small chunks do not leave most warps idle
    const int KP = ntiles == 1 ? (int)((C + GS_THREADS - 1) / GS_THREADS) : GS_KPT;
    auto IDX = [&](int t, int k) -> i64 {
        return k < KP ? c0 + (i64)t * GS_TILE + w * (32 * KP) + k * 32 + lane : (i64)1 << 62;
    };
    (void)FULL; (void)le_mask; (void)gtid; (void)H; (void)BO; (void)ntiles; (void)c1;
    // ---- phase 0: chain lengths, last words, round-0 digits (leading bits of the first word) ----
    {
        u32 mx = 0, empty = 0;
        for (int t = 0; t < ntiles; ++t) {
            i64 b0[GS_KPT], b1[GS_KPT];
            ELEMS(k) {
                const i64 i = IDX(t, k);
                b0[k] = b1[k] = 0;
                if (i < c1) { b0[k] = __ldg(BO + i); b1[k] = __ldg(BO + i + 1); }
            }
            // the first and the last word of every chain, gathered once into the request's record: a
            // member's chain is never longer than its head's, so the "does one chain prefix the
            // other" probe of every round reads the member's side from the record
            u64 lw[GS_KPT], fw[GS_KPT];
            ELEMS(k) {
                lw[k] = fw[k] = 0;
                if (b1[k] > b0[k]) { lw[k] = __ldg(H + b1[k] - 1); fw[k] = __ldg(H + b0[k]); }
            }
            ELEMS(k) {
                const i64 i = IDX(t, k);
                if (i < c1) {
                    const bool has = b1[k] > b0[k];
                    mx = max(mx, (u32)(b1[k] - b0[k]));
                    empty |= has ? 0u : 1u;
                    ulonglong2* rp = (ulonglong2*)(A.rec + i);
                    rp[0] = make_ulonglong2((u64)b0[k], (u64)(u32)(b1[k] - b0[k]));
                    rp[1] = make_ulonglong2(lw[k], fw[k]);
                    A.srank[i] = has ? (0x80000000u | (u32)(fw[k] >> (64 - W0_BITS))) : 0u;
                }
            }
        }
        mx = __reduce_max_sync(FULL, mx);
        empty = __reduce_or_sync(FULL, empty);
        if (lane == 0 && mx) atomicMax(&A.ctl->maxnb, mx);
        if (lane == 0 && empty) atomicOr(&A.ctl->flags, 1u);
        if (gtid == 0) { A.ctl->kand[0] = ~0ull; A.ctl->kand[1] = ~0ull; }
    }
    g.sync();
}

// grid-wide stage: round 0, then refinement rounds while some unresolved segment exceeds cap_seg.
// Leaves the pairs in A.bufs.*[ctl->fin_cb] and the round's counters at index ctl->fin_round % 3.
__device__ __forceinline__ void tree_global(const TreeArgs& A, const KeyLayout& kl, Grid& g, GsSmem& ssm,
                                            TreeSmem& tsm, const GsStage stg) {
    const unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const unsigned le_mask = 0xffffffffu >> (31 - lane);  // lanes <= this one
    const i64 N = A.N;
    const int G = gridDim.x, me = blockIdx.x;
    const i64 gtid = (i64)me * GS_THREADS + threadIdx.x;
    const u64* __restrict__ H = A.hashes;
    const i64* __restrict__ BO = A.blk_off;
    const i64 C = (N + G - 1) / G;
    const i64 c0 = min((i64)me * C, N), c1 = min(c0 + C, N);
    const int ntiles = (int)((C + GS_TILE - 1) / GS_TILE);
    // rows per warp: a chunk of less than a tile is spread over all warps of the CTA (rows beyond KP
    // are out of range), so small chunks do not leave most warps idle
    const int KP = ntiles == 1 ? (int)((C + GS_THREADS - 1) / GS_THREADS) : GS_KPT;
    auto IDX = [&](int t, int k) -> i64 {
        return k < KP ? c0 + (i64)t * GS_TILE + w * (32 * KP) + k * 32 + lane : (i64)1 << 62;
    };
    (void)FULL; (void)le_mask; (void)gtid; (void)H; (void)BO; (void)ntiles; (void)c1;
    int cb = 0, round = 0;
    // ---- round 0: stable sort by the round-0 key (generated on the fly from the digits) ----
    {
        const u32 flags = __ldcg(&A.ctl->flags);
        const u32* __restrict__ d0 = A.srank;
        cb = grid_sort_pairs_gen(A.bufs, N, round0_vary(kl, flags), g, ssm, stg,
                                 [&](i64 i, u64& key, u32& val) { key = round0_key(kl, __ldcg(d0 + i)); val = (u32)i; });
    }
    PEEK_MARK(9);

    for (round = 1;; ++round) {
        g.sync();  // keys / order of the previous phase visible
        PEEK_MARK(10);
        const u64* K = A.bufs.key[cb];
        const u32* cur = A.bufs.val[cb];
        u32* cnt = &A.ctl->unres[round % 3];
        if (gtid == 0) {
            A.ctl->unres[(round + 1) % 3] = 0;
            A.ctl->maxseg[(round + 1) % 3] = 0;
            A.ctl->nbig[(round + 1) % 3] = 0;
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
                        else if (kl.seg_of(km[k]) == kl.seg_of(k0[k])) {
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
        // ---- R1b: segment start of every position, unresolved flag, head = longest chain; sizes
        // of the unresolved segments (the largest decides whether the local stage can take over) ----
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
            u32 n_unres = 0, max_size = 0;
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
                        if (un[k] && (fl[kk] & 2u)) {  // last position of an unresolved segment: its size
                            const u32 size = (u32)(i - (i64)s) + 1u;
                            A.gsz[s] = (i32)size;
                            max_size = max(max_size, size);
                            if (size > (u32)A.quantum && size <= (u32)A.cap_seg) {
                                const u32 slot = atomicAdd(&A.ctl->nbig[round % 3], 1u);
                                PEEK_CHECK((i64)slot < A.N / 64 + 64, "big-segment list overflow");
                                A.biglist[slot] = (u64)(u32)s | ((u64)size << 32);
                            }
                        }
                        r[k] = un[k] ? __ldcg(cur + i) : 0u;
                        PEEK_CHECK((i64)r[k] < N, "R1b: request id out of range");
                    }
                    u32 nbr[SB];
                    SUBS(k) nbr[k] = un[k] ? __ldg(&A.rec[r[k]].na) : 0u;
                    SUBS(k) {  // kept by position for the local stage (its head search needs no gather then)
                        const i64 i = IDX(t, hb * SB + k);
                        if (i < c1) A.posna[i] = (unsigned short)(un[k] && nbr[k] < 0xffffu ? nbr[k] : 0xffffu);
                    }
                    SUBS(k) {
                        // head = longest chain of the segment, lowest position on ties: segmented
                        // max over the row's runs of equal s, one atomic per run
                        const i64 i = IDX(t, hb * SB + k);
                        u64 v = un[k] ? (((u64)nbr[k] << 32) | (u64)(0xffffffffu - (u32)i)) : 0ull;
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
            max_size = __reduce_max_sync(FULL, max_size);
            if (lane == 0 && max_size) atomicMax(&A.ctl->maxseg[round % 3], max_size);
        }
        g.sync();
        PEEK_MARK(11);
        // grid-uniform (read after the barrier): every unresolved segment fits one CTA
        if (__ldcg(&A.ctl->maxseg[round % 3]) <= (u32)A.cap_seg) break;  // the local stage takes over

        // ---- R2: classify every unresolved position against its segment head (keys in place) ----
        {
            u64* Kw = A.bufs.key[cb];
            u64 orv = 0, andv = ~0ull;
            i32 hint = -1;
            int hmode = 0;
            for (int t = 0; t < ntiles; ++t)
            for (int hb = 0; hb < GS_KPT / SB; ++hb) {
                u32 sg[SB], r[SB], h[SB], rk[SB];
                bool un[SB], cmp[SB];
                SUBS(k) {
                    const i64 i = IDX(t, hb * SB + k);
                    sg[k] = 0; r[k] = 0; rk[k] = 0;
                    if (i < c1) { sg[k] = A.seg[i]; r[k] = __ldcg(cur + i); rk[k] = A.srank[i]; }
                    un[k] = (sg[k] >> 31) != 0;
                    PEEK_CHECK((i64)(sg[k] & 0x7fffffffu) < N, "R2: segment start out of range");
                }
                u64 hv[SB], al[SB], k0a[SB], k0b[SB];
                i64 ao[SB], bo[SB];
                i32 na[SB], nb[SB], lo[SB], l[SB];
                SUBS(k) {
                    hv[k] = 0; ao[k] = 0; na[k] = 0; lo[k] = 0; al[k] = 0; k0a[k] = 0;
                    if (un[k]) {
                        const u32 s = sg[k] & 0x7fffffffu;
                        hv[k] = __ldcg(A.seghead + s);
                        lo[k] = __ldcg(A.segdepth + s);
                        rec_load(A.rec, r[k], ao[k], na[k], al[k], k0a[k]);
                    }
                }
                SUBS(k) {
                    PEEK_CHECK(!un[k] || (i64)(0xffffffffu - (u32)hv[k]) < N, "R2: segment head position out of range");
                    h[k] = un[k] ? __ldcg(cur + (0xffffffffu - (u32)hv[k])) : 0u; nb[k] = (i32)(hv[k] >> 32);
                    PEEK_CHECK((i64)h[k] < N && (i64)r[k] < N, "R2: request id out of range");
                }
                SUBS(k) {
                    bo[k] = 0; k0b[k] = 0;
                    if (un[k]) { i32 nh; u64 lh; rec_load(A.rec, h[k], bo[k], nh, lh, k0b[k]); }
                    cmp[k] = un[k] && r[k] != h[k];
                    l[k] = na[k];  // r == h: the head itself
                }
                u64 wa[SB], wb[SB];
                lcp_lockstep<SB>(H, ao, na, bo, nb, lo, cmp, l, al, k0a, k0b, wa, wb, hint, hmode);
                SUBS(k) {
                    const i64 i = IDX(t, hb * SB + k);
                    if (i < c1) {
                        // dense segment rank: few leading key bits vary
                        const u64 nk = un[k] ? class_key(kl, rk[k], l[k], na[k], nb[k], wa[k], wb[k]) : kl.pack(rk[k], 0, 0);
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
    if (gtid == 0) { A.ctl->fin_cb = (u32)cb; A.ctl->fin_round = (u32)round; }
}

// local stage: every work item is finished by one CTA (no CTA waits for another)
__device__ __forceinline__ void tree_local_stage(const TreeArgs& A, const KeyLayout& kg, const KeyLayout& kl, bool whole, int cb, int round,
                                                 GsSmem& ssm, TreeSmem& tsm, unsigned char* dyn_smem) {
    const unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    const i64 N = A.N;
    const LocalBufs lb = local_bufs(dyn_smem);
    // ---- local stage: every work item is finished by one CTA.  Items: the whole queue (small
    // inputs), else the segments above the quantum (one item each), then the quanta of positions ----
    {
        const u64* K = A.bufs.key[cb];
        const u32* cur = A.bufs.val[cb];
        const u32 nbig = whole ? 0u : __ldcg(&A.ctl->nbig[round % 3]);
        const bool any_unres = whole || __ldcg(&A.ctl->unres[round % 3]) != 0;
        const i64 Q = A.quantum;
        const u32 nq = (u32)((N + Q - 1) / Q);
        int stage = whole ? 0 : 1;  // 0 whole queue, 1 big segments, 2 quanta, 3 done
        while (stage < 3) {
            i64 p0 = 0;
            int n = 0;
            if (stage == 0) {
                n = (int)N;
                stage = 3;
            } else {
                if (threadIdx.x == 0) tsm.item = atomicAdd(stage == 1 ? &A.ctl->next_big : &A.ctl->next_q, 1u);
                __syncthreads();
                const u32 it = tsm.item;
                __syncthreads();
                if (stage == 1) {
                    if (it >= nbig) { stage = 2; continue; }
                    const u64 e = __ldcg(A.biglist + it);
                    p0 = (i64)(u32)e;
                    n = (int)(e >> 32);
                    PEEK_CHECK(n > 0 && n <= LOC_CAP && p0 + n <= N, "big work item out of range");
                } else {
                    if (it >= nq) break;
                    const i64 a = (i64)it * Q, b = min(a + Q, N);
                    if (!any_unres) { tree_direct_output(A, cur, a, b); continue; }
                    // positions at the start of the quantum that belong to a segment begun before
                    // it: resolved ones are written here, an unresolved segment is another item's
                    p0 = a;
                    const u32 sa = __ldcg(A.seg + a);
                    if ((i64)(sa & 0x7fffffffu) < a) {
                        if (threadIdx.x == 0) tsm.red = (u32)(b - a);
                        __syncthreads();
                        u32 first = (u32)(b - a);
                        for (i64 j = a + threadIdx.x; j < b; j += GS_THREADS)
                            if ((i64)(__ldcg(A.seg + j) & 0x7fffffffu) >= a) { first = (u32)(j - a); break; }
                        first = __reduce_min_sync(FULL, first);
                        if (lane == 0 && first < (u32)(b - a)) atomicMin(&tsm.red, first);
                        __syncthreads();
                        p0 = a + tsm.red;
                        __syncthreads();
                        if (!(sa >> 31)) tree_direct_output(A, cur, a, p0);
                    }
                    if (p0 >= b) continue;
                    // the segment holding the quantum's last position started inside the range
                    const u32 sb = __ldcg(A.seg + b - 1);
                    const i64 sl = (i64)(sb & 0x7fffffffu);
                    i64 e = b;
                    if (sb >> 31) {
                        const i64 size = __ldcg(A.gsz + sl);
                        e = size > Q ? sl : sl + size;  // above the quantum: an item of the big list
                    }
                    if (e <= p0) continue;
                    int un_any = 0;  // anything left to refine in [p0, e)?
                    for (i64 j = p0 + threadIdx.x; j < e; j += GS_THREADS) un_any |= (int)(__ldcg(A.seg + j) >> 31);
                    un_any = __syncthreads_or(un_any);
                    if (!un_any) { tree_direct_output(A, cur, p0, e); continue; }
                    n = (int)(e - p0);
                    PEEK_CHECK(n > 0 && n <= LOC_CAP && p0 + n <= N, "quantum work item out of range");
                }
            }
            tree_local(A, kg, kl, K, cur, p0, n, whole ? LOCAL_WHOLE_QUEUE : LOCAL_FROM_GLOBAL, ssm, tsm, lb);
        }
    }
}

// groups and clusters from (order, lcp): three grid-wide phases
// SM: LCP and the min hierarchy live in shared memory (one CTA, small queue): plain loads; else they
// are global arrays other CTAs write between the phases: L2 loads
template <bool SM>
__device__ __forceinline__ void tree_signals(const TreeArgs& A, Grid& g, TreeSmem& tsm, i32* lvl_hi,
                                             const i32* LCP, i32* mt_store) {
    auto ldl = [&](const i32* p) -> i32 { return SM ? *p : __ldcg(p); };
    const unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const unsigned le_mask = 0xffffffffu >> (31 - lane);  // lanes <= this one
    const i64 N = A.N;
    const int G = gridDim.x, me = blockIdx.x;
    const i64 gtid = (i64)me * GS_THREADS + threadIdx.x;
    const u64* __restrict__ H = A.hashes;
    const i64* __restrict__ BO = A.blk_off;
    const i64 C = (N + G - 1) / G;
    const i64 c0 = min((i64)me * C, N), c1 = min(c0 + C, N);
    const int ntiles = (int)((C + GS_TILE - 1) / GS_TILE);
    // rows per warp: a chunk of less than a tile is spread over all warps of the CTA (rows beyond KP
    // are out of range), so small chunks do not leave most warps idle
    const int KP = ntiles == 1 ? (int)((C + GS_THREADS - 1) / GS_THREADS) : GS_KPT;
    auto IDX = [&](int t, int k) -> i64 {
        return k < KP ? c0 + (i64)t * GS_TILE + w * (32 * KP) + k * 32 + lane : (i64)1 << 62;
    };
    (void)FULL; (void)le_mask; (void)gtid; (void)H; (void)BO; (void)ntiles; (void)c1;
    const bool want_groups = A.group_id || A.group_size || A.n_groups;
    const bool want_clusters = A.cluster_depth || A.cluster_size || A.cluster_id;
    if (!want_groups && !want_clusters) return;
    MinTree mt;
    mintree_layout(mt, LCP, N, mt_store);
    const i64 gwarp = gtid >> 5, nwarps = ((i64)G * GS_THREADS) >> 5;

    // ---- G1: per-CTA count of group starts (lcp == 0) and the last one; min-hierarchy level 1 ----
    {
        u32 cntw = 0;
        i32 lastw = -1;
        for (int t = 0; t < ntiles; ++t) {
            i32 lv[GS_KPT];
            ELEMS(k) { const i64 i = IDX(t, k); lv[k] = i < c1 ? ldl(LCP + i) : 1; }
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
                if (i < c1) { lv[k] = ldl(LCP + i); if (i + 1 < N) ln[k] = ldl(LCP + i + 1); }
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
                mt.lvl[k] = lvl_hi + off;
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
                l0[k] = ldl(LCP + i);
                if (i + 1 < N) l1[k] = ldl(LCP + i + 1);
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
            w_cur = i < N ? ldl(LCP + i) : 0;
            w_next = i + 32 < N ? ldl(LCP + i + 32) : 0;
            w_prev = (i >= 32 && i - 32 < N) ? ldl(LCP + i - 32) : 0;
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

// k_tree_global -> k_tree_local -> k_tree_signals on one stream; separate kernels because the three
// stages want different resources (the sort stages tiles in shared memory, the local stage keeps a
// whole work item there, the signals want the L1 instead) and none of them needs the others'
// registers alive.  k_tree_small runs a whole small queue in one CTA, one launch.
__global__ void __launch_bounds__(GS_THREADS, 1) k_tree_global(TreeArgs A) {
    extern __shared__ __align__(16) unsigned char dyn_smem[];
    __shared__ GsSmem ssm;
    __shared__ TreeSmem tsm;
    Grid g{&A.ctl->bar, 0};
    PEEK_MARK(1);
    tree_phase0(A, g);
    const KeyLayout kl = make_layout(A.N, __ldcg(&A.ctl->maxnb), global_wmax(A.N));
    tree_global(A, kl, g, ssm, tsm, gs_stage(dyn_smem));
    PEEK_MARK(14);
}

__global__ void __launch_bounds__(GS_THREADS, 1) k_tree_local(TreeArgs A) {
    extern __shared__ __align__(16) unsigned char dyn_smem[];
    __shared__ GsSmem ssm;
    __shared__ TreeSmem tsm;
    PEEK_MARK(15);
    const KeyLayout kg = make_layout(A.N, __ldcg(&A.ctl->maxnb), global_wmax(A.N)), kl = make_layout(A.N, __ldcg(&A.ctl->maxnb), LOC_W);
    tree_local_stage(A, kg, kl, false, (int)__ldcg(&A.ctl->fin_cb), (int)__ldcg(&A.ctl->fin_round), ssm, tsm, dyn_smem);
    PEEK_MARK(20);
}

__global__ void __launch_bounds__(GS_THREADS, 1) k_tree_signals(TreeArgs A) {
    __shared__ TreeSmem tsm;
    __shared__ i32 lvl_hi[LVL_HI_WORDS];
    Grid g{&A.ctl->bar2, 0};
    PEEK_MARK(23);
    tree_signals<false>(A, g, tsm, lvl_hi, A.lcp, A.mt_buf);
}

__global__ void __launch_bounds__(GS_THREADS, 1) k_tree_small(TreeArgs A) {
    extern __shared__ __align__(16) unsigned char dyn_smem[];
    __shared__ GsSmem ssm;
    __shared__ TreeSmem tsm;
    Grid g{&A.ctl->bar, 0};  // one CTA: every grid barrier is a CTA barrier
    PEEK_MARK(1);
    // one CTA: the control block is cleared here instead of by a memset node before the launch
    for (int i = threadIdx.x; i < (int)(sizeof(TreeCtl) / 4); i += GS_THREADS) ((u32*)A.ctl)[i] = 0;
    __syncthreads();
    tree_phase0(A, g);
    const KeyLayout kl = make_layout(A.N, __ldcg(&A.ctl->maxnb), LOC_W);
    tree_local_stage(A, kl, kl, true, 0, 0, ssm, tsm, dyn_smem);
    __syncthreads();
    PEEK_MARK(23);
    {   // the work item's buffers are free now: LCP and the min hierarchy move into shared memory, so
        // the nearest-smaller-value walks of the cluster search cost shared-memory latency
        i32* slcp = (i32*)dyn_smem;
        const i64 N = A.N;
        for (i64 i = threadIdx.x; i < N; i += GS_THREADS) slcp[i] = A.lcp[i];
        i32* smt = slcp + ((N + 1 + 63) / 64) * 64;
        i32* shi = smt + mintree_words(N);
        __syncthreads();
        tree_signals<true>(A, g, tsm, shi, slcp, smt);
    }
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
    A.rec = a.take<ReqRec>(N);
    A.seghead = a.take<u64>(N);
    A.segdepth = a.take<i32>(N);
    A.agg = a.take<i64>(grid);
    A.gsz = a.take<i32>(N);
    A.biglist = a.take<u64>(N / 64 + 64);
    A.posna = a.take<unsigned short>(N);
    A.segrec = a.take<SegRec>(N);
    A.mt_buf = a.take<i32>(mintree_words(N));
}

static constexpr int MAX_GRID = 1024;  // upper bound on the cooperative grid (workspace sizing)

i64 pending_tree_ws_bytes(i64 N) {
    Arena a(nullptr);
    TreeArgs A;
    tree_layout(a, N, MAX_GRID, A);
    return a.used;
}

static int g_tree_local_cap = 0;  // PEEK_OPT_TREE_LOCAL_CAP (0 = automatic)
static constexpr int TREE_SMALL_MAX = 2048;  // queues up to this size run in one CTA from the first step on
void tree_set_option(int key, i64 v) {
    if (key == PEEK_OPT_TREE_LOCAL_CAP) g_tree_local_cap = (int)v;
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
    // what one CTA finishes alone: segments of up to cap_seg positions; those above the quantum are
    // work items of their own, the others are taken a quantum of positions at a time
    if (g_tree_local_cap >= 128 && g_tree_local_cap < LOC_CAP) {  // test hook
        A.cap_seg = g_tree_local_cap;
        A.quantum = A.cap_seg / 2;
    } else if (N <= TREE_SMALL_MAX) {  // the whole queue is one work item of one CTA
        A.cap_seg = LOC_CAP;
        A.quantum = LOC_CAP / 2;
    } else {
        // a work item occupies one SM: mid-size queues get smaller items (and, for their few big
        // segments, more grid-wide rounds) so that the local stage has enough of them to fill the GPU
        const i64 c = N / 8;
        A.cap_seg = (int)(c < 1024 ? 1024 : (c > LOC_CAP ? LOC_CAP : c));
        i64 q = ((N / (2 * (i64)sm_count()) + 127) / 128) * 128;
        if (q < 256) q = 256;
        if (q > A.cap_seg / 2 || c >= LOC_CAP) q = A.cap_seg / 2;  // big queues: plenty of items anyway, fewer is cheaper
        A.quantum = (int)q;
    }
    tree_layout(a, N, MAX_GRID, A);
    void* params[] = {&A};
    const bool want_signals = group_id || group_size || n_groups || cluster_depth || cluster_size || cluster_id;
    const bool whole = !signals_only && N <= (i64)A.cap_seg && (N <= TREE_SMALL_MAX || g_tree_local_cap > 0);
    if (!whole)
        PEEK_CUDA(cudaMemsetAsync(A.ctl, 0, (size_t)((char*)(A.bufs.hist + gs_hist_words(MAX_GRID)) - (char*)A.ctl), st));
    a.arm(st);
    if (whole) {  // the whole queue in one CTA, one launch, no grid barrier
        Prof pr(PROF_TREE, st, 1);
        PEEK_CUDA(func_smem_optin((const void*)k_tree_small, TREE_DYN_SMEM));
        k_tree_small<<<1, GS_THREADS, TREE_DYN_SMEM, st>>>(A);
        PEEK_CUDA(cudaGetLastError());
        return PEEK_OK;
    }
    Prof pr(PROF_TREE, st, (signals_only ? 0 : 2) + (want_signals ? 1 : 0));
    if (!signals_only) {
        PEEK_CUDA(func_smem_optin((const void*)k_tree_global, GS_STAGE_BYTES));
        PEEK_CUDA(cudaLaunchCooperativeKernel((const void*)k_tree_global, dim3(grid), dim3(GS_THREADS), params,
                                              GS_STAGE_BYTES, st));
        PEEK_CUDA(func_smem_optin((const void*)k_tree_local, TREE_DYN_SMEM));
        // the local stage's CTAs draw work items from queues: as many CTAs as there can be items
        i64 lgrid = (N + A.quantum - 1) / A.quantum + N / (A.quantum + 1) + 1;
        const int lmax = persistent_ctas() < MAX_GRID ? persistent_ctas() : MAX_GRID;
        if (lgrid > lmax) lgrid = lmax;
        k_tree_local<<<(unsigned)lgrid, GS_THREADS, TREE_DYN_SMEM, st>>>(A);
        PEEK_CUDA(cudaGetLastError());
    }
    if (want_signals)
        PEEK_CUDA(cudaLaunchCooperativeKernel((const void*)k_tree_signals, dim3(grid), dim3(GS_THREADS), params, 0, st));
    return PEEK_OK;
}

extern "C" peek_status peek_pending_tree(const uint64_t* hashes, const int64_t* blk_off, int64_t N,
                                         int32_t* order, int32_t* lcp, int32_t* group_id,
                                         int32_t* group_size, int32_t* cluster_depth,
                                         int32_t* cluster_size, int64_t* cluster_id, int32_t* n_groups,
                                         void* ws, int64_t ws_bytes, void* stream) {
    if (N < 0 || N >= 0x7fffffffLL) { set_error("peek_pending_tree: N out of range"); return PEEK_ERR_INVALID_ARG; }
    if (N == 0) return PEEK_OK;
    if (!hashes || !blk_off || !order || !lcp) { set_error("peek_pending_tree: NULL argument"); return PEEK_ERR_INVALID_ARG; }
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

// ordered grid-wide inclusive scan (associative op, NOT necessarily commutative).  A thread owns
// UP_ITEMS consecutive elements of a step and has all their loads in flight at once (the loads of
// the compaction are dependent gathers), so a CTA's chunk takes a quarter of the steps - and of the
// CTA barriers - that one element per thread would.  xch: blockDim.x elements of shared memory.
static constexpr int UP_ITEMS = 4;
template <typename T, typename Op, typename Load, typename Store>
__device__ void grid_inscan_ordered(i64 n, Load load, Store store, Op op, T ident, T* agg, T* smem, T* xch, Grid& g) {
    const i64 step = (i64)blockDim.x * UP_ITEMS;
    const i64 chunk = (((n + gridDim.x - 1) / gridDim.x) + step - 1) / step * step;
    const i64 c0 = min((i64)blockIdx.x * chunk, n), c1 = min(c0 + chunk, n);
    T carry = ident;
    for (i64 b = c0; b < c1; b += step) {
        const i64 i0 = b + (i64)threadIdx.x * UP_ITEMS;
        T v[UP_ITEMS];
#pragma unroll
        for (int k = 0; k < UP_ITEMS; ++k) v[k] = i0 + k < c1 ? load(i0 + k) : ident;
        T t = v[0];
#pragma unroll
        for (int k = 1; k < UP_ITEMS; ++k) t = op(t, v[k]);
        T tt;
        block_inscan(t, op, ident, smem, &tt);
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
    for (i64 b = c0; b < c1; b += step) {
        const i64 i0 = b + (i64)threadIdx.x * UP_ITEMS;
        T v[UP_ITEMS];
#pragma unroll
        for (int k = 0; k < UP_ITEMS; ++k) v[k] = i0 + k < c1 ? load(i0 + k) : ident;
#pragma unroll
        for (int k = 1; k < UP_ITEMS; ++k) v[k] = op(v[k - 1], v[k]);  // inclusive inside the thread
        T tt;
        const T inc = block_inscan(v[UP_ITEMS - 1], op, ident, smem, &tt);
        xch[threadIdx.x] = inc;  // the threads before this one = the inclusive value of its left neighbour
        __syncthreads();
        const T before = op(carry, threadIdx.x ? xch[threadIdx.x - 1] : ident);
        __syncthreads();
#pragma unroll
        for (int k = 0; k < UP_ITEMS; ++k)
            if (i0 + k < c1) store(i0 + k, op(before, v[k]));
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
    __shared__ u64 xch[UP_THREADS];
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
                                 upd_pack(0, 0x7fffffffu, 0), A.agg, s64, xch, g);
    }
    const i64 S = A.N_old > 0 ? __ldcg(&A.ctl->S) : 0;
    // ---- 3: every arrival bisects for its place among the survivors ----
    const i64 first_new = A.N_new - A.M;
    if (A.M * 32 <= gsize) {
        // few arrivals (the steady state of a serving loop): a warp per arrival, 32 pivots per step.
        // A comparison is ~10 dependent trips (offsets, the depth bisection of chain_lcp, the branch
        // words); 4 steps of 32 side by side instead of 20 one after the other.
        const unsigned FULL = 0xffffffffu;
        const int lane = threadIdx.x & 31;
        const i64 q = gtid >> 5;
        if (q < A.M) {
            const i64 x = first_new + __ldg(A.b_order + q);
            i64 lo = 0, hi = S;  // survivors before lo sort at or before x, from hi on after x
            while (lo < hi) {
                const i64 len = hi - lo;
                const bool wide = len >= 32;
                auto pivot = [&](int l) -> i64 { return wide ? lo + (len * (l + 1)) / 33 : lo + l; };
                bool before = false;  // this lane's survivor sorts at or before x
                if (wide || lane < len) {
                    i32 l;
                    before = upd_cmp(H, BO, x, __ldcg(A.s_order + pivot(lane)), &l) > 0;
                }
                const int c = __popc(__ballot_sync(FULL, before));  // sorted survivors: a prefix of the lanes
                if (wide) {
                    const i64 nlo = c ? pivot(c - 1) + 1 : lo, nhi = c < 32 ? pivot(c) : hi;
                    lo = nlo; hi = nhi;
                } else {
                    lo += c; hi = lo;
                }
            }
            i32 l = 0;
            if (lane == 0 && lo > 0) upd_cmp(H, BO, x, __ldcg(A.s_order + lo - 1), &l);
            if (lane == 1 && lo < S) upd_cmp(H, BO, x, __ldcg(A.s_order + lo), &l);
            const i32 lR = __shfl_sync(FULL, l, 1);
            if (lane == 0) {
                A.ins[q] = (i32)lo; A.lcpL[q] = l; A.lcpR[q] = lR;
                atomicAdd((unsigned long long*)(A.hist + lo), 1ull);
            }
        }
    } else
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
        grid_inscan_ordered<u64>(S + 1, load, store, [](u64 a, u64 b) { return a + b; }, (u64)0, A.agg, s64, xch, g);
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
    if (!hashes || !blk_off || !order || !lcp || (N_old > 0 && (!old_order || !old_lcp || !remap))) {
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
    a.arm(st);
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
