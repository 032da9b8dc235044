// peek_interleave.cu — a11d: stride interleave of the two admission lanes (Alg. 2 line 22,
// PAPER.md:325, :111; R28).
//
// Slot k belongs to Lane A iff floor((k+1) alpha) > floor(k alpha); the lane admits its first
// request not admitted yet.  The walk is sequential across slots (a lane skips what the other one
// admitted), so ONE CTA runs it, SI_T = 1024 slots per step, every phase of a step in parallel:
//   1  slot types of the step, rank of each slot within its lane (ballot scan)
//   2  candidates: the first not-admitted entries of each list from its cursor (coalesced window
//      reads, a bitmap of admitted requests in shared memory when it fits, ordered compaction) - as
//      many as the lane has slots in the step plus SI_MARGIN for what it may have to skip; if a lane
//      turns out to need more, the step is redone with `cnt` candidates each, which always suffice
//   3  clashes = requests that are candidates of BOTH lanes, found through a stamped shared-memory
//      hash table (never cleared: an entry of an older step reads as empty)
//   4  no clash (the common case): A's i-th slot takes candidate i of A, B's j-th candidate j of B.
//      Else the clashes - and only they - are resolved in time order by one thread: with the clash
//      lists sorted by candidate index on either side, lane X reaches its first unresolved clash x
//      at its slot number (index of x) - (clashes before x that the other lane took); the earlier
//      of the two fronts is final, because a lane reaches later candidates no earlier.  Then the
//      candidates a lane lost are compacted away and slot i takes the lane's i-th survivor.
//      Many clashes (correlated lanes, e.g. a cold cache where cLPM order = arrival order): warp 0
//      walks the step's slots instead, in lock step, with each lane's still-available candidates
//      as bit masks in registers (a slot = find-first-set + one broadcast shared-memory load of the
//      partner index), which bounds a step at ~35 cycles per slot whatever the lanes look like.
//   5  results, bitmap and cursors (everything before a lane's last admitted entry is admitted).
// Shortcut: while both lanes' candidate lists start with the same L requests in the same order, slot t
// takes candidate t whatever its type (both lanes want the same request), so a step whose lists
// agree on L >= SI_RUN candidates admits exactly those and the next step starts L slots later.
#include "peek_common.cuh"

namespace peek {
static constexpr int SI_T = 1024;   // threads of the CTA = slots per step
static constexpr int SI_H = 4096;   // hash table entries (<= 1024 keys per step)
static constexpr int SI_WIN = 2;    // list entries per thread and window read
static constexpr int SI_MARGIN = 128;  // candidates gathered beyond a lane's own slots (first attempt)
static constexpr int SI_RUN = 64;   // common run of both lanes' candidates from which the step is cut short

struct SiSmem {
    i32 CA[SI_T], CB[SI_T];              // candidates (request ids) of the step
    i32 PA[SI_T], PB[SI_T];              // their list positions
    unsigned short slotA[SI_T], slotB[SI_T];  // slot (within the step) of a lane's i-th slot
    short clA[SI_T], clB[SI_T];          // clash partner: by A index -> B index, by B index -> A index; -1 none
    unsigned short LA[SI_T], LB[SI_T];   // clash lists: A indices ascending, B indices ascending
    unsigned short avA[SI_T], avB[SI_T]; // surviving candidates of each lane, in order
    unsigned char res[SI_T];             // by A index: 0 unresolved, 1 taken by A, 2 taken by B
    unsigned long long H[SI_H];          // stamp:21 | request:31 | A index:11
    int wc[2][2][32];                    // per-warp counts of the two-flag scans (double buffered)
    u32 types[32];                       // bit q of word c: slot 32c + q of the step belongs to Lane A
    i64 curA, curB;
    int firstdiff;                       // first candidate index at which the two lanes differ
};

static_assert(sizeof(SiSmem) + 160 * 1024 <= 227 * 1024, "SiSmem + bitmap must fit in shared memory");

// volatile: the bitmap changes under the CTA's own atomics (and may live in global memory)
__device__ __forceinline__ bool si_bit(const u32* bits, i32 r) {
    return (((const volatile u32*)bits)[r >> 5] >> (r & 31)) & 1u;
}
__device__ __forceinline__ u32 si_hash(i32 r) { return ((u32)r * 2654435761u) >> 20; }

// Exclusive offsets of this warp for two per-warp counts (cx, cy uniform in the warp), and the
// block totals.  One __syncthreads.
__device__ __forceinline__ void si_offsets2(SiSmem& S, int& buf, int lane, int w, int cx, int cy, int& px,
                                            int& py, int& tx, int& ty) {
    const unsigned FULL = 0xffffffffu;
    if (lane == 0) { S.wc[buf][0][w] = cx; S.wc[buf][1][w] = cy; }
    __syncthreads();
    int ax = S.wc[buf][0][lane], ay = S.wc[buf][1][lane];
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const int vx = __shfl_up_sync(FULL, ax, d), vy = __shfl_up_sync(FULL, ay, d);
        if (lane >= d) { ax += vx; ay += vy; }
    }
    tx = __shfl_sync(FULL, ax, 31);
    ty = __shfl_sync(FULL, ay, 31);
    px = __shfl_sync(FULL, ax, w) - cx;
    py = __shfl_sync(FULL, ay, w) - cy;
    buf ^= 1;
}

__global__ void __launch_bounds__(SI_T, 1) k_stride_interleave(const i32* __restrict__ lane_a,
                                                              const i32* __restrict__ lane_b, i64 N, double alpha,
                                                              i32* __restrict__ out, u32* gbits, int use_smem) {
    extern __shared__ __align__(16) unsigned char si_raw[];
    SiSmem& S = *reinterpret_cast<SiSmem*>(si_raw);
    u32* si_bits = reinterpret_cast<u32*>(si_raw + sizeof(SiSmem));
    const unsigned FULL = 0xffffffffu;
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const unsigned lt = (1u << lane) - 1u;
    u32* bits = use_smem ? si_bits : gbits;
    const i64 words = (N + 31) >> 5;
    for (i64 x = tid; x < words; x += SI_T) bits[x] = 0;
    for (int x = tid; x < SI_H; x += SI_T) S.H[x] = 0;
    __syncthreads();
    int buf = 0;
    i64 mA = 0, mB = 0;
    unsigned long long stamp = 0;
    i64 k0 = 0;
    int margin = SI_MARGIN;
    while (k0 < N) {
        const int cnt = (int)(N - k0 < SI_T ? N - k0 : SI_T);
        // the stamp has 22 bits in a table entry: when it wraps, every entry is cleared (0 = never used)
        if (++stamp >> 22) {
            __syncthreads();
            for (int x = tid; x < SI_H; x += SI_T) S.H[x] = 0;
            __syncthreads();
            stamp = 1;
        }
        // ---- 1: slot types ----
        const i64 s = k0 + tid;
        const bool live = tid < cnt;
        const bool from_a = live && (i64)__dmul_rn((double)(s + 1), alpha) > (i64)__dmul_rn((double)s, alpha);
        const unsigned balA = __ballot_sync(FULL, from_a);
        int rA, nA, dum0, dum1;
        si_offsets2(S, buf, lane, w, __popc(balA), 0, rA, dum0, nA, dum1);
        rA += __popc(balA & lt);
        const int rB = tid - rA, nB = cnt - nA;
        if (live) {
            if (from_a) S.slotA[rA] = (unsigned short)tid;
            else S.slotB[rB] = (unsigned short)tid;
        }
        if (lane == 0) S.types[w] = balA;
        const int wantA = nA + margin < cnt ? nA + margin : cnt, wantB = nB + margin < cnt ? nB + margin : cnt;
        const int wmin = wantA < wantB ? wantA : wantB;
        if (tid == 0) S.firstdiff = wmin;
        S.clA[tid] = -1;
        S.clB[tid] = -1;
        S.res[tid] = 0;
        // ---- 2: candidates ----
        int fA = 0, fB = 0;
        i64 wA = mA, wB = mB;
        for (;;) {
            const bool needA = fA < wantA && wA < N, needB = fB < wantB && wB < N;
            if (!needA && !needB) break;
            i32 a[SI_WIN], b[SI_WIN];
            bool ga[SI_WIN], gb[SI_WIN];
            const i64 pa = wA + (i64)SI_WIN * tid, pb = wB + (i64)SI_WIN * tid;
#pragma unroll
            for (int u = 0; u < SI_WIN; ++u) {
                a[u] = needA && pa + u < N ? __ldg(lane_a + pa + u) : -1;
                b[u] = needB && pb + u < N ? __ldg(lane_b + pb + u) : -1;
            }
            int ca = 0, cb = 0, ia = 0, ib = 0;  // warp totals, counts of the lower lanes
#pragma unroll
            for (int u = 0; u < SI_WIN; ++u) {
                ga[u] = a[u] >= 0 && !si_bit(bits, a[u]);
                gb[u] = b[u] >= 0 && !si_bit(bits, b[u]);
                const unsigned qa = __ballot_sync(FULL, ga[u]), qb = __ballot_sync(FULL, gb[u]);
                ca += __popc(qa); cb += __popc(qb);
                ia += __popc(qa & lt); ib += __popc(qb & lt);
            }
            int oa, ob, ta, tb;
            si_offsets2(S, buf, lane, w, ca, cb, oa, ob, ta, tb);
            int ra = fA + oa + ia, rb = fB + ob + ib;
#pragma unroll
            for (int u = 0; u < SI_WIN; ++u) {
                if (ga[u]) { if (ra < wantA) { S.CA[ra] = a[u]; S.PA[ra] = (i32)(pa + u); } ++ra; }
                if (gb[u]) { if (rb < wantB) { S.CB[rb] = b[u]; S.PB[rb] = (i32)(pb + u); } ++rb; }
            }
            fA += ta; fB += tb;
            if (needA) wA += (i64)SI_WIN * SI_T;
            if (needB) wB += (i64)SI_WIN * SI_T;
        }
        __syncthreads();  // candidates, slot tables and the cleared clash arrays are visible
        // ---- 3: clashes (every request is on both lists, so both have >= cnt candidates) ----
        const bool hasA = tid < wantA, hasB = tid < wantB;
        i32 mineA = -1, mineB = -1;
        if (hasA) mineA = S.CA[tid];
        if (hasB) mineB = S.CB[tid];
        const unsigned diff = __ballot_sync(FULL, tid < wmin && mineA != mineB);
        if (diff && lane == 0) atomicMin(&S.firstdiff, 32 * w + __ffs(diff) - 1);
        if (hasA) {
            const unsigned long long e = stamp << 42 | (unsigned long long)(u32)mineA << 11 | (unsigned)tid;
            u32 h = si_hash(mineA);
            for (;;) {
                unsigned long long cur = S.H[h];
                if ((cur >> 42) != stamp) {
                    const unsigned long long old = atomicCAS(&S.H[h], cur, e);
                    if (old == cur) break;
                    if ((old >> 42) != stamp) continue;  // lost to an equally stale view: retry this entry
                }
                h = (h + 1) & (SI_H - 1);
            }
        }
        __syncthreads();
        const int L = S.firstdiff;
        if (L == cnt || L >= SI_RUN) {  // a common run: slot t takes candidate t
            if (tid < L) {
                out[s] = mineA;
                atomicOr(&bits[mineA >> 5], 1u << (mineA & 31));
                if (tid == L - 1) { S.curA = (i64)S.PA[tid] + 1; S.curB = (i64)S.PB[tid] + 1; }
            }
            __syncthreads();
            mA = S.curA;
            mB = S.curB;
            k0 += L;
            // correlated lanes: stay with (or move to) full candidate lists while the runs last
            margin = margin == SI_T || (L == wmin && wmin < cnt) ? SI_T : SI_MARGIN;
            continue;
        }
        bool clash = false;
        if (hasB) {
            u32 h = si_hash(mineB);
            for (;;) {
                const unsigned long long cur = S.H[h];
                if ((cur >> 42) != stamp) break;
                if ((i32)((cur >> 11) & 0x7fffffffu) == mineB) {
                    const int ja = (int)(cur & 0x7ffu);
                    S.clB[tid] = (short)ja;
                    S.clA[ja] = (short)tid;
                    clash = true;
                    break;
                }
                h = (h + 1) & (SI_H - 1);
            }
        }
        const int m_any = __syncthreads_or(clash);
        // ---- 4: who takes what ----
        i32 pick = -1, ppos = 0;
        bool dense = false;
        if (!m_any) {
            if (live) {
                pick = from_a ? S.CA[rA] : S.CB[rB];
                ppos = from_a ? S.PA[rA] : S.PB[rB];
            }
        } else {
            const bool inA = hasA && S.clA[tid] >= 0, inB = hasB && S.clB[tid] >= 0;
            const unsigned qa = __ballot_sync(FULL, inA), qb = __ballot_sync(FULL, inB);
            int oa, ob, m, m2;
            si_offsets2(S, buf, lane, w, __popc(qa), __popc(qb), oa, ob, m, m2);
            if (inA) S.LA[oa + __popc(qa & lt)] = (unsigned short)tid;
            if (inB) S.LB[ob + __popc(qb & lt)] = (unsigned short)tid;
            dense = 3 * m >= cnt;
            if (dense) {  // a slot of the walk costs about a third of an event of the loop below
                if (margin < cnt) { margin = SI_T; continue; }  // the walk wants `cnt` candidates per lane
                __syncthreads();
                if (w == 0) {  // lane l holds the availability of candidates 32l .. 32l+31 of either lane
                    const int rem = cnt - 32 * lane;
                    u32 avA = rem >= 32 ? FULL : (rem > 0 ? (1u << rem) - 1u : 0u), avB = avA;
                    int wa = 0, wb = 0, na = 0, nb = 0;
                    u32 fA = __shfl_sync(FULL, avA, 0), fB = fA;  // the lanes' front words, uniform copies
                    for (int c = 0; 32 * c < cnt; ++c) {
                        const u32 types = S.types[c];
                        const int nq = cnt - 32 * c < 32 ? cnt - 32 * c : 32;
                        for (int q = 0; q < nq; ++q) {
                            if ((types >> q) & 1u) {
                                if (!fA) {
                                    wa = __ffs(__ballot_sync(FULL, avA != 0)) - 1;
                                    fA = __shfl_sync(FULL, avA, wa);
                                }
                                const int idx = 32 * wa + __ffs(fA) - 1;
                                fA &= fA - 1;
                                if (lane == wa) avA = fA;
                                const int p = S.clA[idx];
                                if (p >= 0) {
                                    const u32 bit = 1u << (p & 31);
                                    if (lane == (p >> 5)) avB &= ~bit;
                                    if ((p >> 5) == wb) fB &= ~bit;
                                }
                                if (lane == 0) S.avA[na] = (unsigned short)idx;
                                ++na;
                            } else {
                                if (!fB) {
                                    wb = __ffs(__ballot_sync(FULL, avB != 0)) - 1;
                                    fB = __shfl_sync(FULL, avB, wb);
                                }
                                const int idx = 32 * wb + __ffs(fB) - 1;
                                fB &= fB - 1;
                                if (lane == wb) avB = fB;
                                const int p = S.clB[idx];
                                if (p >= 0) {
                                    const u32 bit = 1u << (p & 31);
                                    if (lane == (p >> 5)) avA &= ~bit;
                                    if ((p >> 5) == wa) fA &= ~bit;
                                }
                                if (lane == 0) S.avB[nb] = (unsigned short)idx;
                                ++nb;
                            }
                        }
                    }
                }
                __syncthreads();
            } else {
                __syncthreads();
                if (tid == 0) {
                    int ia = 0, ib = 0, dA = 0, dB = 0;
                    for (;;) {
                        while (ia < m && S.res[S.LA[ia]] != 0) { ++dA; ++ia; }  // only B's takes wait at A's front
                        while (ib < m) {
                            const unsigned char r = S.res[S.clB[S.LB[ib]]];
                            if (r == 0) break;
                            dB += r == 1;
                            ++ib;
                        }
                        int tA = 1 << 20, tB = 1 << 20;
                        if (ia < m) { const int sa = (int)S.LA[ia] - dA; if (sa < nA) tA = S.slotA[sa]; }
                        if (ib < m) { const int sb = (int)S.LB[ib] - dB; if (sb < nB) tB = S.slotB[sb]; }
                        if (tA == tB) break;  // both lanes are out of slots
                        if (tA < tB) { S.res[S.LA[ia]] = 1; ++ia; }
                        else { S.res[S.clB[S.LB[ib]]] = 2; ++ib; }
                    }
                }
                __syncthreads();
                // survivors of each lane: candidates the other lane did not take
                const bool svA = hasA && !(S.res[tid] == 2);
                const bool svB = hasB && !(S.clB[tid] >= 0 && S.res[S.clB[tid]] == 1);
                const unsigned va = __ballot_sync(FULL, svA), vb = __ballot_sync(FULL, svB);
                int t0, t1;
                si_offsets2(S, buf, lane, w, __popc(va), __popc(vb), oa, ob, t0, t1);
                if (t0 < nA || t1 < nB) { margin = SI_T; continue; }  // a lane skipped more than the margin
                if (svA) S.avA[oa + __popc(va & lt)] = (unsigned short)tid;
                if (svB) S.avB[ob + __popc(vb & lt)] = (unsigned short)tid;
                __syncthreads();
            }
            if (live) {
                const int j = from_a ? S.avA[rA] : S.avB[rB];
                pick = from_a ? S.CA[j] : S.CB[j];
                ppos = from_a ? S.PA[j] : S.PB[j];
            }
        }
        // ---- 5: results, bitmap, cursors ----
        if (live) {
            out[s] = pick;
            atomicOr(&bits[pick >> 5], 1u << (pick & 31));
            if (from_a && rA == nA - 1) S.curA = (i64)ppos + 1;
            if (!from_a && rB == nB - 1) S.curB = (i64)ppos + 1;
        }
        __syncthreads();
        if (nA > 0) mA = S.curA;
        if (nB > 0) mB = S.curB;
        k0 += cnt;
        margin = m_any && margin == SI_T && dense ? SI_T : SI_MARGIN;  // the slot walk wants full lists again
    }
}
}  // namespace peek

using namespace peek;

static const i64 SI_SMEM_BITS = 160 * 1024;  // bitmap bytes that fit in shared memory beside SiSmem

extern "C" peek_status peek_stride_interleave(const int32_t* lane_a, const int32_t* lane_b, int64_t N,
                                              double alpha, int32_t* out, void* ws, int64_t ws_bytes,
                                              void* stream) {
    if (N < 0 || N >= 0x7fffffffLL || !(alpha >= 0.0 && alpha <= 1.0)) {
        set_error("peek_stride_interleave: N out of range or alpha outside [0, 1]");
        return PEEK_ERR_INVALID_ARG;
    }
    if (N == 0) return PEEK_OK;
    if (!lane_a || !lane_b || !out) { set_error("peek_stride_interleave: NULL argument"); return PEEK_ERR_INVALID_ARG; }
    const i64 bytes = ((N + 31) / 32) * 4;
    const int use_smem = bytes <= SI_SMEM_BITS;
    if (!use_smem && (!ws || ((uintptr_t)ws & 255) || ws_bytes < bytes)) {
        set_error("peek_stride_interleave: workspace NULL, misaligned or too small");
        return PEEK_ERR_WORKSPACE;
    }
    PEEK_CUDA(func_smem_optin((const void*)k_stride_interleave, (int)(sizeof(SiSmem) + SI_SMEM_BITS)));
    cudaStream_t st = (cudaStream_t)stream;
    Prof pr(PROF_RANK_FULL, st, 1);
    k_stride_interleave<<<1, SI_T, sizeof(SiSmem) + (use_smem ? (size_t)bytes : 0), st>>>(lane_a, lane_b, N, alpha, out, (u32*)ws,
                                                                       use_smem);
    PEEK_CUDA(cudaGetLastError());
    return PEEK_OK;
}
