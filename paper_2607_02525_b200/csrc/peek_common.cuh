// peek_common.cuh — shared host/device helpers of libpeek.so (sm_100a only).
// Nothing here is shared with oracle/: the constants and the mixer below are this
// library's own statement of DESIGN.md R1.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include "../../include/peek.h"

typedef uint64_t u64;
typedef int64_t i64;
typedef int32_t i32;
typedef uint32_t u32;

namespace peek {

// ---- host side ---------------------------------------------------------------------------
void set_error(const char* fmt, ...);
peek_status cuda_fail(cudaError_t e, const char* what);
int sm_count();  // SMs of the current device (148 on B200)
int persistent_ctas();  // grid of the persistent cooperative kernels (PEEK_OPT_GRID_LIMIT)
// opt `func` in to `bytes` of dynamic shared memory on the CURRENT device (the attribute belongs to the
// device's context, so it is remembered per device; thread-safe)
bool grid_limited();
cudaError_t func_smem_optin(const void* func, int bytes);
// A library-owned side stream per device for calls that run two independent kernels side by side
// (fork: `side` waits for `fork` recorded on the caller's stream; join: the caller's stream waits
// for `join` recorded on `side`).  side_fork returns false when the call must stay on one stream
// (a stream under capture, or no side stream could be made); on true it
// holds side_mutex() until side_join, so two host threads never interleave their record/wait pairs.
struct SideStream { cudaStream_t side; cudaEvent_t fork, join; };
bool side_fork(cudaStream_t st, SideStream* ss);
cudaError_t side_join(cudaStream_t st, const SideStream& ss);

// tracing slots (peek_profile_*)
enum ProfSlot {
    PROF_HASH_SCAN = 0, PROF_HASH_CONTENT, PROF_HASH_CHAIN, PROF_TREE, PROF_LPM_RADIX, PROF_LPM_HASH,
    PROF_LPM_RESOLVE, PROF_LPM_DUAL, PROF_DEMAND, PROF_RANK, PROF_SIGNALS, PROF_RANK_FULL, PROF_OFFLINE, PROF_NSLOTS
};
void prof_begin(int slot, cudaStream_t st);
void prof_end(int slot, cudaStream_t st, int launches);
struct Prof {  // brackets the kernels launched during its lifetime
    int slot, launches;
    cudaStream_t st;
    Prof(int s, cudaStream_t stream, int n) : slot(s), launches(n), st(stream) { prof_begin(slot, st); }
    ~Prof() { prof_end(slot, st, launches); }
};

#define PEEK_CUDA(call)                                            \
    do {                                                           \
        cudaError_t e__ = (call);                                  \
        if (e__ != cudaSuccess) return peek::cuda_fail(e__, #call); \
    } while (0)

static inline i64 align_up(i64 x, i64 a) { return (x + a - 1) / a * a; }

// ---- checked build (-DPEEK_CHECKED: libpeek_checked.so) ---------------------------------------
// compute-sanitizer is closed on this pool, so memory safety gets a build of its own: every index
// computed from device data is range-checked against the extent the arrays were passed with
// (PEEK_CHECK: trap), and every piece of workspace is followed by a 256-byte canary that
// is armed before the call's first kernel and verified after its last one.
// A failed check traps (the call's stream reports a launch failure at the next synchronisation).
// -DPEEK_CHECK_PRINT also prints the source line first; a device printf inside the big persistent
// kernels needs more than the default 1 KB of stack (cudaLimitStackSize), so it is off by default.
#if defined(PEEK_CHECKED) && defined(PEEK_CHECK_PRINT)
#define PEEK_CHECK(cond, what)                                                                   \
    do {                                                                                         \
        if (!(cond)) {                                                                           \
            printf("PEEK_CHECKED %s:%d: %s\n", __FILE__, __LINE__, what);                        \
            __trap();                                                                            \
        }                                                                                        \
    } while (0)
#elif defined(PEEK_CHECKED)
#define PEEK_CHECK(cond, what) do { if (!(cond)) __trap(); } while (0)
#endif
#ifdef PEEK_CHECKED
static constexpr int CANARY_MAX = 48;
struct CanaryList { long long off[CANARY_MAX]; int n; };
static __global__ void k_canary(unsigned char* base, CanaryList L, int verify) {
    const int p = blockIdx.x;
    if (p >= L.n) return;
    unsigned char* c = base + L.off[p] + threadIdx.x;
    if (!verify) *c = 0xC5;
    else if (*c != 0xC5) {
        printf("PEEK_CHECKED workspace canary %d (offset %lld) overwritten at byte %d\n", p, L.off[p], (int)threadIdx.x);
        __trap();
    }
}
#else
#define PEEK_CHECK(cond, what) do { } while (0)
#endif

// Bump allocator over the caller's workspace (256-byte aligned pieces).
struct Arena {
    char* base;
    i64 used;
    explicit Arena(void* p) : base((char*)p), used(0) {}
    template <typename T>
    T* take(i64 n) {
        T* r = (T*)(base ? base + used : nullptr);
        used += align_up((n > 0 ? n : 1) * (i64)sizeof(T), 256);
#ifdef PEEK_CHECKED
        if (canaries.n < CANARY_MAX) canaries.off[canaries.n++] = used;
        used += 256;
#endif
        return r;
    }
#ifdef PEEK_CHECKED
    CanaryList canaries{{0}, 0};
    cudaStream_t armed_on = nullptr;
    bool armed = false;
    // after the call's memsets, before its first kernel
    void arm(cudaStream_t st) {
        if (!base || !canaries.n) return;
        k_canary<<<canaries.n, 256, 0, st>>>((unsigned char*)base, canaries, 0);
        armed = true;
        armed_on = st;
    }
    ~Arena() {  // after the call's last kernel has been enqueued
        if (armed) k_canary<<<canaries.n, 256, 0, armed_on>>>((unsigned char*)base, canaries, 1);
    }
#else
    void arm(cudaStream_t) {}
#endif
};

// ---- device side -------------------------------------------------------------------------
#define PEEK_EMPTY 0xFFFFFFFFFFFFFFFFull

__host__ __device__ constexpr u64 mix64(u64 x) {  // splitmix64 finaliser
    x ^= x >> 30;
    x *= 0xBF58476D1CE4E5B9ull;
    x ^= x >> 27;
    x *= 0x94D049BB133111EBull;
    x ^= x >> 31;
    return x;
}
__host__ __device__ constexpr u64 pos_mult(int j) { return mix64((u64)j + 1) | 1ull; }

__device__ __forceinline__ int lane_id() { return threadIdx.x & 31; }

// streaming 128-bit load that does not allocate in L1 (read-once data)
__device__ __forceinline__ int4 ld_stream_v4(const void* p) {
    int4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.s32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
                 : "l"(p));
    return r;
}
// 64-bit loads with an L2 eviction policy: the probed table is re-read by every call and should stay
// in L2 (evict last); words of the hash array are read once per call (evict first)
__device__ __forceinline__ u64 ld_u64_keep(const u64* p) {
    u64 pol, v;
    asm("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));  // not volatile: one per thread, hoisted out of loops
    asm volatile("ld.global.nc.L2::cache_hint.u64 %0, [%1], %2;" : "=l"(v) : "l"(p), "l"(pol));
    return v;
}
__device__ __forceinline__ u64 ld_u64_once(const u64* p) {
    u64 pol, v;
    asm("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    asm volatile("ld.global.nc.L2::cache_hint.u64 %0, [%1], %2;" : "=l"(v) : "l"(p), "l"(pol));
    return v;
}
// ---- tagged table probes (peek_demand_rank, peek_lpm, peek_clpm_signals) -------------------------
// Tables of at least TAGS_MIN_S slots get a
// one-byte tag per slot first - 0 for an empty slot, else a fingerprint of its key (k_table_tags: one
// streaming pass over the table).  A probe then walks the TAGS, which do stay in L2, and reads a key only
// where the fingerprint matches: most pending blocks are not cached, and an absent key now costs a
// byte from an L2-resident array instead of a random sector of the table.
static constexpr i64 TAGS_MIN_S = (i64)1 << 16;
// 7-bit tags (1..127): with the top bit of every byte clear, "byte == 0" is a carry-free add per byte
__device__ __forceinline__ u32 key_tag(u64 key) { const u32 t = (u32)(key >> 57); return t ? t : 1u; }
__device__ __forceinline__ u64 ld_tagword(const unsigned char* p) { return ld_u64_keep((const u64*)p); }
static __global__ void __launch_bounds__(256) k_table_tags(const u64* __restrict__ t_keys, i64 S, unsigned char* __restrict__ tags,
                                                    i32* __restrict__ demand) {
    // thread = 8 consecutive slots (64 bytes of keys in, 8 bytes of tags out, the slots' 8 counters
    // cleared when `demand` is given: that call's memset rides along); S is a power of two >= 8 here
    const i64 g = (i64)blockIdx.x * 256 + threadIdx.x;
    if (g * 8 >= S) return;
    const ulonglong2* kp = (const ulonglong2*)(t_keys + g * 8);
    u64 out = 0;
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const ulonglong2 v = __ldg(kp + q);
        const u64 t0 = v.x == PEEK_EMPTY ? 0u : key_tag(v.x), t1 = v.y == PEEK_EMPTY ? 0u : key_tag(v.y);
        out |= (t0 << (16 * q)) | (t1 << (16 * q + 8));
    }
    *(u64*)(tags + g * 8) = out;
    if (demand) {
        int4* d = (int4*)(demand + g * 8);
        d[0] = make_int4(0, 0, 0, 0);
        d[1] = make_int4(0, 0, 0, 0);
    }
}
// slot of `key` or -1.  The probe sequence p, p+1, ... is walked eight tags at a time: `w` is the aligned
// tag word that holds slot p (already loaded); bytes below p & 7 are not on the sequence.  zero_bytes()
// marks (0x80) exactly the zero bytes of a word whose bytes are all <= 0x7f - byte + 0x7f sets the top
// bit iff the byte is not 0 and never carries into its neighbour - so the markers of the empty slots
// (w) and of the slots whose tag equals the key's (w ^ want) are both exact, and the first marker on
// the sequence decides: empty -> absent, tag match -> compare the key.
__device__ __forceinline__ u64 zero_bytes(u64 v) {
    const u32 m7 = 0x7f7f7f7fu, hi = 0x80808080u;
    const u32 lo32 = ~((u32)v + m7) & hi, hi32 = ~((u32)(v >> 32) + m7) & hi;  // no carries: halves are independent
    return ((u64)hi32 << 32) | lo32;
}
__device__ __forceinline__ i64 table_slot_tagged(const u64* __restrict__ t_keys, const unsigned char* __restrict__ tags,
                                                 u64 mask, u64 key, u64 p, u64 w) {
    const u64 want = (u64)key_tag(key) * 0x0101010101010101ull;
    u64 base = p & ~7ull;
    u64 live = ~0ull << (8 * (p & 7));  // bytes on the probe sequence
    for (;;) {
        const u64 zw = zero_bytes(w) & live;
        u64 ev = zw | (zero_bytes(w ^ want) & live);
        while (ev) {
            const u64 first = ev & (~ev + 1);  // lowest marker
            if (zw & first) return -1;         // an empty slot comes first: the key is absent
            const u64 slot = base + (u64)((__ffsll((long long)first) - 1) >> 3);
            if (ld_u64_keep(t_keys + slot) == key) return (i64)slot;
            ev ^= first;                       // another key with the same tag
        }
        base = (base + 8) & mask;
        live = ~0ull;
        w = ld_tagword(tags + base);
    }
}

__device__ __forceinline__ u32 ld_acquire_u32(const u32* p) {
    u32 v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

// Grid-wide barrier for persistent kernels launched with cudaLaunchCooperativeKernel (all CTAs
// co-resident).  `ctr` is a zero-initialised device word that only ever grows; `epoch` is the
// caller's running target (starts at 0, same in every thread).  The gpu-scope fences publish
// this CTA's writes and drop stale L1 lines before the next phase reads other CTAs' data.
__device__ __forceinline__ void grid_barrier(u32* ctr, u32& epoch) {
    if (gridDim.x == 1) {  // small inputs run in one CTA: a CTA barrier is a grid barrier
        __syncthreads();
        return;
    }
    epoch += gridDim.x;
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        atomicAdd(ctr, 1u);
        while (ld_acquire_u32(ctr) < epoch) __nanosleep(32);
        __threadfence();
    }
    __syncthreads();
}

// Phase timeline of the persistent kernels (development builds only: -DPEEK_TRACE; the product
// build has none of this): CTA 0 stamps %globaltimer at PEEK_MARK(id); each translation unit keeps
// its own buffer and exports a reader with PEEK_TRACE_EXPORT(name).
#ifdef PEEK_TRACE
static __device__ unsigned long long g_trace[1024];
static __device__ int g_trace_n;
#define PEEK_MARK(id)                                                                      \
    do {                                                                                   \
        if (blockIdx.x == 0 && threadIdx.x == 0) {                                         \
            unsigned long long t__;                                                        \
            asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t__));                        \
            int n__ = g_trace_n++;                                                         \
            if (n__ < 1024) g_trace[n__] = (t__ << 10) | (unsigned long long)((id) & 1023); \
        }                                                                                  \
    } while (0)
static inline int32_t trace_read_tu(unsigned long long* out, int32_t cap) {
    int n = 0;
    cudaDeviceSynchronize();
    cudaMemcpyFromSymbol(&n, g_trace_n, sizeof(int));
    if (n > 1024) n = 1024;
    if (n > cap) n = cap;
    if (n > 0) cudaMemcpyFromSymbol(out, g_trace, sizeof(unsigned long long) * n);
    int z = 0;
    cudaMemcpyToSymbol(g_trace_n, &z, sizeof(int));
    return n;
}
#define PEEK_TRACE_EXPORT(name) \
    extern "C" int32_t name(unsigned long long* out, int32_t cap) { return peek::trace_read_tu(out, cap); }
#else
#define PEEK_MARK(id) do { } while (0)
#define PEEK_TRACE_EXPORT(name)
#endif

__device__ __forceinline__ int bits_for(u64 maxval) {  // bits needed to hold 0..maxval
    return maxval == 0 ? 1 : 64 - __clzll((long long)maxval);
}

// CTA-wide exclusive scan of one i64 per thread (blockDim.x <= 1024, multiple of 32).
// `smem` holds >= 33 i64.  Returns the exclusive prefix; *total gets the CTA sum.
__device__ __forceinline__ i64 block_exscan_i64(i64 v, i64* smem, i64* total) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
    i64 inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        i64 t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) smem[w] = inc;
    __syncthreads();
    if (w == 0) {
        i64 s = lane < nw ? smem[lane] : 0;
        i64 si = s;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            i64 t = __shfl_up_sync(0xffffffffu, si, o);
            if (lane >= o) si += t;
        }
        if (lane < nw) smem[lane] = si - s;
        if (lane == 31) smem[32] = si;
    }
    __syncthreads();
    i64 r = smem[w] + inc - v;
    *total = smem[32];
    __syncthreads();
    return r;
}

}  // namespace peek
