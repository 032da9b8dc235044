// gather_probe.cu - measurement utility of the harness (NOT part of libpeek.so): the random
// 32-byte-sector gather ceiling of SURVEY.md section 8(d), the honest roofline of the probe /
// child-lookup / bisection kernels.  `reads` independent 16-byte loads at addresses drawn by a
// counter-based generator (splitmix64 finaliser of seed + read index), uniform over the 32-byte
// sectors of buf[0 .. bytes) [device, 32-byte aligned]; the xor of everything read goes to sink[0]
// [device] so the loads cannot be elided.  Enqueues one kernel on `stream`; time it with events.
#include <cuda_runtime.h>
#include <stdint.h>

typedef uint64_t u64;
typedef int64_t i64;

static __device__ __forceinline__ u64 mixer(u64 x) {
    x ^= x >> 30; x *= 0xBF58476D1CE4E5B9ull; x ^= x >> 27; x *= 0x94D049BB133111EBull; x ^= x >> 31;
    return x;
}
static constexpr int RG_THREADS = 256, RG_PER_THREAD = 8;
__global__ void __launch_bounds__(RG_THREADS) k_random_gather(const uint4* __restrict__ buf, u64 sectors,
                                                             i64 reads, u64 seed, u64* __restrict__ sink) {
    const i64 t = (i64)blockIdx.x * RG_THREADS + threadIdx.x, nthreads = (i64)gridDim.x * RG_THREADS;
    u64 acc = 0;
    for (i64 i0 = t; i0 < reads; i0 += nthreads * RG_PER_THREAD) {
        uint4 v[RG_PER_THREAD];
#pragma unroll
        for (int u = 0; u < RG_PER_THREAD; ++u) {  // RG_PER_THREAD independent loads in flight
            const i64 i = i0 + u * nthreads;
            const u64 sct = mixer(seed + (u64)i * 0x9E3779B97F4A7C15ull) % sectors;
            v[u] = i < reads ? __ldg(buf + 2 * sct) : make_uint4(0, 0, 0, 0);
        }
#pragma unroll
        for (int u = 0; u < RG_PER_THREAD; ++u) acc ^= ((u64)v[u].x << 32 | v[u].y) ^ ((u64)v[u].z << 32 | v[u].w);
    }
    acc ^= __shfl_xor_sync(0xffffffffu, acc, 16);
    acc ^= __shfl_xor_sync(0xffffffffu, acc, 8);
    acc ^= __shfl_xor_sync(0xffffffffu, acc, 4);
    acc ^= __shfl_xor_sync(0xffffffffu, acc, 2);
    acc ^= __shfl_xor_sync(0xffffffffu, acc, 1);
    if ((threadIdx.x & 31) == 0 && acc) atomicXor((unsigned long long*)sink, (unsigned long long)acc);
}

// 0 = ok, -1 = bad argument, -4 = CUDA error
extern "C" int harness_random_gather(const void* buf, int64_t bytes, int64_t reads, uint64_t seed, uint64_t* sink,
                                     void* stream) {
    if (!buf || !sink || bytes < 32 || reads < 0 || ((uintptr_t)buf & 31)) return -1;
    if (reads == 0) return 0;
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    i64 want = (reads + RG_THREADS * RG_PER_THREAD - 1) / (RG_THREADS * RG_PER_THREAD);
    i64 cap = (i64)sms * 64;
    unsigned grid = (unsigned)(want < cap ? want : cap);
    k_random_gather<<<grid, RG_THREADS, 0, (cudaStream_t)stream>>>((const uint4*)buf, (u64)(bytes / 32), reads, seed, sink);
    return cudaGetLastError() == cudaSuccess ? 0 : -4;
}
