// In-run roofline probes (BASELINE.json north_star: throughput is reported "as achieved fraction of the FP32-issue,
// L2-atomic and HBM roofline measured by in-run microbenchmarks").  Three tiny kernels, timed with CUDA events on
// the context's stream:
//   FP32 issue : 8 independent FFMA chains per thread, enough warps to fill every SM -> lane-instructions / s
//   L2 atomic  : red.global.add.u64 to pseudo-random addresses of a 32 MB window (L2-resident, like the int64 dose
//                grid of a phase), and to one hot address per warp                     -> lane-atomics / s
//   HBM        : float4 copy of a buffer much larger than the L2                       -> bytes (read + written) / s
#include "internal.h"

#include <cuda_runtime.h>

namespace pbs4d {

namespace {

constexpr int kFmaIters = 4096, kFmaChains = 8;

__global__ void __launch_bounds__(256) probe_fma_kernel(float* out, float a, float b)
{
    float x[kFmaChains];
#pragma unroll
    for (int c = 0; c < kFmaChains; ++c) x[c] = (float)(threadIdx.x + c);
    for (int it = 0; it < kFmaIters; ++it) {
#pragma unroll
        for (int c = 0; c < kFmaChains; ++c) x[c] = fmaf(x[c], a, b);
    }
    float s = 0.0f;
#pragma unroll
    for (int c = 0; c < kFmaChains; ++c) s += x[c];
    if (s == 123.456f) out[0] = s;                       // never true; keeps the chains alive
}

constexpr int kRedPerThread = 256;

__global__ void __launch_bounds__(256) probe_red_kernel(unsigned long long* win, unsigned mask, int hot)
{
    unsigned h = (blockIdx.x * blockDim.x + threadIdx.x) * 2654435761u + 12345u;
    const unsigned warp_slot = ((blockIdx.x * blockDim.x + threadIdx.x) >> 5) * 16u;
    for (int it = 0; it < kRedPerThread; ++it) {
        h = h * 1664525u + 1013904223u;
        const unsigned idx = hot ? (warp_slot & mask) : ((h >> 4) & mask);
        atomicAdd(win + idx, 1ull);
    }
}

__global__ void __launch_bounds__(256) probe_copy_kernel(const float4* __restrict__ src, float4* __restrict__ dst, size_t n)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) dst[i] = src[i];
}

template <class F> cudaError_t timed(cudaStream_t st, int reps, float& best_ms, F&& launch)
{
    cudaEvent_t e0, e1;
    cudaError_t e = cudaEventCreate(&e0); if (e != cudaSuccess) return e;
    e = cudaEventCreate(&e1); if (e != cudaSuccess) { cudaEventDestroy(e0); return e; }
    best_ms = 1.0e30f;
    for (int r = 0; r < reps + 1; ++r) {                 // first repetition is the warm-up
        cudaEventRecord(e0, st);
        launch();
        cudaEventRecord(e1, st);
        e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) break;
        float ms = 0.0f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (r > 0 && ms < best_ms) best_ms = ms;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    return e != cudaSuccess ? e : cudaGetLastError();
}

}  // namespace

cudaError_t probe_fp32_issue(int sm_count, cudaStream_t st, double* lane_inst_per_s)
{
    float* out = nullptr;
    cudaError_t e = cudaMalloc(&out, sizeof(float)); if (e != cudaSuccess) return e;
    const int blocks = sm_count * 8;
    float ms = 0.0f;
    e = timed(st, 3, ms, [&] { probe_fma_kernel<<<blocks, 256, 0, st>>>(out, 0.999f, 0.001f); });
    cudaFree(out);
    *lane_inst_per_s = (double)blocks * 256.0 * kFmaIters * kFmaChains / (ms * 1.0e-3);
    return e;
}

cudaError_t probe_l2_atomic(int sm_count, int hot, cudaStream_t st, double* lane_atomics_per_s)
{
    const size_t words = (size_t)4 << 20;                // 4 Mi x 8 B = 32 MB window
    unsigned long long* win = nullptr;
    cudaError_t e = cudaMalloc(&win, words * 8); if (e != cudaSuccess) return e;
    cudaMemsetAsync(win, 0, words * 8, st);
    const int blocks = sm_count * 16;
    float ms = 0.0f;
    e = timed(st, 3, ms, [&] { probe_red_kernel<<<blocks, 256, 0, st>>>(win, (unsigned)(words - 1), hot); });
    cudaFree(win);
    *lane_atomics_per_s = (double)blocks * 256.0 * kRedPerThread / (ms * 1.0e-3);
    return e;
}

cudaError_t probe_hbm_copy(int sm_count, cudaStream_t st, double* bytes_per_s)
{
    const size_t n = (size_t)64 << 20;                   // 64 Mi float4 = 1 GiB per buffer
    float4 *a = nullptr, *b = nullptr;
    cudaError_t e = cudaMalloc(&a, n * sizeof(float4)); if (e != cudaSuccess) return e;
    e = cudaMalloc(&b, n * sizeof(float4)); if (e != cudaSuccess) { cudaFree(a); return e; }
    cudaMemsetAsync(a, 0, n * sizeof(float4), st);
    float ms = 0.0f;
    e = timed(st, 5, ms, [&] { probe_copy_kernel<<<sm_count * 16, 256, 0, st>>>(a, b, n); });
    cudaFree(a); cudaFree(b);
    *bytes_per_s = 2.0 * (double)n * sizeof(float4) / (ms * 1.0e-3);
    return e;
}

}  // namespace pbs4d
