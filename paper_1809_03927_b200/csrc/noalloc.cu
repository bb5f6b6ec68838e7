// pbs4d_hu_to_density_noalloc: the HU -> density step ("converting Hounsfield Units to
// material density") for callers that must not allocate device memory.
//
// Who that is.  A host process that has handed (nearly) all of the GPU's memory to its own pool -- a treatment-planning
// server with a caching allocator, a PyTorch process -- leaves nothing for a cudaMalloc made behind its back, which then
// fails although the pool has room.  A delivery-time or adaptive-replanning loop with a latency budget cannot afford
// cudaMalloc / cudaFree either: both take driver locks and cudaFree waits for the whole device, stalling every other
// stream of the process.  pbs4d_set_ct_phases allocates (context buffers for the table, the scratch and the densities);
// this entry point does the same conversion with the caller's input and output buffers and nothing else.
//
// How.  The conversion needs scratch: the piecewise-linear table function evaluated once for each of the 65536 possible
// int16 HU values (the per-voxel kernel is then a lookup).  Here that scratch is g_hu_lut below, a file-scope device
// array that is part of the library image: every GPU that loads libpbs4d.so holds its 512 KiB from the first use of the
// library on that GPU until the process exits, whether or not this entry point is ever called.  Its size does not depend
// on the voxel count, so the only scratch-driven limit is the fixed one of 65536 entries; the table points travel as
// kernel arguments (at most PBS4D_NOALLOC_MAX_TABLE_PTS of them).
//
// A host-side detail that matters: in host code the name g_hu_lut is the host's handle of the symbol, not a device
// address -- handing it to a kernel makes the kernel fault, or scribble over host memory on systems where the GPU can
// reach it.  The device address comes from cudaGetSymbolAddress, asked once per device with that device current
// (device_setup below), and it is that address the kernels receive.
//
// The arithmetic is that of grids.cu (table_density, hu_to_density_same_grid), restated here because the array, the
// symbol lookup and the kernels that use it have to share one translation unit; this file is built with -fmad=false like
// grids.cu, so both paths round operation by operation and give the same bits (tests/test_zz_no_alloc.py).
#include "pbs4d.h"

#include <atomic>
#include <cstdarg>
#include <cstdio>

#include <cuda_runtime.h>

namespace {

constexpr int kLutEntries = 65536;                 // one per int16 value: index = HU + 32768
constexpr int kMaxDevices = 64;                    // per-device set-up records (device ordinals beyond are refused)

static_assert(sizeof(double) * kLutEntries == PBS4D_NOALLOC_SCRATCH_BYTES, "header states the scratch size");

// The scratch.  Shared by every call on a device and never cleared: each call rewrites all 65536 entries before its
// lookup kernel reads any (stream order), so nothing in it has to start at zero and nothing of the previous call is
// used.  Two calls that overlap on the GPU (different streams, no dependency) race on it.
static __device__ __align__(256) double g_hu_lut[kLutEntries];

struct TablePoints {
    int   n;
    float hu[PBS4D_NOALLOC_MAX_TABLE_PTS];
    float rho[PBS4D_NOALLOC_MAX_TABLE_PTS];
};

// piecewise-linear, clamped at the ends (reading A4); the same operations in the same order as grids.cu
__device__ __forceinline__ double table_density(double hu, const TablePoints& T)
{
    const int n = T.n;
    if (hu <= (double)T.hu[0]) return (double)T.rho[0];
    if (hu >= (double)T.hu[n - 1]) return (double)T.rho[n - 1];
    int k = 0;
    while (k < n - 2 && hu >= (double)T.hu[k + 1]) ++k;
    const double f = (hu - (double)T.hu[k]) / ((double)T.hu[k + 1] - (double)T.hu[k]);
    return (double)T.rho[k] + f * ((double)T.rho[k + 1] - (double)T.rho[k]);
}

__global__ void __launch_bounds__(256)
noalloc_lut_kernel(const __grid_constant__ TablePoints T, double* __restrict__ lut)
{
    const int v = blockIdx.x * blockDim.x + threadIdx.x;
    if (v < kLutEntries) lut[v] = table_density((double)(v - 32768), T);
}

// HBM-bound: 2 B read + 4 B written per voxel; eight voxels per thread when both pointers are 16-byte aligned
__global__ void __launch_bounds__(256)
noalloc_density_kernel(long long nvox, const int16_t* __restrict__ hu, const double* __restrict__ lut,
                       float* __restrict__ out)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    const long long first = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const bool aligned = ((reinterpret_cast<uintptr_t>(hu) | reinterpret_cast<uintptr_t>(out)) & 15) == 0;
    long long done = 0;
    if (aligned) {
        const long long n8 = nvox >> 3;
        for (long long i = first; i < n8; i += stride) {
            const int4 raw = __ldg(reinterpret_cast<const int4*>(hu) + i);
            const int w[4] = { raw.x, raw.y, raw.z, raw.w };
            float r[8];
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                r[2 * k]     = (float)lut[(int)(short)(w[k] & 0xFFFF) + 32768];
                r[2 * k + 1] = (float)lut[(w[k] >> 16) + 32768];
            }
            float4* o = reinterpret_cast<float4*>(out) + 2 * i;
            o[0] = make_float4(r[0], r[1], r[2], r[3]);
            o[1] = make_float4(r[4], r[5], r[6], r[7]);
        }
        done = n8 << 3;
    }
    for (long long i = done + first; i < nvox; i += stride) out[i] = (float)lut[(int)hu[i] + 32768];
}

// Per-device set-up, done by the first call on each device: the device address of the scratch and the SM count.
// Filled under benign races (every thread computes the same values); `lut` is published last.
struct DeviceSetup {
    std::atomic<double*> lut{nullptr};
    std::atomic<int>     sm_count{0};
};
DeviceSetup g_setup[kMaxDevices];

int report(char* err, int32_t err_cap, int code, const char* fmt, ...)
{
    if (err && err_cap > 0) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(err, (size_t)err_cap, fmt, ap);
        va_end(ap);
    }
    return code;
}

// the current device's set-up record, made on first use; nullptr + *why on failure
DeviceSetup* device_setup(int dev, cudaError_t* why)
{
    DeviceSetup& s = g_setup[dev];
    if (s.lut.load(std::memory_order_acquire)) return &s;
    int sms = 0;
    *why = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (*why != cudaSuccess) return nullptr;
    double* p = nullptr;
    *why = cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_hu_lut);      // device `dev` is current (caller checked)
    if (*why != cudaSuccess) return nullptr;
    if (!p) { *why = cudaErrorInvalidSymbol; return nullptr; }
    s.sm_count.store(sms > 0 ? sms : 148, std::memory_order_relaxed);
    s.lut.store(p, std::memory_order_release);
    return &s;
}

}  // namespace

extern "C" int pbs4d_hu_to_density_noalloc(const int16_t* hu_dev, int64_t n_voxels, int32_t n_pts, const float* hu_pts,
                                           const float* rho_pts, float* rho_dev, void* cuda_stream, char* err,
                                           int32_t err_cap)
{
    if (err && err_cap > 0) err[0] = '\0';
    if (n_pts < 2 || n_pts > PBS4D_NOALLOC_MAX_TABLE_PTS)
        return report(err, err_cap, PBS4D_ERR_ARG,
                      "hu_to_density_noalloc: n_pts = %d, the table takes 2 to %d points (fixed: no memory is allocated)",
                      (int)n_pts, PBS4D_NOALLOC_MAX_TABLE_PTS);
    if (n_voxels < 0 || n_voxels > PBS4D_NOALLOC_MAX_VOXELS)
        return report(err, err_cap, PBS4D_ERR_ARG, "hu_to_density_noalloc: n_voxels = %lld, allowed 0 to %lld",
                      (long long)n_voxels, (long long)PBS4D_NOALLOC_MAX_VOXELS);
    if (!hu_pts || !rho_pts || (n_voxels > 0 && (!hu_dev || !rho_dev)))
        return report(err, err_cap, PBS4D_ERR_ARG, "hu_to_density_noalloc: null pointer");
    TablePoints T;
    T.n = n_pts;
    for (int i = 0; i < PBS4D_NOALLOC_MAX_TABLE_PTS; ++i) { T.hu[i] = 0.0f; T.rho[i] = 0.0f; }
    for (int i = 0; i < n_pts; ++i) {
        if (!(rho_pts[i] > 0.0f) || (i && !(hu_pts[i] > hu_pts[i - 1])))
            return report(err, err_cap, PBS4D_ERR_ARG,
                          "hu_to_density_noalloc: table must ascend in HU with positive densities (point %d)", i);
        T.hu[i] = hu_pts[i];
        T.rho[i] = rho_pts[i];
    }

    int dev = -1;
    cudaError_t ce = cudaGetDevice(&dev);
    if (ce != cudaSuccess)
        return report(err, err_cap, PBS4D_ERR_CUDA, "hu_to_density_noalloc: no CUDA device (%s); there is no CPU fallback",
                      cudaGetErrorString(ce));
    if (dev < 0 || dev >= kMaxDevices)
        return report(err, err_cap, PBS4D_ERR_ARG, "hu_to_density_noalloc: device ordinal %d beyond %d", dev, kMaxDevices - 1);
    DeviceSetup* s = device_setup(dev, &ce);
    if (!s)
        return report(err, err_cap, PBS4D_ERR_CUDA, "hu_to_density_noalloc: set-up on device %d failed: %s", dev,
                      cudaGetErrorString(ce));
    if (n_voxels == 0) return PBS4D_OK;

    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    double* lut = s->lut.load(std::memory_order_relaxed);
    noalloc_lut_kernel<<<kLutEntries / 256, 256, 0, st>>>(T, lut);
    long long blocks = (n_voxels / 8 + 255) / 256 + 1;
    const long long cap = (long long)s->sm_count.load(std::memory_order_relaxed) * 16;
    if (blocks > cap) blocks = cap;
    noalloc_density_kernel<<<(unsigned)blocks, 256, 0, st>>>((long long)n_voxels, hu_dev, lut, rho_dev);
    ce = cudaGetLastError();
    if (ce != cudaSuccess)
        return report(err, err_cap, PBS4D_ERR_CUDA, "hu_to_density_noalloc: launch failed: %s", cudaGetErrorString(ce));
    return PBS4D_OK;
}
