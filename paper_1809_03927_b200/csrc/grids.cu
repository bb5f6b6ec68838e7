// Per-voxel grid kernels: HU -> density ("converting Hounsfield Units to material
// density") with optional overlap-volume resampling onto the dose grid, and int64 energy -> fp32 dose in Gy.
// Memory-bound, one thread per output voxel, coalesced along x.  This translation unit is compiled with
// -fmad=false: the double-precision expressions below are evaluated operation by operation, so that the density
// handed to the accumulation stage is reproducible to the last bit.
#include "internal.h"

#include <cuda_runtime.h>

namespace pbs4d {

namespace {

__device__ __forceinline__ double table_density(double hu, int n, const float* __restrict__ hp,
                                                const float* __restrict__ rp)
{
    if (hu <= (double)hp[0]) return (double)rp[0];
    if (hu >= (double)hp[n - 1]) return (double)rp[n - 1];
    int k = 0;
    while (k < n - 2 && hu >= (double)hp[k + 1]) ++k;
    const double f = (hu - (double)hp[k]) / ((double)hp[k + 1] - (double)hp[k]);
    return (double)rp[k] + f * ((double)rp[k + 1] - (double)rp[k]);
}

// HU is a 16-bit integer: the table function is evaluated once per possible value (65536 doubles, 512 KB, resident in
// the L2) and the per-voxel kernels look it up -- the same double as evaluating it per voxel, without 42 million
// double-precision divisions per phase of config 5.
__global__ void density_lut_kernel(int n_pts, const float* __restrict__ hp, const float* __restrict__ rp,
                                   double* __restrict__ lut)
{
    const int v = blockIdx.x * blockDim.x + threadIdx.x;                     // 0 .. 65535  <->  HU -32768 .. 32767
    if (v < 65536) lut[v] = table_density((double)(v - 32768), n_pts, hp, rp);
}

// HBM-bound: 2 B read + 4 B written per voxel; eight voxels per thread (one 128-bit load, two 128-bit stores)
__global__ void __launch_bounds__(256)
hu_to_density_same_grid(long long nvox, const int16_t* __restrict__ hu, const double* __restrict__ lut,
                        float* __restrict__ out)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    const long long n8 = nvox >> 3;
    const bool aligned = ((reinterpret_cast<uintptr_t>(hu) | reinterpret_cast<uintptr_t>(out)) & 15) == 0;
    long long done = 0;
    if (aligned) {
        for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n8; i += stride) {
            const int4 raw = __ldg(reinterpret_cast<const int4*>(hu) + i);
            const int w[4] = { raw.x, raw.y, raw.z, raw.w };
            float r[8];
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                r[2 * k]     = (float)__ldg(lut + ((int)(short)(w[k] & 0xFFFF) + 32768));
                r[2 * k + 1] = (float)__ldg(lut + ((w[k] >> 16) + 32768));
            }
            float4* o = reinterpret_cast<float4*>(out) + 2 * i;
            o[0] = make_float4(r[0], r[1], r[2], r[3]);
            o[1] = make_float4(r[4], r[5], r[6], r[7]);
        }
        done = n8 << 3;
    }
    for (long long i = done + (long long)blockIdx.x * blockDim.x + threadIdx.x; i < nvox; i += stride)
        out[i] = (float)__ldg(lut + ((int)hu[i] + 32768));
}

// dose-grid voxel = overlap-volume-weighted mean of the densities of the CT voxels it intersects
__global__ void hu_to_density_resample(pbs4d_grid ct, pbs4d_grid dg, const int16_t* __restrict__ hu,
                                       const double* __restrict__ lut, double rho_first, float* __restrict__ out)
{
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z;
    if (x >= dg.nx || y >= dg.ny || z >= dg.nz) return;
    const double ch[3] = { (double)ct.hx, (double)ct.hy, (double)ct.hz };
    const double co[3] = { (double)ct.ox, (double)ct.oy, (double)ct.oz };
    const int    cn[3] = { ct.nx, ct.ny, ct.nz };
    const double dh[3] = { (double)dg.hx, (double)dg.hy, (double)dg.hz };
    const double d0[3] = { (double)dg.ox, (double)dg.oy, (double)dg.oz };
    const int    id[3] = { x, y, z };
    int lo[3], hi[3]; double a[3], b[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        a[k] = d0[k] + (double)id[k] * dh[k];
        b[k] = a[k] + dh[k];
        lo[k] = max((int)floor((a[k] - co[k]) / ch[k]), 0);
        hi[k] = min((int)ceil((b[k] - co[k]) / ch[k]), cn[k]);
    }
    double acc = 0.0, wsum = 0.0;
    for (int kz = lo[2]; kz < hi[2]; ++kz)
        for (int ky = lo[1]; ky < hi[1]; ++ky)
            for (int kx = lo[0]; kx < hi[0]; ++kx) {
                const int ic[3] = { kx, ky, kz };
                double wv = 1.0;
#pragma unroll
                for (int k = 0; k < 3; ++k) {
                    const double ca = co[k] + (double)ic[k] * ch[k], cb = ca + ch[k];
                    const double ov = fmin(b[k], cb) - fmax(a[k], ca);
                    wv *= ov > 0.0 ? ov : 0.0;
                }
                if (wv > 0.0) {
                    acc  += wv * __ldg(lut + ((int)hu[((size_t)kz * cn[1] + ky) * cn[0] + kx] + 32768));
                    wsum += wv;
                }
            }
    out[((size_t)z * dg.ny + y) * dg.nx + x] = (float)(wsum > 0.0 ? acc / wsum : rho_first);
}

// a7 / T12: D = Q 2^-k 1.602176634e-10 / (rho V_cm3)  [Gy]; optionally per proton.  A voxel without mass (never the
// case for densities accepted by set_ct_phases / set_density_phases) gets dose 0 instead of 0/0.
__device__ __forceinline__ float dose_of(long long q, float rho, double inv_scale, double vol_cm3, double per_protons)
{
    if (q == 0) return 0.0f;                 // 0 2^-k c / m = +0 for every finite m > 0 (and 0 for m <= 0): no arithmetic
    const double mass = (double)rho * vol_cm3;
    double D = (double)q * inv_scale * 1.602176634e-10 / mass;
    if (per_protons > 0.0) D /= per_protons;
    return mass > 0.0 ? (float)D : 0.0f;
}

// HBM-bound: 12 B read + 4 B written per voxel, two voxels per thread (128-bit load of the energies); a beam touches a
// small part of the grid, so most voxels take the q == 0 exit and the double-precision divisions do not show
__global__ void __launch_bounds__(256)
finalize_dose_kernel(long long nvox, const float* __restrict__ rho, const long long* __restrict__ Q,
                     double inv_scale, double vol_cm3, double per_protons, float* __restrict__ dose)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    const long long n2 = nvox >> 1;
    const bool aligned = ((reinterpret_cast<uintptr_t>(Q) & 15) | (reinterpret_cast<uintptr_t>(rho) & 7) |
                          (reinterpret_cast<uintptr_t>(dose) & 7)) == 0;
    long long done = 0;
    if (aligned) {
        for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n2; i += stride) {
            const longlong2 q = *(reinterpret_cast<const longlong2*>(Q) + i);
            float2 d = make_float2(0.0f, 0.0f);
            if (q.x | q.y) {
                const float2 r = *(reinterpret_cast<const float2*>(rho) + i);
                d.x = dose_of(q.x, r.x, inv_scale, vol_cm3, per_protons);
                d.y = dose_of(q.y, r.y, inv_scale, vol_cm3, per_protons);
            }
            *(reinterpret_cast<float2*>(dose) + i) = d;
        }
        done = n2 << 1;
    }
    for (long long i = done + (long long)blockIdx.x * blockDim.x + threadIdx.x; i < nvox; i += stride)
        dose[i] = dose_of(Q[i], rho[i], inv_scale, vol_cm3, per_protons);
}

// densities handed in directly (set_density_phases) must be finite and inside [kRhoMin, kRhoMax]: rho = 0 would give
// 0/0 in the dose, rho = Inf a zero step limit (a history that never advances)
__global__ void validate_density_kernel(size_t n, const float* __restrict__ rho, int* __restrict__ bad)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    bool any = false;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const float r = rho[i];
        any |= !(r >= 1.0e-6f && r <= 100.0f);               // also true for NaN
    }
    if (__any_sync(0xffffffffu, any) && (threadIdx.x & 31) == 0) atomicOr(bad, 1);
}


// DVF construction (Sec. 2.D.1: "construct the DVFs ... one-thread-per-deformation-grid-voxel ... to
// calculate r_f for all voxels"; App. B): Eq. 8 r_0 = start + i dX U + j dY V + k dZ W, W = U x V;
// Eq. 7 r_f = M_Post (M_Pre [r_0; 1] + [Delta; 0]).  Double precision, one rounding per operation (this TU is built
// with -fmad=false), outputs r_f and r_f - r_0 in fp32.  HBM-bound: 12 B read, 12-24 B written per grid voxel.
struct DvfBuildParams {
    int nx, ny, nz;
    double start[3], delta[3], U[3], V[3], W[3], pre[16], post[16];
    const float* __restrict__ dx; const float* __restrict__ dy; const float* __restrict__ dz;
    float* rf; float* disp; size_t n;
};

__device__ __forceinline__ void mat4_apply(const double* M, const double v[4], double out[4])
{
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        double s = M[4 * r + 0] * v[0];
        s = s + M[4 * r + 1] * v[1];
        s = s + M[4 * r + 2] * v[2];
        s = s + M[4 * r + 3] * v[3];
        out[r] = s;
    }
}

__global__ void __launch_bounds__(256) dvf_build_kernel(const __grid_constant__ DvfBuildParams P)
{
    const int i = blockIdx.y * blockDim.x + threadIdx.x;
    const int j = blockIdx.x % P.ny, k = blockIdx.x / P.ny;          // rows on grid.x (up to 2^31 - 1)
    if (i >= P.nx) return;
    const size_t v = ((size_t)k * P.ny + j) * P.nx + i;
    double r0[4], a[4], b[4];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        double s = P.U[c] * P.delta[0] * (double)i;
        s = s + P.V[c] * P.delta[1] * (double)j;
        s = s + P.W[c] * P.delta[2] * (double)k;
        r0[c] = s + P.start[c];
    }
    r0[3] = 1.0;
    mat4_apply(P.pre, r0, a);
    a[0] = a[0] + (double)P.dx[v]; a[1] = a[1] + (double)P.dy[v]; a[2] = a[2] + (double)P.dz[v];
    mat4_apply(P.post, a, b);
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        if (P.rf)   P.rf[(size_t)c * P.n + v]   = (float)b[c];
        if (P.disp) P.disp[(size_t)c * P.n + v] = (float)(b[c] - r0[c]);
    }
}

}  // namespace

void launch_dvf_build(const pbs4d_dicom_dvf& g, const float* delta_dev, float* rf_dev, float* disp_dev, cudaStream_t st)
{
    DvfBuildParams P;
    P.nx = g.nx; P.ny = g.ny; P.nz = g.nz; P.n = (size_t)g.nx * g.ny * g.nz;
    for (int c = 0; c < 3; ++c) { P.start[c] = g.start[c]; P.delta[c] = g.delta[c]; P.U[c] = g.row_cos[c]; P.V[c] = g.col_cos[c]; }
    P.W[0] = g.row_cos[1] * g.col_cos[2] - g.row_cos[2] * g.col_cos[1];
    P.W[1] = g.row_cos[2] * g.col_cos[0] - g.row_cos[0] * g.col_cos[2];
    P.W[2] = g.row_cos[0] * g.col_cos[1] - g.row_cos[1] * g.col_cos[0];
    for (int e = 0; e < 16; ++e) { P.pre[e] = g.pre[e]; P.post[e] = g.post[e]; }
    P.dx = delta_dev; P.dy = delta_dev + P.n; P.dz = delta_dev + 2 * P.n;
    P.rf = rf_dev; P.disp = disp_dev;
    dim3 grid((unsigned)(g.ny * g.nz), (g.nx + 255) / 256);
    dvf_build_kernel<<<grid, 256, 0, st>>>(P);
}

int sm_count_of_current_device(void)
{
    int dev = 0, n = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n < 1) n = 148;
    return n;
}

int launch_validate_density(const float* rho, size_t n, int* flag_dev, cudaStream_t st)
{
    const int blocks = (int)min((long long)((n + 255) / 256), (long long)sm_count_of_current_device() * 16);
    validate_density_kernel<<<blocks, 256, 0, st>>>(n, rho, flag_dev);
    return 0;
}

void launch_hu_to_density(const pbs4d_grid& ct, const int16_t* hu, const pbs4d_grid* dose_grid, int32_t n_pts,
                          const float* hp, const float* rp, float rho_first, double* lut, float* rho_out, cudaStream_t st)
{
    density_lut_kernel<<<256, 256, 0, st>>>(n_pts, hp, rp, lut);             // 3 us; rebuilt per call: no state to keep
    if (!dose_grid) {
        const long long nvox = (long long)ct.nx * ct.ny * ct.nz;
        const int blocks = (int)min((nvox / 8 + 255) / 256 + 1, (long long)sm_count_of_current_device() * 16);
        hu_to_density_same_grid<<<blocks, 256, 0, st>>>(nvox, hu, lut, rho_out);
    } else {
        dim3 b(32, 8, 1), g((dose_grid->nx + 31) / 32, (dose_grid->ny + 7) / 8, dose_grid->nz);
        hu_to_density_resample<<<g, b, 0, st>>>(ct, *dose_grid, hu, lut, (double)rho_first, rho_out);
    }
}

void launch_finalize_dose(const pbs4d_grid& g, const float* rho, const long long* Q, int32_t fixed_shift,
                          double per_protons, float* dose, cudaStream_t st)
{
    const long long nvox = (long long)g.nx * g.ny * g.nz;
    const double vol_cm3 = (double)g.hx * (double)g.hy * (double)g.hz * 1.0e-3;
    const int blocks = (int)min((nvox + 255) / 256, (long long)sm_count_of_current_device() * 16);
    finalize_dose_kernel<<<blocks, 256, 0, st>>>(nvox, rho, Q, ldexp(1.0, -fixed_shift), vol_cm3, per_protons, dose);
}

}  // namespace pbs4d
