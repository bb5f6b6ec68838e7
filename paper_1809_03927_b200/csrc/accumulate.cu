// Energy-/mass-transfer subvoxel dose accumulation (Sec. 2.D.2).
//
//   push   (Eq. 4-6): each source voxel j is split into nsx*nsy*nsz subvoxels; M = rho_j v_k, E = M D_j (Eq. 4); the
//                     subvoxel centre is mapped by the trilinearly interpolated DVF T^{S->R} (Eq. 1)
//                     and E, M are summed into the reference voxel containing the image (Eq. 6).
//   finalize (Eq. 5, 2): D_i^S = sum E / sum M per source phase, D_i = D_i^R + sum_S D_i^S, masked to the volume
//                     covered by all DVFs.
//
// The paper ran one thread per source voxel with an n^3 device loop and two float atomics per subvoxel
// (PAPER.md:122-124).  Here the sums are int64 fixed point (order-independent, so the result is unique and
// bit-reproducible), the subvoxel volume -- a common factor of Eq. 4 -- is dropped, and consecutive subvoxels of a
// voxel that land in the same reference voxel are merged into one pair of red.global.add.u64.
// Coordinate arithmetic is strict fp32: every operation is an explicit round-to-nearest intrinsic (never fused),
// in the order fixed by DESIGN.md "Accumulation arithmetic"; this TU is also built with -fmad=false.
#include "internal.h"

#include <cuda_runtime.h>

namespace pbs4d {

namespace {

struct AxisMap { float p; int i0, i1; float w; bool ok; };

// subvoxel centre on one axis and its DVF-grid cell/weight
__device__ __forceinline__ AxisMap axis_map(float o, float h, int i, int a, int ns, float od, float hd, int nd)
{
    AxisMap m;
    const float f = __fdiv_rn(__fadd_rn((float)a, 0.5f), (float)ns);
    m.p = __fadd_rn(o, __fmul_rn(__fadd_rn((float)i, f), h));
    float g = __fsub_rn(__fdiv_rn(__fsub_rn(m.p, od), hd), 0.5f);
    m.ok = (g >= -0.5f) && (g < __fsub_rn((float)nd, 0.5f));
    g = fminf(fmaxf(g, 0.0f), (float)(nd - 1));
    int k = (int)floorf(g);
    k = max(min(k, nd - 2), 0);
    m.i0 = k;
    m.i1 = min(k + 1, nd - 1);
    m.w  = __fsub_rn(g, (float)k);
    return m;
}

__device__ __forceinline__ float lerp_rn(float A, float B, float w)
{
    return __fadd_rn(A, __fmul_rn(w, __fsub_rn(B, A)));
}

__device__ __forceinline__ bool dest_index(float q, float o, float h, int n, int& ix)
{
    const float fl = floorf(__fdiv_rn(__fsub_rn(q, o), h));
    if (!(fl >= 0.0f) || !(fl < (float)n)) return false;
    ix = (int)fl;
    return true;
}

struct PushParams {
    pbs4d_grid src, dvf, ref;
    const float* __restrict__ dose;
    const float* __restrict__ rho;
    const float* __restrict__ ux;
    const float* __restrict__ uy;
    const float* __restrict__ uz;
    int nsx, nsy, nsz;
    unsigned long long* E;
    unsigned long long* M;
    AccCounters* counters;
};

__global__ void __launch_bounds__(256)
emtm_push_kernel(const PushParams P)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = blockIdx.z;
    unsigned long long n_ref = 0, n_dvf = 0;
    if (i < P.src.nx && j < P.src.ny) {
        const size_t v = ((size_t)k * P.src.ny + j) * P.src.nx + i;
        const float rho = P.rho[v], dose = P.dose[v];
        const long long m_q = __double2ll_rn(__dmul_rn((double)rho, 16777216.0));
        const long long e_q = __double2ll_rn(__dmul_rn(__dmul_rn((double)rho, (double)dose), 4294967296.0));
        long long run_dst = -1; long long run_cnt = 0;
        const int dnx = P.dvf.nx, dny = P.dvf.ny;
        for (int c = 0; c < P.nsz; ++c) {
            const AxisMap mz = axis_map(P.src.oz, P.src.hz, k, c, P.nsz, P.dvf.oz, P.dvf.hz, P.dvf.nz);
            for (int b = 0; b < P.nsy; ++b) {
                const AxisMap my = axis_map(P.src.oy, P.src.hy, j, b, P.nsy, P.dvf.oy, P.dvf.hy, P.dvf.ny);
                const size_t r00 = ((size_t)mz.i0 * dny + my.i0) * dnx, r01 = ((size_t)mz.i0 * dny + my.i1) * dnx;
                const size_t r10 = ((size_t)mz.i1 * dny + my.i0) * dnx, r11 = ((size_t)mz.i1 * dny + my.i1) * dnx;
                for (int a = 0; a < P.nsx; ++a) {
                    const AxisMap mx = axis_map(P.src.ox, P.src.hx, i, a, P.nsx, P.dvf.ox, P.dvf.hx, P.dvf.nx);
                    if (!(mx.ok && my.ok && mz.ok)) { n_dvf += 1; continue; }
                    float q[3];
                    const float* comp[3] = { P.ux, P.uy, P.uz };
                    const float  pc[3]   = { mx.p, my.p, mz.p };
#pragma unroll
                    for (int d = 0; d < 3; ++d) {
                        const float* u = comp[d];
                        const float c00 = lerp_rn(__ldg(u + r00 + mx.i0), __ldg(u + r00 + mx.i1), mx.w);
                        const float c01 = lerp_rn(__ldg(u + r01 + mx.i0), __ldg(u + r01 + mx.i1), mx.w);
                        const float c10 = lerp_rn(__ldg(u + r10 + mx.i0), __ldg(u + r10 + mx.i1), mx.w);
                        const float c11 = lerp_rn(__ldg(u + r11 + mx.i0), __ldg(u + r11 + mx.i1), mx.w);
                        const float c0  = lerp_rn(c00, c01, my.w);
                        const float c1  = lerp_rn(c10, c11, my.w);
                        q[d] = __fadd_rn(pc[d], lerp_rn(c0, c1, mz.w));
                    }
                    int ix, iy, iz;
                    if (!dest_index(q[0], P.ref.ox, P.ref.hx, P.ref.nx, ix) ||
                        !dest_index(q[1], P.ref.oy, P.ref.hy, P.ref.ny, iy) ||
                        !dest_index(q[2], P.ref.oz, P.ref.hz, P.ref.nz, iz)) { n_ref += 1; continue; }
                    const long long dst = ((long long)iz * P.ref.ny + iy) * P.ref.nx + ix;
                    if (dst == run_dst) { run_cnt += 1; continue; }
                    if (run_cnt) {
                        atomicAdd(P.E + run_dst, (unsigned long long)(run_cnt * e_q));
                        atomicAdd(P.M + run_dst, (unsigned long long)(run_cnt * m_q));
                    }
                    run_dst = dst; run_cnt = 1;
                }
            }
        }
        if (run_cnt) {
            atomicAdd(P.E + run_dst, (unsigned long long)(run_cnt * e_q));
            atomicAdd(P.M + run_dst, (unsigned long long)(run_cnt * m_q));
        }
    }
    // drop counters: warp-reduce, one atomic per warp
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        n_ref += __shfl_xor_sync(0xffffffffu, n_ref, off);
        n_dvf += __shfl_xor_sync(0xffffffffu, n_dvf, off);
    }
    if (((threadIdx.y * blockDim.x + threadIdx.x) & 31) == 0) {
        if (n_ref) atomicAdd(&P.counters->dropped_ref, n_ref);
        if (n_dvf) atomicAdd(&P.counters->dropped_dvf, n_dvf);
    }
}

constexpr int kMaxSrc = 32;
struct FinalizeParams {
    pbs4d_grid ref;
    const float* __restrict__ dose_ref;
    int n_src;
    const long long* E[kMaxSrc];
    const long long* M[kMaxSrc];
    pbs4d_grid dvf[kMaxSrc];
    float* out;
};

__device__ __forceinline__ bool covered_axis(float o, float h, int i, float od, float hd, int nd)
{
    const float p = __fadd_rn(o, __fmul_rn(__fadd_rn((float)i, 0.5f), h));
    const float g = __fsub_rn(__fdiv_rn(__fsub_rn(p, od), hd), 0.5f);
    return (g >= -0.5f) && (g < __fsub_rn((float)nd, 0.5f));
}

__global__ void __launch_bounds__(256)
emtm_finalize_kernel(const __grid_constant__ FinalizeParams P)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = blockIdx.z;
    if (i >= P.ref.nx || j >= P.ref.ny) return;
    const size_t v = ((size_t)k * P.ref.ny + j) * P.ref.nx + i;
    bool covered = true;
    for (int s = 0; s < P.n_src && covered; ++s)
        covered = covered_axis(P.ref.ox, P.ref.hx, i, P.dvf[s].ox, P.dvf[s].hx, P.dvf[s].nx) &&
                  covered_axis(P.ref.oy, P.ref.hy, j, P.dvf[s].oy, P.dvf[s].hy, P.dvf[s].ny) &&
                  covered_axis(P.ref.oz, P.ref.hz, k, P.dvf[s].oz, P.dvf[s].hz, P.dvf[s].nz);
    if (!covered) { P.out[v] = 0.0f; return; }
    double D = (double)P.dose_ref[v];
    for (int s = 0; s < P.n_src; ++s) {
        const long long m = P.M[s][v];
        if (m != 0) D = __dadd_rn(D, __dmul_rn(__ddiv_rn((double)P.E[s][v], (double)m), 1.0 / 256.0));
    }
    P.out[v] = (float)D;
}

}  // namespace

void launch_emtm_push(const pbs4d_grid& src, const float* dose, const float* rho, const pbs4d_grid& dvf_grid,
                      const float* disp, const pbs4d_grid& ref, int nsx, int nsy, int nsz,
                      long long* E, long long* M, AccCounters* counters, cudaStream_t st)
{
    PushParams P;
    P.src = src; P.dvf = dvf_grid; P.ref = ref; P.dose = dose; P.rho = rho;
    const size_t plane = (size_t)dvf_grid.nx * dvf_grid.ny * dvf_grid.nz;
    P.ux = disp; P.uy = disp + plane; P.uz = disp + 2 * plane;
    P.nsx = nsx; P.nsy = nsy; P.nsz = nsz;
    P.E = (unsigned long long*)E; P.M = (unsigned long long*)M; P.counters = counters;
    dim3 b(32, 8, 1), g((src.nx + 31) / 32, (src.ny + 7) / 8, src.nz);
    emtm_push_kernel<<<g, b, 0, st>>>(P);
}

void launch_emtm_finalize(const pbs4d_grid& ref, const float* dose_ref, int n_src, const long long* const* E_host,
                          const long long* const* M_host, const pbs4d_grid* dvf_grids_host, float* out,
                          cudaStream_t st)
{
    FinalizeParams P;
    P.ref = ref; P.dose_ref = dose_ref; P.n_src = n_src; P.out = out;
    for (int s = 0; s < n_src && s < kMaxSrc; ++s) { P.E[s] = E_host[s]; P.M[s] = M_host[s]; P.dvf[s] = dvf_grids_host[s]; }
    dim3 b(32, 8, 1), g((ref.nx + 31) / 32, (ref.ny + 7) / 8, ref.nz);
    emtm_finalize_kernel<<<g, b, 0, st>>>(P);
}

}  // namespace pbs4d
