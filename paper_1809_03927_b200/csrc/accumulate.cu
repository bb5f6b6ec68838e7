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

#include <algorithm>

namespace pbs4d {

namespace {

// One axis of the subvoxel -> DVF-cell map (A2, A3): subvoxel centre p, lower DVF node i0, upper node i0 + d1,
// weight w, and whether the centre lies inside the DVF grid's voxel extent.  It depends on (voxel index, subvoxel
// index) of that axis only, so a CTA computes it once per axis for its tile and keeps it in shared memory.
struct __align__(16) AxisEntry { float p, w; int i0; int flags; };      // flags: bit0 = d1, bit1 = ok

__device__ __forceinline__ AxisEntry axis_map(float o, float h, int i, int a, int ns, float od, float hd, int nd)
{
    AxisEntry m;
    const float f = __fdiv_rn(__fadd_rn((float)a, 0.5f), (float)ns);
    m.p = __fadd_rn(o, __fmul_rn(__fadd_rn((float)i, f), h));
    float g = __fsub_rn(__fdiv_rn(__fsub_rn(m.p, od), hd), 0.5f);
    const bool ok = (g >= -0.5f) && (g < __fsub_rn((float)nd, 0.5f));
    g = fminf(fmaxf(g, 0.0f), (float)(nd - 1));
    int k = (int)floorf(g);
    k = max(min(k, nd - 2), 0);
    m.i0 = k;
    m.w  = __fsub_rn(g, (float)k);
    m.flags = (min(k + 1, nd - 1) - k) | (ok ? 2 : 0);
    return m;
}

__device__ __forceinline__ float lerp_rn(float A, float B, float w)
{
    return __fadd_rn(A, __fmul_rn(w, __fsub_rn(B, A)));
}

// A4: ix = floorf((q - o) / h) with the IEEE quotient, inside iff 0 <= ix < n.  The division is replaced by a
// multiplication with inv_h = RN(1/h): y = RN(d inv_h) differs from the IEEE quotient RN(d / h) by at most
// (2^-23 + 2^-24) |y|, so both have the same floor unless y lies within that distance of an integer; in that (rare)
// case the quotient itself is evaluated.  The result is bit-identical to the plain definition.
__device__ __forceinline__ float floor_quotient(float d, float h, float inv_h)
{
    const float y  = __fmul_rn(d, inv_h);
    float fl = floorf(y);
    const float fr  = __fsub_rn(y, fl);
    const float tol = __fmul_rn(fabsf(y), 4.0e-7f);
    if (!(fr >= tol && fr <= __fsub_rn(1.0f, tol))) fl = floorf(__fdiv_rn(d, h));      // also catches NaN/Inf
    return fl;
}

// planar [3][N] displacement field -> one float4 {ux, uy, uz, 0} per DVF node, so that a trilinear corner is one
// 128-bit load instead of three 32-bit loads
__global__ void dvf_interleave_kernel(size_t n, const float* __restrict__ ux, const float* __restrict__ uy,
                                      const float* __restrict__ uz, float4* __restrict__ out)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride)
        out[i] = make_float4(ux[i], uy[i], uz[i], 0.0f);
}

constexpr int kTileX = 32, kTileY = 4, kChunkZMax = 8;

struct PushParams {
    pbs4d_grid src, dvf, ref;
    const float* __restrict__ dose;
    const float* __restrict__ rho;
    const float4* __restrict__ U;            // interleaved DVF
    float inv_hrx, inv_hry, inv_hrz;         // RN(1 / h) of the reference grid
    int nsx, nsy, nsz;
    int chunk_z;                             // source voxels along z handled by one thread (<= kChunkZMax)
    unsigned long long* E;
    unsigned long long* M;
    AccCounters* counters;
};

__global__ void __launch_bounds__(kTileX * kTileY)
emtm_push_kernel(const __grid_constant__ PushParams P)
{
    extern __shared__ AxisEntry s_map[];
    AxisEntry* sx = s_map;                               // [nsx][32]   (subvoxel-major: conflict-free 128-bit reads)
    AxisEntry* sy = sx + kTileX * P.nsx;                 // [4][nsy]
    AxisEntry* sz = sy + kTileY * P.nsy;                 // [chunk_z * nsz]
    longlong2* s_em = reinterpret_cast<longlong2*>(sz + P.chunk_z * P.nsz);   // [chunk_z][128] (e_q, m_q) per voxel
    const int tid = threadIdx.y * kTileX + threadIdx.x;
    const int i = blockIdx.x * kTileX + threadIdx.x;
    const int j = blockIdx.y * kTileY + threadIdx.y;
    const int k0 = blockIdx.z * P.chunk_z;               // this CTA covers source voxels k0 .. k0 + kz_n - 1 along z
    const int kz_n = min(P.chunk_z, P.src.nz - k0);
    const int n_x = kTileX * P.nsx, n_y = kTileY * P.nsy, n_z = kz_n * P.nsz;
    for (int e = tid; e < n_x + n_y + n_z; e += kTileX * kTileY) {
        if (e < n_x)
            s_map[e] = axis_map(P.src.ox, P.src.hx, blockIdx.x * kTileX + (e & (kTileX - 1)), e / kTileX, P.nsx,
                                P.dvf.ox, P.dvf.hx, P.dvf.nx);
        else if (e < n_x + n_y)
            s_map[e] = axis_map(P.src.oy, P.src.hy, blockIdx.y * kTileY + (e - n_x) / P.nsy, (e - n_x) % P.nsy, P.nsy,
                                P.dvf.oy, P.dvf.hy, P.dvf.ny);
        else
            sz[e - n_x - n_y] = axis_map(P.src.oz, P.src.hz, k0 + (e - n_x - n_y) / P.nsz, (e - n_x - n_y) % P.nsz, P.nsz,
                                         P.dvf.oz, P.dvf.hz, P.dvf.nz);
    }
    const bool mine = i < P.src.nx && j < P.src.ny;
    if (mine) {
        for (int kk = 0; kk < kz_n; ++kk) {              // A1: integer mass and energy of this thread's voxels
            const size_t v = ((size_t)(k0 + kk) * P.src.ny + j) * P.src.nx + i;
            const float rho = __ldg(P.rho + v), dose = __ldg(P.dose + v);
            s_em[kk * (kTileX * kTileY) + tid] =
                make_longlong2(__double2ll_rn(__dmul_rn(__dmul_rn((double)rho, (double)dose), 4294967296.0)),
                               __double2ll_rn(__dmul_rn((double)rho, 16777216.0)));
        }
    }
    __syncthreads();

    unsigned n_ref = 0, n_dvf = 0;
    if (mine) {
        const int nsx = P.nsx, nsy = P.nsy, nsz = P.nsz;
        const int dnx = P.dvf.nx, dny = P.dvf.ny;
        const int dx1 = dnx > 1 ? 1 : 0;                 // upper x node = lower + 1 unless the DVF grid is 1 node wide
        const float orx = P.ref.ox, ory = P.ref.oy, orz = P.ref.oz, hrx = P.ref.hx, hry = P.ref.hy, hrz = P.ref.hz;
        const float ihx = P.inv_hrx, ihy = P.inv_hry, ihz = P.inv_hrz;
        const float fnx = (float)P.ref.nx, fny = (float)P.ref.ny, fnz = (float)P.ref.nz;
        const int rnx = P.ref.nx, rny = P.ref.ny;
        const AxisEntry* sxl = sx + threadIdx.x;
        const AxisEntry* syl = sy + threadIdx.y * nsy;
        // Loop nest: y, x outside, z INSIDE.  The integer sums do not depend on the order in which subvoxels are
        // visited, so the nest is arranged for reuse: all subvoxels of a (b, a) column that fall into the same DVF
        // z-cell share the 8 corner vectors and the 6 x- and y-lerps per component (A3); only the z-lerp, q = p + u
        // and the destination index are evaluated per subvoxel.  Each value is computed by exactly the operations
        // of the contract, so the result stays bit-identical.
        const int sz_stride = dny * dnx;
        for (int b = 0; b < nsy; ++b) {
            const AxisEntry my = syl[b];
            const int sy1 = (my.flags & 1) * dnx;
            for (int a = 0; a < nsx; ++a) {
                const AxisEntry mx = sxl[a * kTileX];
                const bool ok_xy = (mx.flags & my.flags & 2) != 0;
                const float4* __restrict__ col = P.U + my.i0 * dnx + mx.i0;       // (y0, x0) of the column, z = 0
                int cell_z = -1;
                float c0x = 0.f, c0y = 0.f, c0z = 0.f, c1x = 0.f, c1y = 0.f, c1z = 0.f;
                for (int kk = 0; kk < kz_n; ++kk) {
                    const longlong2 em = s_em[kk * (kTileX * kTileY) + tid];
                    const long long e_q = em.x, m_q = em.y;
                    int run_dst = -1, run_cnt = 0;
                    for (int c = 0; c < nsz; ++c) {
                        const AxisEntry mz = sz[kk * nsz + c];
                        if (mz.i0 != cell_z) {                                    // new DVF z-cell: corners + x/y lerps
                            cell_z = mz.i0;
                            const float4* __restrict__ p00 = col + mz.i0 * sz_stride;
                            const float4* __restrict__ p10 = p00 + (mz.flags & 1) * sz_stride;
                            const float4 a000 = __ldg(p00), a001 = __ldg(p00 + dx1);
                            const float4 a010 = __ldg(p00 + sy1), a011 = __ldg(p00 + sy1 + dx1);
                            const float4 a100 = __ldg(p10), a101 = __ldg(p10 + dx1);
                            const float4 a110 = __ldg(p10 + sy1), a111 = __ldg(p10 + sy1 + dx1);
#define PBS4D_BILERP(A, B, C, D, cmp) lerp_rn(lerp_rn(A.cmp, B.cmp, mx.w), lerp_rn(C.cmp, D.cmp, mx.w), my.w)
                            c0x = PBS4D_BILERP(a000, a001, a010, a011, x); c1x = PBS4D_BILERP(a100, a101, a110, a111, x);
                            c0y = PBS4D_BILERP(a000, a001, a010, a011, y); c1y = PBS4D_BILERP(a100, a101, a110, a111, y);
                            c0z = PBS4D_BILERP(a000, a001, a010, a011, z); c1z = PBS4D_BILERP(a100, a101, a110, a111, z);
#undef PBS4D_BILERP
                        }
                        const bool ok = ok_xy && (mz.flags & 2);
                        const float qx = __fadd_rn(mx.p, lerp_rn(c0x, c1x, mz.w));  // q = p + u (A4)
                        const float qy = __fadd_rn(my.p, lerp_rn(c0y, c1y, mz.w));
                        const float qz = __fadd_rn(mz.p, lerp_rn(c0z, c1z, mz.w));
                        const float fx = floor_quotient(__fsub_rn(qx, orx), hrx, ihx);
                        const float fy = floor_quotient(__fsub_rn(qy, ory), hry, ihy);
                        const float fz = floor_quotient(__fsub_rn(qz, orz), hrz, ihz);
                        const bool inside = fx >= 0.0f && fx < fnx && fy >= 0.0f && fy < fny && fz >= 0.0f && fz < fnz;
                        n_dvf += ok ? 0u : 1u;
                        n_ref += (ok && !inside) ? 1u : 0u;
                        const int dst = (ok && inside) ? ((int)fz * rny + (int)fy) * rnx + (int)fx : -1;
                        // merge consecutive subvoxels of the voxel that land in the same reference voxel
                        if (dst != run_dst) {
                            if (run_dst >= 0) {
                                atomicAdd(P.E + run_dst, (unsigned long long)(run_cnt * e_q));
                                atomicAdd(P.M + run_dst, (unsigned long long)(run_cnt * m_q));
                            }
                            run_dst = dst; run_cnt = 0;
                        }
                        run_cnt += 1;
                    }
                    if (run_dst >= 0) {
                        atomicAdd(P.E + run_dst, (unsigned long long)(run_cnt * e_q));
                        atomicAdd(P.M + run_dst, (unsigned long long)(run_cnt * m_q));
                    }
                }
            }
        }
    }
    // drop counters: warp-reduce, one atomic per warp
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        n_ref += __shfl_xor_sync(0xffffffffu, n_ref, off);
        n_dvf += __shfl_xor_sync(0xffffffffu, n_dvf, off);
    }
    if (threadIdx.x == 0) {
        if (n_ref) atomicAdd(&P.counters->dropped_ref, (unsigned long long)n_ref);
        if (n_dvf) atomicAdd(&P.counters->dropped_dvf, (unsigned long long)n_dvf);
    }
}

constexpr int kMaxSrc = 32;
struct CoverParams { pbs4d_grid ref; int n_src; pbs4d_grid dvf[kMaxSrc]; unsigned char* flags; };

// mask (A6): a reference voxel is kept iff its centre lies inside the voxel extent of every source
// DVF.  The test is separable, so it is evaluated once per axis index into flags[nx | ny | nz] (1 = covered).
__global__ void emtm_cover_kernel(const __grid_constant__ CoverParams P)
{
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    const int nx = P.ref.nx, ny = P.ref.ny, nz = P.ref.nz;
    if (e >= nx + ny + nz) return;
    const int axis = e < nx ? 0 : (e < nx + ny ? 1 : 2);
    const int i = axis == 0 ? e : (axis == 1 ? e - nx : e - nx - ny);
    const float o = axis == 0 ? P.ref.ox : (axis == 1 ? P.ref.oy : P.ref.oz);
    const float h = axis == 0 ? P.ref.hx : (axis == 1 ? P.ref.hy : P.ref.hz);
    const float p = __fadd_rn(o, __fmul_rn(__fadd_rn((float)i, 0.5f), h));
    bool covered = true;
    for (int s = 0; s < P.n_src; ++s) {
        const pbs4d_grid& d = P.dvf[s];
        const float od = axis == 0 ? d.ox : (axis == 1 ? d.oy : d.oz);
        const float hd = axis == 0 ? d.hx : (axis == 1 ? d.hy : d.hz);
        const int   nd = axis == 0 ? d.nx : (axis == 1 ? d.ny : d.nz);
        const float g = __fsub_rn(__fdiv_rn(__fsub_rn(p, od), hd), 0.5f);
        covered = covered && (g >= -0.5f) && (g < __fsub_rn((float)nd, 0.5f));
    }
    P.flags[e] = covered ? 1 : 0;
}

struct FinalizeParams {
    pbs4d_grid ref;
    const float* __restrict__ dose_ref;
    int n_src;
    const long long* E[kMaxSrc];
    const long long* M[kMaxSrc];
    const unsigned char* __restrict__ flags;
    float* out;
};

__device__ __forceinline__ double ratio_add(double D, long long e, long long m)
{
    return m != 0 ? __dadd_rn(D, __dmul_rn(__ddiv_rn((double)e, (double)m), 1.0 / 256.0)) : D;
}

// Eq. 5 then Eq. 2 per reference voxel.  HBM-bound: (16 n_src + 4) B read + 4 B written per voxel; one thread
// handles two x-adjacent voxels so the int64 sums move as 128-bit loads (rows are 16-byte aligned when nx is even;
// odd nx takes the scalar path).
template <bool kPair>
__global__ void __launch_bounds__(128)
emtm_finalize_kernel(const __grid_constant__ FinalizeParams P)
{
    const int row = blockIdx.x;                          // j + ny * k (grid.x: up to 2^31-1 rows)
    const int nx = P.ref.nx, ny = P.ref.ny;
    const int j = row % ny, k = row / ny;
    const bool row_ok = P.flags[nx + j] && P.flags[nx + ny + k];
    const size_t base = (size_t)row * nx;
    if (kPair) {
        const int i = 2 * (blockIdx.y * blockDim.x + threadIdx.x);
        if (i >= nx) return;
        const size_t v = base + i;
        const bool c0 = row_ok && P.flags[i], c1 = row_ok && P.flags[i + 1];
        const float2 dr = *reinterpret_cast<const float2*>(P.dose_ref + v);
        double D0 = (double)dr.x, D1 = (double)dr.y;
        for (int s = 0; s < P.n_src; ++s) {
            const longlong2 e = *reinterpret_cast<const longlong2*>(P.E[s] + v);
            const longlong2 m = *reinterpret_cast<const longlong2*>(P.M[s] + v);
            D0 = ratio_add(D0, e.x, m.x);
            D1 = ratio_add(D1, e.y, m.y);
        }
        *reinterpret_cast<float2*>(P.out + v) = make_float2(c0 ? (float)D0 : 0.0f, c1 ? (float)D1 : 0.0f);
    } else {
        const int i = blockIdx.y * blockDim.x + threadIdx.x;
        if (i >= nx) return;
        const size_t v = base + i;
        double D = (double)P.dose_ref[v];
        for (int s = 0; s < P.n_src; ++s) D = ratio_add(D, P.E[s][v], P.M[s][v]);
        P.out[v] = (row_ok && P.flags[i]) ? (float)D : 0.0f;
    }
}

// ------------------------------------------------------------------------------------------------------------------
// Dose-interpolation method (DIM, Eq. 3): pull.  One thread per reference voxel loops over its
// nsx*nsy*nsz subvoxel centres r_ik: displacement T^{R->S}(r_ik) by trilinear interpolation of the (float4) DVF,
// q = r + u, trilinear dose of the source phase at q (clamp-to-edge inside the source grid's voxel extent, 0
// outside), sum in double in (c, b, a) order, D_i^S = sum / n^3, added to a double accumulator that was initialised
// with D_i^R (Eq. 2: phases are added in ascending order, one launch per source phase on one stream).
// No atomics: every reference voxel is owned by one thread.
// ------------------------------------------------------------------------------------------------------------------
struct PullParams {
    pbs4d_grid ref, dvf, src;
    const float4* __restrict__ U;            // T^{R->S}, interleaved, on grid dvf (reference frame)
    const float* __restrict__ dose;          // source-phase dose on grid src
    double* acc;                             // [ref voxels]
    int nsx, nsy, nsz;
    AccCounters* counters;
};

struct Cell { int i0, d1; float w; bool ok; };
__device__ __forceinline__ Cell cell_of(float p, float o, float h, int n)
{
    Cell c;
    float g = __fsub_rn(__fdiv_rn(__fsub_rn(p, o), h), 0.5f);
    c.ok = (g >= -0.5f) && (g < __fsub_rn((float)n, 0.5f));
    g = fminf(fmaxf(g, 0.0f), (float)(n - 1));
    int k = (int)floorf(g);
    k = max(min(k, n - 2), 0);
    c.i0 = k;
    c.d1 = min(k + 1, n - 1) - k;
    c.w  = __fsub_rn(g, (float)k);
    return c;
}

__global__ void __launch_bounds__(kTileX * kTileY)
dim_pull_kernel(const __grid_constant__ PullParams P)
{
    extern __shared__ AxisEntry s_map[];
    AxisEntry* sx = s_map;
    AxisEntry* sy = sx + kTileX * P.nsx;
    AxisEntry* sz = sy + kTileY * P.nsy;
    const int tid = threadIdx.y * kTileX + threadIdx.x;
    const int i = blockIdx.x * kTileX + threadIdx.x;
    const int j = blockIdx.y * kTileY + threadIdx.y;
    const int k = blockIdx.z;
    const int n_x = kTileX * P.nsx, n_y = kTileY * P.nsy;
    for (int e = tid; e < n_x + n_y + P.nsz; e += kTileX * kTileY) {
        if (e < n_x)
            s_map[e] = axis_map(P.ref.ox, P.ref.hx, blockIdx.x * kTileX + (e & (kTileX - 1)), e / kTileX, P.nsx,
                                P.dvf.ox, P.dvf.hx, P.dvf.nx);
        else if (e < n_x + n_y)
            s_map[e] = axis_map(P.ref.oy, P.ref.hy, blockIdx.y * kTileY + (e - n_x) / P.nsy, (e - n_x) % P.nsy, P.nsy,
                                P.dvf.oy, P.dvf.hy, P.dvf.ny);
        else
            s_map[e] = axis_map(P.ref.oz, P.ref.hz, k, e - n_x - n_y, P.nsz, P.dvf.oz, P.dvf.hz, P.dvf.nz);
    }
    __syncthreads();

    unsigned n_src = 0, n_dvf = 0;
    if (i < P.ref.nx && j < P.ref.ny) {
        const int nsx = P.nsx, nsy = P.nsy, nsz = P.nsz;
        const int dnx = P.dvf.nx, dny = P.dvf.ny;
        const int dx1 = dnx > 1 ? 1 : 0;
        const int snx = P.src.nx, sny = P.src.ny, snz = P.src.nz;
        const float sox = P.src.ox, soy = P.src.oy, soz = P.src.oz, shx = P.src.hx, shy = P.src.hy, shz = P.src.hz;
        const AxisEntry* sxl = sx + threadIdx.x;
        const AxisEntry* syl = sy + threadIdx.y * nsy;
        double sum = 0.0;
        for (int c = 0; c < nsz; ++c) {
            const AxisEntry mz = sz[c];
            for (int b = 0; b < nsy; ++b) {
                const AxisEntry my = syl[b];
                const int r00 = (mz.i0 * dny + my.i0) * dnx;
                const int sy1 = (my.flags & 1) * dnx, sz1 = (mz.flags & 1) * dny * dnx;
                const float4* __restrict__ p00 = P.U + r00;
                const float4* __restrict__ p01 = p00 + sy1;
                const float4* __restrict__ p10 = p00 + sz1;
                const float4* __restrict__ p11 = p10 + sy1;
                const bool ok_zy = (mz.flags & my.flags & 2) != 0;
                for (int a = 0; a < nsx; ++a) {
                    const AxisEntry mx = sxl[a * kTileX];
                    if (!(ok_zy && (mx.flags & 2))) { n_dvf += 1; continue; }
                    const int x0 = mx.i0;
                    const float4 a000 = __ldg(p00 + x0), a001 = __ldg(p00 + x0 + dx1);
                    const float4 a010 = __ldg(p01 + x0), a011 = __ldg(p01 + x0 + dx1);
                    const float4 a100 = __ldg(p10 + x0), a101 = __ldg(p10 + x0 + dx1);
                    const float4 a110 = __ldg(p11 + x0), a111 = __ldg(p11 + x0 + dx1);
#define PBS4D_TRILERP(cmp) lerp_rn(lerp_rn(lerp_rn(a000.cmp, a001.cmp, mx.w), lerp_rn(a010.cmp, a011.cmp, mx.w), my.w), \
                                   lerp_rn(lerp_rn(a100.cmp, a101.cmp, mx.w), lerp_rn(a110.cmp, a111.cmp, mx.w), my.w), mz.w)
                    const float qx = __fadd_rn(mx.p, PBS4D_TRILERP(x));
                    const float qy = __fadd_rn(my.p, PBS4D_TRILERP(y));
                    const float qz = __fadd_rn(mz.p, PBS4D_TRILERP(z));
#undef PBS4D_TRILERP
                    const Cell cx = cell_of(qx, sox, shx, snx), cy = cell_of(qy, soy, shy, sny),
                               cz = cell_of(qz, soz, shz, snz);
                    if (!(cx.ok && cy.ok && cz.ok)) { n_src += 1; continue; }
                    const float* __restrict__ d00 = P.dose + ((size_t)cz.i0 * sny + cy.i0) * snx + cx.i0;
                    const float* __restrict__ d01 = d00 + cy.d1 * snx;
                    const float* __restrict__ d10 = d00 + (size_t)cz.d1 * sny * snx;
                    const float* __restrict__ d11 = d10 + cy.d1 * snx;
                    const float c00 = lerp_rn(__ldg(d00), __ldg(d00 + cx.d1), cx.w);
                    const float c01 = lerp_rn(__ldg(d01), __ldg(d01 + cx.d1), cx.w);
                    const float c10 = lerp_rn(__ldg(d10), __ldg(d10 + cx.d1), cx.w);
                    const float c11 = lerp_rn(__ldg(d11), __ldg(d11 + cx.d1), cx.w);
                    const float val = lerp_rn(lerp_rn(c00, c01, cy.w), lerp_rn(c10, c11, cy.w), cz.w);
                    sum = __dadd_rn(sum, (double)val);
                }
            }
        }
        const size_t v = ((size_t)k * P.ref.ny + j) * P.ref.nx + i;
        const double n3 = __dmul_rn(__dmul_rn((double)nsx, (double)nsy), (double)nsz);
        P.acc[v] = __dadd_rn(P.acc[v], __ddiv_rn(sum, n3));
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        n_src += __shfl_xor_sync(0xffffffffu, n_src, off);
        n_dvf += __shfl_xor_sync(0xffffffffu, n_dvf, off);
    }
    if (threadIdx.x == 0) {
        if (n_src) atomicAdd(&P.counters->dropped_ref, (unsigned long long)n_src);
        if (n_dvf) atomicAdd(&P.counters->dropped_dvf, (unsigned long long)n_dvf);
    }
}

__global__ void dim_init_kernel(size_t n, const float* __restrict__ dose_ref, double* __restrict__ acc)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) acc[i] = (double)dose_ref[i];
}

__global__ void __launch_bounds__(128)
dim_final_kernel(pbs4d_grid ref, const double* __restrict__ acc, const unsigned char* __restrict__ flags,
                 float* __restrict__ out)
{
    const int row = blockIdx.x;
    const int nx = ref.nx, ny = ref.ny;
    const int j = row % ny, k = row / ny;
    const bool row_ok = flags[nx + j] && flags[nx + ny + k];
    const int i = blockIdx.y * blockDim.x + threadIdx.x;
    if (i >= nx) return;
    const size_t v = (size_t)row * nx + i;
    out[v] = (row_ok && flags[i]) ? (float)acc[v] : 0.0f;
}

}  // namespace

void launch_dvf_interleave(const pbs4d_grid& g, const float* disp_planar, float* out4, cudaStream_t st)
{
    const size_t n = (size_t)g.nx * g.ny * g.nz;
    const int blocks = (int)std::min<size_t>((n + 255) / 256, (size_t)148 * 16);
    dvf_interleave_kernel<<<blocks, 256, 0, st>>>(n, disp_planar, disp_planar + n, disp_planar + 2 * n,
                                                  reinterpret_cast<float4*>(out4));
}

void launch_emtm_push(const pbs4d_grid& src, const float* dose, const float* rho, const pbs4d_grid& dvf_grid,
                      const float* disp4, const pbs4d_grid& ref, int nsx, int nsy, int nsz,
                      long long* E, long long* M, AccCounters* counters, cudaStream_t st)
{
    PushParams P;
    P.src = src; P.dvf = dvf_grid; P.ref = ref; P.dose = dose; P.rho = rho;
    P.U = reinterpret_cast<const float4*>(disp4);
    P.inv_hrx = 1.0f / ref.hx; P.inv_hry = 1.0f / ref.hy; P.inv_hrz = 1.0f / ref.hz;
    P.nsx = nsx; P.nsy = nsy; P.nsz = nsz;
    P.E = (unsigned long long*)E; P.M = (unsigned long long*)M; P.counters = counters;
    // z-chunk per thread: with <= 2 subvoxels per voxel along z, neighbouring voxels share DVF z-cells and a column of
    // 8 voxels per thread halves the x/y-lerp work and amortises the CTA prologue (measured +12 % at n = 2); with more
    // subvoxels per voxel the sharing is already inside the voxel and longer columns only cost registers (-10 % at n = 8)
    P.chunk_z = nsz <= 2 ? kChunkZMax : 1;
    dim3 b(kTileX, kTileY, 1), g((src.nx + kTileX - 1) / kTileX, (src.ny + kTileY - 1) / kTileY,
                                 (src.nz + P.chunk_z - 1) / P.chunk_z);
    const size_t smem = (size_t)(kTileX * nsx + kTileY * nsy + P.chunk_z * nsz) * sizeof(AxisEntry) +
                        (size_t)P.chunk_z * kTileX * kTileY * sizeof(longlong2);
    static bool configured = false;
    if (!configured) {                                   // up to 57 KB at 64 subvoxels per axis
        cudaFuncSetAttribute(emtm_push_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024);
        configured = true;
    }
    emtm_push_kernel<<<g, b, smem, st>>>(P);
}

void launch_emtm_finalize(const pbs4d_grid& ref, const float* dose_ref, int n_src, const long long* const* E_host,
                          const long long* const* M_host, const pbs4d_grid* dvf_grids_host, unsigned char* flags_dev,
                          float* out, cudaStream_t st)
{
    CoverParams C;
    C.ref = ref; C.n_src = n_src; C.flags = flags_dev;
    for (int s = 0; s < n_src && s < kMaxSrc; ++s) C.dvf[s] = dvf_grids_host[s];
    const int n_axis = ref.nx + ref.ny + ref.nz;
    emtm_cover_kernel<<<(n_axis + 127) / 128, 128, 0, st>>>(C);

    FinalizeParams P;
    P.ref = ref; P.dose_ref = dose_ref; P.n_src = n_src; P.out = out; P.flags = flags_dev;
    for (int s = 0; s < n_src && s < kMaxSrc; ++s) { P.E[s] = E_host[s]; P.M[s] = M_host[s]; }
    const bool pair = (ref.nx % 2 == 0) && (reinterpret_cast<uintptr_t>(out) % 8 == 0) &&
                      (reinterpret_cast<uintptr_t>(dose_ref) % 8 == 0);
    const int per_row = pair ? ref.nx / 2 : ref.nx;
    dim3 g(ref.ny * ref.nz, (per_row + 127) / 128);
    if (pair) emtm_finalize_kernel<true><<<g, 128, 0, st>>>(P);
    else      emtm_finalize_kernel<false><<<g, 128, 0, st>>>(P);
}

void launch_dim_init(const pbs4d_grid& ref, const float* dose_ref, double* acc, cudaStream_t st)
{
    const size_t n = (size_t)ref.nx * ref.ny * ref.nz;
    const int blocks = (int)std::min<size_t>((n + 255) / 256, (size_t)148 * 16);
    dim_init_kernel<<<blocks, 256, 0, st>>>(n, dose_ref, acc);
}

void launch_dim_pull(const pbs4d_grid& ref, int nsx, int nsy, int nsz, const pbs4d_grid& dvf_grid, const float* disp4,
                     const pbs4d_grid& src, const float* dose_src, double* acc, AccCounters* counters, cudaStream_t st)
{
    PullParams P;
    P.ref = ref; P.dvf = dvf_grid; P.src = src; P.U = reinterpret_cast<const float4*>(disp4); P.dose = dose_src;
    P.acc = acc; P.nsx = nsx; P.nsy = nsy; P.nsz = nsz; P.counters = counters;
    dim3 b(kTileX, kTileY, 1), g((ref.nx + kTileX - 1) / kTileX, (ref.ny + kTileY - 1) / kTileY, ref.nz);
    const size_t smem = (size_t)(kTileX * nsx + kTileY * nsy + nsz) * sizeof(AxisEntry);
    dim_pull_kernel<<<g, b, smem, st>>>(P);
}

void launch_dim_final(const pbs4d_grid& ref, int n_src, const pbs4d_grid* dvf_grids_host, const double* acc,
                      unsigned char* flags_dev, float* out, cudaStream_t st)
{
    CoverParams C;
    C.ref = ref; C.n_src = n_src; C.flags = flags_dev;
    for (int s = 0; s < n_src && s < kMaxSrc; ++s) C.dvf[s] = dvf_grids_host[s];
    const int n_axis = ref.nx + ref.ny + ref.nz;
    emtm_cover_kernel<<<(n_axis + 127) / 128, 128, 0, st>>>(C);
    dim3 g(ref.ny * ref.nz, (ref.nx + 127) / 128);
    dim_final_kernel<<<g, 128, 0, st>>>(ref, acc, flags_dev, out);
}

}  // namespace pbs4d
