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
#include <cmath>

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

// A4: ix = floorf((q - o) / h) with the IEEE quotient Q = RN(RN(q - o) / h), inside iff 0 <= ix < n.
// Fast path (FMA/ALU pipes only, no division, no conversion instruction, no call):
//   y = fma(q, inv_h, c),  inv_h = RN(1/h),  c = RN(-o inv_h - 0.5)      ~  Q - 0.5
//   t = y + 1.5 2^23  rounds y to the nearest integer r = t - 1.5 2^23 (exact for |y| < 2^22), and r is also the
//   difference of the bit patterns of t and 1.5 2^23.  Unless Q lies close to an integer, floor(Q) = r.
// |y - (Q - 0.5)| <= 2^-24 (|Q| + |q inv_h| + |c| + |y|) + ulp(c)/2: the rounding of q - o that the contract
// prescribes is a relative 2^-24 on Q, inv_h carries a relative 2^-24, c and y one rounding each.  The launcher
// turns this into a per-axis tolerance tol = 4e-7 (n + 2 + 2 |o| / h); when fr = y - r is within tol of +-0.5, Q is
// that close to an integer and the decision is taken exactly (exact_floor).  For |y| >= 2^22 (and +-Inf) the integer
// comes out >= 2^22 - 1 or negative, i.e. outside every grid the fast path is used for (the launcher passes
// tol = +Inf -- always exact -- when a reference dimension exceeds 4e6); NaN fails the comparison and goes exact.
constexpr float kMagic     = 12582912.0f;          // 1.5 * 2^23
constexpr int   kMagicBits = 0x4B400000;

__device__ __forceinline__ bool fast_floor(float q, float inv_h, float c, float half_minus_tol, int& ix)
{
    const float y  = __fmaf_rn(q, inv_h, c);
    const float t  = __fadd_rn(y, kMagic);
    const float fr = __fsub_rn(y, __fsub_rn(t, kMagic));
    ix = __float_as_int(t) - kMagicBits;
    return !(fabsf(fr) <= half_minus_tol);         // true: Q is too close to an integer (or NaN) -> exact_floor
}

// Exact floorf(RN(e / h)) for e = RN(q - o), decided without a division instruction or subroutine (the kernel's
// inner loop stays free of calls).  yq = RN(e inv_h) is within 2^-23 |yq| of Q = RN(e / h); k = the integer nearest
// to yq.  If yq is not that close to k, floor(Q) = floor(yq).  Otherwise Q >= k  <=>  e / h >= m, where m is the
// midpoint between k and the float below it (a tie rounds to k, whose significand is even for every integer
// k < 2^23)  <=>  (double)e >= m (double)h, and that product is exact in double (m has <= 26, h 24 significant bits).
// Returns the index if it is inside [0, n), else -1.  (e / h underflowing to -0 for e < 0 would be floored to -0 =
// "inside" by the definition; that needs |e| < 2^-149 h and cannot occur for coordinates in mm.)
__device__ __forceinline__ int exact_floor(float e, float h, float inv_h, int n)
{
    const float yq = __fmul_rn(e, inv_h);
    if (!(fabsf(yq) < 4194304.0f)) return -1;                          // beyond any grid (or NaN)
    const float k = rintf(yq);
    int fl;
    if (fabsf(__fsub_rn(yq, k)) > __fmul_rn(fabsf(yq), 3.0e-7f) + 1.0e-30f) fl = (int)floorf(yq);
    else if (k < 1.0f) fl = (k == 0.0f && e >= 0.0f) ? 0 : -1;
    else {
        const int kb = __float_as_int(k);
        const int ex = (kb >> 23) - 127;                               // k = 2^ex * 1.f
        const int half_gap_exp = ex - 24 - ((kb & 0x7FFFFF) == 0 ? 1 : 0);      // half the gap to the float below k
        const double m = __dsub_rn((double)k, __hiloint2double((1023 + half_gap_exp) << 20, 0));
        fl = ((double)e >= __dmul_rn(m, (double)h)) ? (int)k : (int)k - 1;
    }
    return (unsigned)fl < (unsigned)n ? fl : -1;
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
    float cx, cy, cz;                        // RN(-o inv_h - 0.5) per axis (fast_floor)
    float htx, hty, htz;                     // 0.5 - tol per axis (fast_floor)
    int nsx, nsy, nsz;
    int chunk_z;                             // source voxels along z handled by one thread (<= kChunkZMax)
    unsigned long long* E;
    unsigned long long* M;
    AccCounters* counters;
};

// the four DVF nodes (x0|x0+1, y0|y0+1) of one z-node that a subvoxel column interpolates between
struct Quad { float4 a00, a01, a10, a11; };

__device__ __forceinline__ Quad load_quad(const float4* __restrict__ p, int dx1, int sy1)
{
    Quad q;
    q.a00 = __ldg(p); q.a01 = __ldg(p + dx1); q.a10 = __ldg(p + sy1); q.a11 = __ldg(p + sy1 + dx1);
    return q;
}

// x- then y-interpolation of the three displacement components at one z-node (A3: 2 + 1 of the 7 lerps)
__device__ __forceinline__ void bilerp3(const Quad& q, float wx, float wy, float& cx, float& cy, float& cz)
{
    cx = lerp_rn(lerp_rn(q.a00.x, q.a01.x, wx), lerp_rn(q.a10.x, q.a11.x, wx), wy);
    cy = lerp_rn(lerp_rn(q.a00.y, q.a01.y, wx), lerp_rn(q.a10.y, q.a11.y, wx), wy);
    cz = lerp_rn(lerp_rn(q.a00.z, q.a01.z, wx), lerp_rn(q.a10.z, q.a11.z, wx), wy);
}

// Thread = a column of chunk_z source voxels along z at (i, j); CTA = 32 x 4 such columns.
// Loop nest: subvoxel (b, a) of the column outside, ALL its z-subvoxels inside.  The integer sums do not depend on
// the visiting order, so the nest is arranged for reuse:
//   * the z-sequence of DVF cells is the same for every thread of the CTA (the z-axis map lives in shared memory), so
//     the "new z-cell" branch is warp-uniform;
//   * the x- and y-lerps (A3) are evaluated once per z-NODE of the column: walking up, the upper node of one cell is
//     the lower node of the next, and the difference c1 - c0 of the z-lerp is formed once per cell;
//   * per subvoxel only the z-lerp (mul, add per component), q = p + u, q - o, the product with RN(1/h) and the
//     floor (fast_floor) remain -- all on the FMA/ALU pipes, no conversion or division instruction;
//   * consecutive subvoxels of a voxel that land in the same reference voxel are merged into one pair of
//     red.global.add.u64; drop counters are derived from per-column counts, not per subvoxel.
// Each value is produced by exactly the operations of the contract, so the
// result stays bit-identical to the oracle.
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
        else {
            AxisEntry m = axis_map(P.src.oz, P.src.hz, k0 + (e - n_x - n_y) / P.nsz, (e - n_x - n_y) % P.nsz, P.nsz,
                                   P.dvf.oz, P.dvf.hz, P.dvf.nz);
            // a z-subvoxel outside the DVF extent is dropped (A3): a NaN coordinate sends it through exact_floor,
            // which returns "outside", so the inner loop needs no per-subvoxel flag test
            if (!(m.flags & 2)) m.p = __int_as_float(0x7fc00000);
            sz[e - n_x - n_y] = m;
        }
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
        const float fcx = P.cx, fcy = P.cy, fcz = P.cz, htx = P.htx, hty = P.hty, htz = P.htz;
        const int rnx = P.ref.nx, rny = P.ref.ny, rnz = P.ref.nz;
        const AxisEntry* sxl = sx + threadIdx.x;
        const AxisEntry* syl = sy + threadIdx.y * nsy;
        const int sz_stride = dny * dnx;
        int okz = 0;                                     // z-subvoxels of the column inside the DVF extent (CTA-uniform)
        for (int s = 0; s < n_z; ++s) okz += (sz[s].flags >> 1) & 1;
        unsigned landed = 0, eligible = 0;
        for (int b = 0; b < nsy; ++b) {
            const AxisEntry my = syl[b];
            const int sy1 = (my.flags & 1) * dnx;
            for (int a = 0; a < nsx; ++a) {
                const AxisEntry mx = sxl[a * kTileX];
                if (!(mx.flags & my.flags & 2)) continue;                         // whole column outside the DVF extent
                eligible += (unsigned)okz;
                const float4* __restrict__ col = P.U + my.i0 * dnx + mx.i0;       // (y0, x0) of the column, z = 0
                int node_hi = -1;                                                 // z-node whose bilerp is held in c1*
                float c0x = 0.f, c0y = 0.f, c0z = 0.f, c1x = 0.f, c1y = 0.f, c1z = 0.f, ddx = 0.f, ddy = 0.f, ddz = 0.f;
                int cell_z = -1;
                const AxisEntry* mzp = sz;
                for (int kk = 0; kk < kz_n; ++kk) {
                    const longlong2 em = s_em[kk * (kTileX * kTileY) + tid];
                    const long long e_q = em.x, m_q = em.y;
                    int run_dst = -1; unsigned run_cnt = 0u;
                    for (int c = 0; c < nsz; ++c, ++mzp) {
                        const AxisEntry mz = *mzp;
                        if (mz.i0 != cell_z) {                                    // new DVF z-cell (warp-uniform branch)
                            cell_z = mz.i0;
                            const int hi = mz.i0 + (mz.flags & 1);
                            if (mz.i0 == node_hi) { c0x = c1x; c0y = c1y; c0z = c1z; }
                            else bilerp3(load_quad(col + (size_t)mz.i0 * sz_stride, dx1, sy1), mx.w, my.w, c0x, c0y, c0z);
                            if (hi == mz.i0) { c1x = c0x; c1y = c0y; c1z = c0z; }
                            else bilerp3(load_quad(col + (size_t)hi * sz_stride, dx1, sy1), mx.w, my.w, c1x, c1y, c1z);
                            node_hi = hi;
                            ddx = __fsub_rn(c1x, c0x); ddy = __fsub_rn(c1y, c0y); ddz = __fsub_rn(c1z, c0z);
                        }
                        // z-lerp (A3), q = p + u (A4), destination index
                        const float qx = __fadd_rn(mx.p, __fadd_rn(c0x, __fmul_rn(mz.w, ddx)));
                        const float qy = __fadd_rn(my.p, __fadd_rn(c0y, __fmul_rn(mz.w, ddy)));
                        const float qz = __fadd_rn(mz.p, __fadd_rn(c0z, __fmul_rn(mz.w, ddz)));
                        int ix, iy, iz;
                        const bool near_x = fast_floor(qx, ihx, fcx, htx, ix);
                        const bool near_y = fast_floor(qy, ihy, fcy, hty, iy);
                        const bool near_z = fast_floor(qz, ihz, fcz, htz, iz);
                        if (near_x | near_y | near_z) {                           // rare: decide exactly
                            ix = exact_floor(__fsub_rn(qx, orx), hrx, ihx, rnx);
                            iy = exact_floor(__fsub_rn(qy, ory), hry, ihy, rny);
                            iz = exact_floor(__fsub_rn(qz, orz), hrz, ihz, rnz);
                        }
                        const bool outside = ((unsigned)ix >= (unsigned)rnx) | ((unsigned)iy >= (unsigned)rny) |
                                             ((unsigned)iz >= (unsigned)rnz);
                        const int dst = outside ? -1 : (iz * rny + iy) * rnx + ix;
                        // merge consecutive subvoxels of the voxel that land in the same reference voxel
                        if (dst != run_dst) {
                            if (run_dst >= 0) {
                                atomicAdd(P.E + run_dst, (unsigned long long)e_q * run_cnt);
                                atomicAdd(P.M + run_dst, (unsigned long long)m_q * run_cnt);
                                landed += run_cnt;
                            }
                            run_dst = dst; run_cnt = 0u;
                        }
                        run_cnt += 1u;
                    }
                    if (run_dst >= 0) {
                        atomicAdd(P.E + run_dst, (unsigned long long)e_q * run_cnt);
                        atomicAdd(P.M + run_dst, (unsigned long long)m_q * run_cnt);
                        landed += run_cnt;
                    }
                }
            }
        }
        n_dvf = (unsigned)(nsx * nsy * n_z) - eligible;   // subvoxel centres outside the DVF grid's extent (A3)
        n_ref = eligible - landed;                        // mapped outside the reference grid (A4)
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
    int chunk_z;                             // reference voxels along z handled by one thread
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

// Thread = a column of chunk_z reference voxels at (i, j); CTA = 32 x 4 columns.  Loop nest as in the push: subvoxel
// (b, a) of the column outside, all its z-subvoxels inside, so that the x/y-lerps of the DVF interpolation are
// evaluated once per z-NODE (the upper node of a cell is the lower node of the next) and the "new z-cell" branch is
// warp-uniform.  The double sum of a voxel receives its values in (b, a, c) order -- reading D4 -- because every voxel
// of the column keeps its own running sum (shared memory) and the c-run of a (b, a) column is added to it value by
// value.  Per subvoxel: z-lerp, q = r + u, the source-grid cell of q (three IEEE divisions: the continuous index is
// needed as a value, not only its floor), 8 dose loads, 7 lerps, one double add.
__global__ void __launch_bounds__(kTileX * kTileY)
dim_pull_kernel(const __grid_constant__ PullParams P)
{
    extern __shared__ AxisEntry s_map[];
    AxisEntry* sx = s_map;
    AxisEntry* sy = sx + kTileX * P.nsx;
    AxisEntry* sz = sy + kTileY * P.nsy;
    double* s_sum = reinterpret_cast<double*>(sz + P.chunk_z * P.nsz);       // [chunk_z][128] running sums
    const int tid = threadIdx.y * kTileX + threadIdx.x;
    const int i = blockIdx.x * kTileX + threadIdx.x;
    const int j = blockIdx.y * kTileY + threadIdx.y;
    const int k0 = blockIdx.z * P.chunk_z;
    const int kz_n = min(P.chunk_z, P.ref.nz - k0);
    const int n_x = kTileX * P.nsx, n_y = kTileY * P.nsy, n_z = kz_n * P.nsz;
    for (int e = tid; e < n_x + n_y + n_z; e += kTileX * kTileY) {
        if (e < n_x)
            s_map[e] = axis_map(P.ref.ox, P.ref.hx, blockIdx.x * kTileX + (e & (kTileX - 1)), e / kTileX, P.nsx,
                                P.dvf.ox, P.dvf.hx, P.dvf.nx);
        else if (e < n_x + n_y)
            s_map[e] = axis_map(P.ref.oy, P.ref.hy, blockIdx.y * kTileY + (e - n_x) / P.nsy, (e - n_x) % P.nsy, P.nsy,
                                P.dvf.oy, P.dvf.hy, P.dvf.ny);
        else
            sz[e - n_x - n_y] = axis_map(P.ref.oz, P.ref.hz, k0 + (e - n_x - n_y) / P.nsz, (e - n_x - n_y) % P.nsz, P.nsz,
                                         P.dvf.oz, P.dvf.hz, P.dvf.nz);
    }
    for (int kk = 0; kk < kz_n; ++kk) s_sum[kk * (kTileX * kTileY) + tid] = 0.0;
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
        const int sz_stride = dny * dnx;
        for (int b = 0; b < nsy; ++b) {
            const AxisEntry my = syl[b];
            const int sy1 = (my.flags & 1) * dnx;
            for (int a = 0; a < nsx; ++a) {
                const AxisEntry mx = sxl[a * kTileX];
                if (!(mx.flags & my.flags & 2)) { n_dvf += (unsigned)n_z; continue; }      // column outside the DVF extent
                const float4* __restrict__ col = P.U + my.i0 * dnx + mx.i0;
                int node_hi = -1, cell_z = -1;
                float c0x = 0.f, c0y = 0.f, c0z = 0.f, c1x = 0.f, c1y = 0.f, c1z = 0.f, ddx = 0.f, ddy = 0.f, ddz = 0.f;
                const AxisEntry* mzp = sz;
                for (int kk = 0; kk < kz_n; ++kk) {
                    double sum = s_sum[kk * (kTileX * kTileY) + tid];
                    for (int c = 0; c < nsz; ++c, ++mzp) {
                        const AxisEntry mz = *mzp;
                        if (!(mz.flags & 2)) { n_dvf += 1; continue; }                     // warp-uniform
                        if (mz.i0 != cell_z) {                                             // new DVF z-cell (uniform)
                            cell_z = mz.i0;
                            const int hi = mz.i0 + (mz.flags & 1);
                            if (mz.i0 == node_hi) { c0x = c1x; c0y = c1y; c0z = c1z; }
                            else bilerp3(load_quad(col + (size_t)mz.i0 * sz_stride, dx1, sy1), mx.w, my.w, c0x, c0y, c0z);
                            if (hi == mz.i0) { c1x = c0x; c1y = c0y; c1z = c0z; }
                            else bilerp3(load_quad(col + (size_t)hi * sz_stride, dx1, sy1), mx.w, my.w, c1x, c1y, c1z);
                            node_hi = hi;
                            ddx = __fsub_rn(c1x, c0x); ddy = __fsub_rn(c1y, c0y); ddz = __fsub_rn(c1z, c0z);
                        }
                        const float qx = __fadd_rn(mx.p, __fadd_rn(c0x, __fmul_rn(mz.w, ddx)));
                        const float qy = __fadd_rn(my.p, __fadd_rn(c0y, __fmul_rn(mz.w, ddy)));
                        const float qz = __fadd_rn(mz.p, __fadd_rn(c0z, __fmul_rn(mz.w, ddz)));
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
                    s_sum[kk * (kTileX * kTileY) + tid] = sum;
                }
            }
        }
        const double n3 = __dmul_rn(__dmul_rn((double)nsx, (double)nsy), (double)nsz);
        for (int kk = 0; kk < kz_n; ++kk) {
            const size_t v = ((size_t)(k0 + kk) * P.ref.ny + j) * P.ref.nx + i;
            P.acc[v] = __dadd_rn(P.acc[v], __ddiv_rn(s_sum[kk * (kTileX * kTileY) + tid], n3));
        }
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

cudaError_t configure_accumulate(void)
{
    // the push kernel's axis maps + per-voxel (e_q, m_q) stage need up to 57 KB of dynamic shared memory at 64
    // subvoxels per axis.  A per-device attribute: pbs4d_create calls this for every context.
    cudaError_t e = cudaFuncSetAttribute(emtm_push_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(dim_pull_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024);
    return e;
}

void launch_dvf_interleave(const pbs4d_grid& g, const float* disp_planar, float* out4, cudaStream_t st)
{
    const size_t n = (size_t)g.nx * g.ny * g.nz;
    const int blocks = (int)std::min<size_t>((n + 255) / 256, (size_t)sm_count_of_current_device() * 16);
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
    // fast_floor constants per axis: c = RN(-o inv_h - 0.5); tolerance 4e-7 (n + 2 + 2 |o| / h) (see fast_floor);
    // 0.5 - tol < 0 (always exact) for grids too long for the 2^22 range of the bit trick
    auto cst = [](float o, float inv_h) { return (float)(-(double)o * (double)inv_h - 0.5); };
    auto hmt = [](int n, float o, float h) {
        const double tol = 4.0e-7 * ((double)n + 2.0 + 2.0 * std::fabs((double)o) / (double)h);
        return (n <= 4000000 && tol < 0.25) ? (float)(0.5 - tol) : -1.0f;
    };
    P.cx = cst(ref.ox, P.inv_hrx); P.cy = cst(ref.oy, P.inv_hry); P.cz = cst(ref.oz, P.inv_hrz);
    P.htx = hmt(ref.nx, ref.ox, ref.hx); P.hty = hmt(ref.ny, ref.oy, ref.hy); P.htz = hmt(ref.nz, ref.oz, ref.hz);
    P.nsx = nsx; P.nsy = nsy; P.nsz = nsz;
    P.E = (unsigned long long*)E; P.M = (unsigned long long*)M; P.counters = counters;
    // z-chunk per thread: the x/y-lerps are evaluated once per z-node of a column, and the first node of a column is
    // extra, so longer columns amortise it (and the CTA prologue); measured on config 4 (chunk 1 -> this choice):
    // n = 4 5.09 -> 4.19 ms, n = 8 29.9 -> 27.4 ms, (2,2,5) 1.69 -> 1.34 ms per 9 phases of 128^3
    P.chunk_z = nsz <= 2 ? kChunkZMax : 4;
    dim3 b(kTileX, kTileY, 1), g((src.nx + kTileX - 1) / kTileX, (src.ny + kTileY - 1) / kTileY,
                                 (src.nz + P.chunk_z - 1) / P.chunk_z);
    const size_t smem = (size_t)(kTileX * nsx + kTileY * nsy + P.chunk_z * nsz) * sizeof(AxisEntry) +
                        (size_t)P.chunk_z * kTileX * kTileY * sizeof(longlong2);
    emtm_push_kernel<<<g, b, smem, st>>>(P);             // > 48 KB possible: configure_accumulate() opted in
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
    const int blocks = (int)std::min<size_t>((n + 255) / 256, (size_t)sm_count_of_current_device() * 16);
    dim_init_kernel<<<blocks, 256, 0, st>>>(n, dose_ref, acc);
}

void launch_dim_pull(const pbs4d_grid& ref, int nsx, int nsy, int nsz, const pbs4d_grid& dvf_grid, const float* disp4,
                     const pbs4d_grid& src, const float* dose_src, double* acc, AccCounters* counters, cudaStream_t st)
{
    PullParams P;
    P.ref = ref; P.dvf = dvf_grid; P.src = src; P.U = reinterpret_cast<const float4*>(disp4); P.dose = dose_src;
    P.acc = acc; P.nsx = nsx; P.nsy = nsy; P.nsz = nsz; P.counters = counters;
    P.chunk_z = nsz <= 2 ? kChunkZMax : 4;               // as for the push: longer columns amortise the first z-node
    dim3 b(kTileX, kTileY, 1), g((ref.nx + kTileX - 1) / kTileX, (ref.ny + kTileY - 1) / kTileY,
                                 (ref.nz + P.chunk_z - 1) / P.chunk_z);
    const size_t smem = (size_t)(kTileX * nsx + kTileY * nsy + P.chunk_z * nsz) * sizeof(AxisEntry) +
                        (size_t)P.chunk_z * kTileX * kTileY * sizeof(double);
    dim_pull_kernel<<<g, b, smem, st>>>(P);              // <= 52 KB: configure_accumulate() opted in
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
