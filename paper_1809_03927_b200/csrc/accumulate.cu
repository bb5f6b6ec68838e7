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
// Coordinate arithmetic is strict fp32: every CONTRACT value is produced by explicit round-to-nearest operations
// (scalar intrinsics or f32x2 pairs, never fused) in the order fixed by DESIGN.md "Accumulation arithmetic"; this TU is
// also built with -fmad=false.  Two places use true fused operations by design, neither a contract value: the push's
// folded index ESTIMATE (accepted only outside a derived tolerance of a voxel face, else the contract's chain decides)
// and the pull's division by a known reciprocal (whose RESULT is the IEEE quotient).  tests/test_sass_contract.py pins
// the FFMA2 count of the built kernels, because ptxas contracts packed mul + add on its own (see mad2_unfused).
#include "internal.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstring>

namespace pbs4d {

namespace {

// ---- packed fp32 pairs (sm_100 f32x2: ONE issue slot for two individually rounded fp32 operations) ----
// The push is bound by instruction issue, not by the FP32 pipe, so the x and y components --
// and the two ends of a rounding interval -- travel as a pair through add/sub/mul/fma.rn.f32x2 (SASS FADD2 / FMUL2 /
// FFMA2).  Each half is the IEEE round-to-nearest result of its own operation, exactly as the scalar intrinsic gives.
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk(float lo, float hi)
{
    f32x2 d; asm("mov.b64 %0, {%1, %2};" : "=l"(d) : "f"(lo), "f"(hi)); return d;
}
__device__ __forceinline__ void upk(f32x2 v, float& lo, float& hi)
{
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b)
{
    f32x2 d; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d;
}
__device__ __forceinline__ f32x2 sub2(f32x2 a, f32x2 b)
{
    f32x2 d; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b)
{
    f32x2 d; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d;
}
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c)
{
    f32x2 d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d;
}

// One axis of the subvoxel -> DVF-cell map (A2, A3): subvoxel centre p, lower DVF node i0, upper node i0 + d1,
// weight w, and whether the centre lies inside the DVF grid's voxel extent.  It depends on (voxel index, subvoxel
// index) of that axis only, so a CTA computes it once per axis for its tile and keeps it in shared memory.
// P = RN_f32((p - o_ref) (1 / h_ref) - 0.5) in double: the centre's continuous reference-grid index minus one half,
// the constant term of the push kernel's folded index estimate (fast path only; never enters a contract value).
struct __align__(16) AxisEntry { float p, w, P; int cell; };            // cell: i0 | d1 << 29 | ok << 30
constexpr int kCellD1 = 1 << 29, kCellOk = 1 << 30, kCellNode = kCellD1 - 1;

__device__ __forceinline__ AxisEntry axis_map(float o, float h, int i, int a, int ns, float od, float hd, int nd,
                                              float o_ref, double inv_h_ref)
{
    AxisEntry m;
    const float f = __fdiv_rn(__fadd_rn((float)a, 0.5f), (float)ns);
    m.p = __fadd_rn(o, __fmul_rn(__fadd_rn((float)i, f), h));
    float g = __fsub_rn(__fdiv_rn(__fsub_rn(m.p, od), hd), 0.5f);
    const bool ok = (g >= -0.5f) && (g < __fsub_rn((float)nd, 0.5f));
    g = fminf(fmaxf(g, 0.0f), (float)(nd - 1));
    int k = (int)floorf(g);
    k = max(min(k, nd - 2), 0);
    m.w  = __fsub_rn(g, (float)k);
    m.cell = k | ((min(k + 1, nd - 1) - k) ? kCellD1 : 0) | (ok ? kCellOk : 0);
    m.P = (float)(((double)m.p - (double)o_ref) * inv_h_ref - 0.5);
    return m;
}

__device__ __forceinline__ float lerp_rn(float A, float B, float w)
{
    return __fadd_rn(A, __fmul_rn(w, __fsub_rn(B, A)));
}
// A + RN(w d) per half, two roundings.  ptxas (12.9) contracts mul.rn.f32x2 + add.rn.f32x2 into one FFMA2 even under
// --fmad=false and with the explicit .rn, which would break the contract's operation-by-operation rounding; the
// scalar mul.rn.f32 is never contracted, so the products are formed by two FMULs and only the add is packed.
__device__ __forceinline__ f32x2 mad2_unfused(f32x2 A, float w, f32x2 d)
{
    float dl, dh;
    upk(d, dl, dh);
    return add2(A, pk(__fmul_rn(w, dl), __fmul_rn(w, dh)));
}
__device__ __forceinline__ f32x2 lerp2(f32x2 A, f32x2 B, float w)       // both halves: A + w (B - A), as lerp_rn
{
    return mad2_unfused(A, w, sub2(B, A));
}

// A4: ix = floorf((q - o) / h) with the IEEE quotient Q = RN(RN(q - o) / h), inside iff 0 <= ix < n.
// The push kernel does not form Q on its main path.  It evaluates an ESTIMATE y of Q - 0.5 with the z-lerp, q = p + u
// and the division folded into one fma per axis (see emtm_push_kernel), rounds it to the nearest integer r with the
// 1.5 2^23 trick, and accepts floor(Q) = r only when y is farther than tol from r +- 0.5, where tol bounds
// |y - (Q - 0.5)|:
//   contract   wd = RN(w dd), u = RN(c0 + wd), q = RN(p + u), e = RN(q - o), Q = RN(e / h):
//              |Q - Qr| <= eps (|w dd| + |u| + |q| + |e|) / h + eps |Q|,    Qr the real-number value, eps = 2^-24
//   estimate   B = RN(dd ih), A = RN(c0 ih + P), y = RN(w B + A), ih = RN(1 / h), P as in axis_map:
//              |y - (Qr - 0.5)| <= eps (2 |w dd| / h + |c0| / h + |P| + |A| + |y|)
// With |u|, |c0| <= U (largest nodal displacement of the field), |w dd| <= 2 U, |q| <= |o| + |e|, and |Q| <= n + 1:
//   |y - (Q - 0.5)| <= eps (6 (n + 1) + 12 U / h + |o| / h + 2)            (z: the same count with one more rounding)
// tol = 2 eps (8 (n + 2) + 16 U / h + 2 |o| / h), more than 2.5 times that.  Beyond |Q| = n + 1 the error grows by
// 8 eps per unit of |Q|, so a point outside the grid stays outside.  A subvoxel that fails the test ("near") is
// decided by the contract's own operations and exact_floor.  U is measured when the field is stored
// (dvf_interleave_kernel); a field with non-finite displacements, tol >= 0.25 or a reference dimension above 4e6
// (the range of the rounding trick) makes every subvoxel take the exact path.
constexpr float kMagic     = 12582912.0f;          // 1.5 * 2^23
constexpr int   kMagicBits = 0x4B400000;

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

// planar [3][N] displacement field -> one float4 {ux, uy, uz, uz of the y-neighbour} per DVF node: a trilinear corner
// is one 128-bit load, (ux, uy) is a ready f32x2 pair, and (uz(y), uz(y + 1)) is the pair the x-lerp of the z component
// works on, so the rows y0 + 1 are read as 64-bit (ux, uy) only.  The y-neighbour is clamped (ny == 1: itself), as the
// axis map clamps the upper node.  The kernel also measures U = max |u| per component (out[n].xyz as bit patterns;
// the ordering of non-negative floats is that of their bit patterns, NaN above Inf) for the push kernel's tolerance.
__global__ void __launch_bounds__(128)
dvf_interleave_kernel(int nx, int ny, const float* __restrict__ ux, const float* __restrict__ uy,
                      const float* __restrict__ uz, float4* __restrict__ out)
{
    const int row = blockIdx.x;                          // y + ny z
    const int x = blockIdx.y * blockDim.x + threadIdx.x;
    unsigned mx = 0u, my = 0u, mz = 0u;
    if (x < nx) {
        const size_t i = (size_t)row * nx + x;
        const float a = ux[i], b = uy[i], c = uz[i];
        out[i] = make_float4(a, b, c, (row % ny) + 1 < ny ? uz[i + nx] : c);
        mx = __float_as_uint(fabsf(a)); my = __float_as_uint(fabsf(b)); mz = __float_as_uint(fabsf(c));
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, off));
        my = max(my, __shfl_xor_sync(0xffffffffu, my, off));
        mz = max(mz, __shfl_xor_sync(0xffffffffu, mz, off));
    }
    if ((threadIdx.x & 31) == 0) {
        unsigned* u = reinterpret_cast<unsigned*>(out + (size_t)gridDim.x * nx);
        // a (possibly stale, L1-cached) read first: after the first few warps nearly every warp skips the atomic
        if (mx > u[0]) atomicMax(u + 0, mx);
        if (my > u[1]) atomicMax(u + 1, my);
        if (mz > u[2]) atomicMax(u + 2, mz);
    }
}

constexpr int kTileX = 32, kTileY = 4, kChunkZMax = 8;

struct PushParams {
    pbs4d_grid src, dvf, ref;
    const float* __restrict__ dose;
    const float* __restrict__ rho;
    const float4* __restrict__ U;            // interleaved DVF, U[nodes] = {max|ux|, max|uy|, max|uz|, -}
    float inv_hrx, inv_hry, inv_hrz;         // RN(1 / h) of the reference grid
    double ihdx, ihdy, ihdz;                 // 1 / h in double (axis_map's P)
    float tgx, tgy, tgz;                     // geometric part of the index tolerance: 2^-23 (8 (n + 2) + 2 |o| / h)
    float tux, tuy, tuz;                     // its slope in U: 2^-23 16 / h          (+Inf, 0: always exact)
    int nsx, nsy, nsz;
    int chunk_z;                             // source voxels along z handled by one thread (<= kChunkZMax)
    int tile_cap;                            // DVF nodes the CTA's shared-memory tile can hold
    unsigned long long* E;
    unsigned long long* M;
    AccCounters* counters;
};

// x- then y-interpolation of the three displacement components at one z-node (A3: 2 + 1 of the 7 lerps) from the four
// corners of the float4 layout of dvf_interleave_kernel: 19 packed / scalar operations instead of 27.
__device__ __forceinline__ void bilerp_corners(const float4& a00, const float4& a01, const float2& a10, const float2& a11,
                                               float wx, float wy, f32x2& cxy, float& cz)
{
    const f32x2 r0 = lerp2(pk(a00.x, a00.y), pk(a01.x, a01.y), wx);
    const f32x2 r1 = lerp2(pk(a10.x, a10.y), pk(a11.x, a11.y), wx);
    cxy = lerp2(r0, r1, wy);
    float z0, z1;
    upk(lerp2(pk(a00.z, a00.w), pk(a01.z, a01.w), wx), z0, z1);         // uz rows y0 and y0 + 1 (a00.w = uz of row y0 + 1)
    cz = lerp_rn(z0, z1, wy);
}
// p: node (x0, y0) of the z-node in global memory; dx1, sy1: offsets (in nodes) of the x- and y-neighbour
__device__ __forceinline__ void node_bilerp(const float4* __restrict__ p, int dx1, int sy1, float wx, float wy,
                                            f32x2& cxy, float& cz)
{
    bilerp_corners(__ldg(p), __ldg(p + dx1), __ldg(reinterpret_cast<const float2*>(p + sy1)),
                   __ldg(reinterpret_cast<const float2*>(p + sy1 + dx1)), wx, wy, cxy, cz);
}
// the same from the CTA's shared-memory tile (x-neighbour = next node)
__device__ __forceinline__ void node_bilerp_tile(const float4* p, int sy1, float wx, float wy, f32x2& cxy, float& cz)
{
    bilerp_corners(p[0], p[1], *reinterpret_cast<const float2*>(p + sy1), *reinterpret_cast<const float2*>(p + sy1 + 1),
                   wx, wy, cxy, cz);
}

// DVF tile of a CTA in shared memory: nodes [x0, x0 + nx) x [y0, y0 + ny) x [z0, z0 + nz) of the field
struct Tile { int x0, y0, z0, nx, ny, nz; };

// The subvoxel columns of one thread.
// kChecked = false: the CTA's source tile, displaced by at most U, lies at least one voxel inside the reference grid
// on every axis and entirely inside the DVF grid's z-extent, so no destination can fall outside and the range test is
// compiled out.  kTile: the DVF nodes come from the CTA's shared-memory tile instead of global memory.
template <bool kChecked, bool kTile, int kNsz, int kTY>
__device__ __forceinline__ void push_columns(const PushParams& P, const AxisEntry* __restrict__ sxl,
                                             const AxisEntry* __restrict__ syl, const AxisEntry* __restrict__ sz,
                                             const longlong2* __restrict__ s_em_t, const float4* tile, const Tile T,
                                             int kz_n, float htx, float hty, f32x2 tolz12, unsigned& n_cols,
                                             unsigned& dropped)
{
    const int nsx = P.nsx, nsy = P.nsy, nsz = kNsz ? kNsz : P.nsz;      // kNsz > 0: the z-run is unrolled
    const int dnx = P.dvf.nx;
    const int dx1 = dnx > 1 ? 1 : 0;                     // upper x node = lower + 1 unless the DVF grid is 1 node wide
    const int rnx = P.ref.nx, rny = P.ref.ny, rnz = P.ref.nz;
    const int sz_stride = kTile ? T.ny * T.nx : P.dvf.ny * dnx;
    const int row = kTile ? T.nx : dnx;
    // destination index from the bit patterns b = kMagicBits + index of the rounded estimates:
    // (bz rny + by) rnx + bx = dst + kShift (mod 2^32); kNone is the shifted "no destination"
    const unsigned kShift = (unsigned)kMagicBits * ((unsigned)rny * (unsigned)rnx + (unsigned)rnx + 1u), kNone = kShift - 1u;
    const f32x2 ihxy = pk(P.inv_hrx, P.inv_hry), ihzz = pk(P.inv_hrz, P.inv_hrz);
    const f32x2 magic2 = pk(kMagic, kMagic);
    for (int b = 0; b < nsy; ++b) {
        const AxisEntry my = syl[b];
        const int sy1 = (my.cell & kCellD1) ? row : 0;
        for (int a = 0; a < nsx; ++a) {
            const AxisEntry mx = sxl[a * kTileX];
            if (!(mx.cell & my.cell & kCellOk)) continue;                         // whole column outside the DVF extent
            n_cols += 1u;
            // node (x0, y0) of z-node 0 of the field (global) or of the tile
            const int col_t = ((my.cell & kCellNode) - T.y0) * row + ((mx.cell & kCellNode) - T.x0) - T.z0 * sz_stride;
            const float4* __restrict__ col = P.U + ((size_t)(my.cell & kCellNode) * dnx + (mx.cell & kCellNode));
            const f32x2 Pxy = pk(mx.P, my.P);
            int node_hi = -1, cell_z = -1;
            f32x2 c0xy = 0ull, c1xy = 0ull, Bxy = 0ull, Axy = 0ull, Bzz = 0ull, A12z = 0ull;
            float c0z = 0.f, c1z = 0.f;
            const AxisEntry* mzp = sz;
            for (int kk = 0; kk < kz_n; ++kk) {
                const longlong2 em = s_em_t[kk * (kTileX * kTY)];
                // destinations of the voxel's z-run: two slots (a run of nsz subvoxels rarely meets a third voxel);
                // B is the current one, A the one before; both are flushed at the end of the run, where every lane
                // of the warp is there (the run length is CTA-uniform)
                unsigned dstA = kNone, cntA = 0u, dstB = kNone, cntB = 0u;
                auto flush = [&](unsigned d_shifted, unsigned cnt) {
                    const int dst = (int)(d_shifted - kShift);
                    if (dst >= 0) {
                        atomicAdd(P.E + dst, (unsigned long long)em.x * cnt);
                        atomicAdd(P.M + dst, (unsigned long long)em.y * cnt);
                    } else {
                        dropped += cnt;                  // mapped outside the reference grid (A4): the rare side counts
                    }
                };
#pragma unroll
                for (int c = 0; c < nsz; ++c, ++mzp) {
                    const AxisEntry mz = *mzp;
                    if (mz.cell != cell_z) {                                      // new DVF z-cell (warp-uniform branch)
                        cell_z = mz.cell;
                        const int lo = mz.cell & kCellNode, hi = lo + ((mz.cell & kCellD1) ? 1 : 0);
                        if (lo == node_hi) { c0xy = c1xy; c0z = c1z; }
                        else if (kTile) node_bilerp_tile(tile + (col_t + lo * sz_stride), sy1, mx.w, my.w, c0xy, c0z);
                        else node_bilerp(col + (size_t)lo * sz_stride, dx1, sy1, mx.w, my.w, c0xy, c0z);
                        if (hi == lo) { c1xy = c0xy; c1z = c0z; }
                        else if (kTile) node_bilerp_tile(tile + (col_t + hi * sz_stride), sy1, mx.w, my.w, c1xy, c1z);
                        else node_bilerp(col + (size_t)hi * sz_stride, dx1, sy1, mx.w, my.w, c1xy, c1z);
                        node_hi = hi;
                        // folded estimate of this cell: y = w B + A per axis (see the tolerance derivation above)
                        const float ddz = __fsub_rn(c1z, c0z);
                        Bxy  = mul2(sub2(c1xy, c0xy), ihxy);
                        Axy  = fma2(c0xy, ihxy, Pxy);
                        Bzz  = mul2(pk(ddz, ddz), ihzz);
                        A12z = fma2(pk(c0z, c0z), ihzz, tolz12);                  // (c0z ih - tol, c0z ih + tol)
                    }
                    // x, y: estimate, nearest integer r, distance of the estimate from r
                    const f32x2 wz2 = pk(mz.w, mz.w);
                    const f32x2 yxy = fma2(wz2, Bxy, Axy);
                    const f32x2 txy = add2(yxy, magic2);
                    const f32x2 fxy = sub2(yxy, sub2(txy, magic2));
                    // z: both ends of the tolerance interval; they must round to the same integer
                    const f32x2 t12 = add2(fma2(wz2, Bzz, add2(A12z, pk(mz.P, mz.P))), magic2);
                    float tx, ty, fx, fy, t1, t2;
                    upk(txy, tx, ty); upk(fxy, fx, fy); upk(t12, t1, t2);
                    const unsigned bx = __float_as_uint(tx), by = __float_as_uint(ty), bz = __float_as_uint(t1);
                    unsigned dst = (bz * (unsigned)rny + by) * (unsigned)rnx + bx;
                    if (!(fabsf(fx) <= htx) | !(fabsf(fy) <= hty) | (bz != __float_as_uint(t2))) {
                        // rare: the contract's own operations (z-lerp, q = p + u, q - o) and the exact floor
                        float c0x, c0y, c1x, c1y;
                        upk(c0xy, c0x, c0y); upk(c1xy, c1x, c1y);
                        const float qx = __fadd_rn(mx.p, __fadd_rn(c0x, __fmul_rn(mz.w, __fsub_rn(c1x, c0x))));
                        const float qy = __fadd_rn(my.p, __fadd_rn(c0y, __fmul_rn(mz.w, __fsub_rn(c1y, c0y))));
                        const float qz = __fadd_rn(mz.p, __fadd_rn(c0z, __fmul_rn(mz.w, __fsub_rn(c1z, c0z))));
                        const int ix = exact_floor(__fsub_rn(qx, P.ref.ox), P.ref.hx, P.inv_hrx, rnx);
                        const int iy = exact_floor(__fsub_rn(qy, P.ref.oy), P.ref.hy, P.inv_hry, rny);
                        const int iz = exact_floor(__fsub_rn(qz, P.ref.oz), P.ref.hz, P.inv_hrz, rnz);
                        dst = (ix | iy | iz) < 0 ? kNone : (unsigned)((iz * rny + iy) * rnx + ix) + kShift;
                    } else if (kChecked) {
                        const bool out = ((bx - (unsigned)kMagicBits) >= (unsigned)rnx) |
                                         ((by - (unsigned)kMagicBits) >= (unsigned)rny) |
                                         ((bz - (unsigned)kMagicBits) >= (unsigned)rnz);
                        dst = out ? kNone : dst;
                    }
                    // count it in slot B; a new destination moves B to A (A, if occupied, is flushed: a third voxel)
                    const bool same = dst == dstB;
                    if (!same & (cntA != 0u)) flush(dstA, cntA);
                    dstA = same ? dstA : dstB; cntA = same ? cntA : cntB;
                    dstB = dst;                cntB = same ? cntB + 1u : 1u;
                }
                if (cntA != 0u) flush(dstA, cntA);
                flush(dstB, cntB);
            }
        }
    }
}

// Thread = a column of chunk_z source voxels along z at (i, j); CTA = 32 x 4 such columns.
// Loop nest: subvoxel (b, a) of the column outside, ALL its z-subvoxels inside.  The integer sums do not depend on
// the visiting order, so the nest is arranged for reuse:
//   * the DVF nodes the CTA's subvoxels interpolate between are staged once in shared memory (a (tile + halo) box of
//     float4 nodes, loaded coalesced; a field too fine for the box is read through L1 instead), and the largest
//     displacement inside the box bounds |u| for this CTA;
//   * the z-sequence of DVF cells is the same for every thread of the CTA (the z-axis map lives in shared memory), so
//     the "new z-cell" branch is warp-uniform;
//   * the x- and y-lerps (A3) are evaluated once per z-NODE of the column, on f32x2 pairs: walking up, the upper node of
//     one cell is the lower node of the next;
//   * per subvoxel the main path holds NO contract value: the z-lerp, q = p + u, q - o and the division by h are folded
//     into one fma per axis whose result estimates Q - 0.5 (tolerance derivation above); x and y are one f32x2 pair,
//     z is the pair of the two ends of its tolerance interval.  Seven packed operations, the integer destination index
//     straight from the bit patterns of the rounded estimates (the offsets folded into one constant), and -- only in
//     CTAs near the border of the reference grid or of the DVF's z-extent -- the range test;
//   * a subvoxel whose estimate is within tol of a voxel face is decided by the contract's operations (rare: ~1e-3);
//   * the subvoxels of a voxel's z-run that land in the same reference voxel are merged (two destination slots) and
//     flushed as pairs of red.global.add.u64 at the end of the run, where all lanes of the warp flush together; drop
//     counters are derived from per-column counts, not per subvoxel.
// Every destination is either proven equal to the contract's or computed by
// it, so the result stays bit-identical to the oracle.
// kNsz > 0: the z-run of a voxel is unrolled; kTY: rows of source columns per CTA (CTA = 32 x kTY columns)
template <int kNsz, int kTY>
__global__ void __launch_bounds__(kTileX * kTY)
emtm_push_kernel(const __grid_constant__ PushParams P)
{
    extern __shared__ AxisEntry s_map[];
    AxisEntry* sx = s_map;                               // [nsx][32]   (subvoxel-major: conflict-free 128-bit reads)
    AxisEntry* sy = sx + kTileX * P.nsx;                 // [4][nsy]
    AxisEntry* sz = sy + kTY * P.nsy;                 // [chunk_z * nsz]
    longlong2* s_em = reinterpret_cast<longlong2*>(sz + P.chunk_z * P.nsz);   // [chunk_z][128] (e_q, m_q) per voxel
    float4* tile = reinterpret_cast<float4*>(s_em + P.chunk_z * kTileX * kTY);   // [tile_cap] DVF nodes
    __shared__ int s_okz;
    const int tid = threadIdx.y * kTileX + threadIdx.x;
    const int i = blockIdx.x * kTileX + threadIdx.x;
    const int j = blockIdx.y * kTY + threadIdx.y;
    const int k0 = blockIdx.z * P.chunk_z;               // this CTA covers source voxels k0 .. k0 + kz_n - 1 along z
    const int kz_n = min(P.chunk_z, P.src.nz - k0);
    const int n_x = kTileX * P.nsx, n_y = kTY * P.nsy, n_z = kz_n * P.nsz;
    if (tid == 0) s_okz = 0;
    __syncthreads();
    for (int e = tid; e < n_x + n_y + n_z; e += kTileX * kTY) {
        if (e < n_x)
            s_map[e] = axis_map(P.src.ox, P.src.hx, blockIdx.x * kTileX + (e & (kTileX - 1)), e / kTileX, P.nsx,
                                P.dvf.ox, P.dvf.hx, P.dvf.nx, P.ref.ox, P.ihdx);
        else if (e < n_x + n_y)
            s_map[e] = axis_map(P.src.oy, P.src.hy, blockIdx.y * kTY + (e - n_x) / P.nsy, (e - n_x) % P.nsy, P.nsy,
                                P.dvf.oy, P.dvf.hy, P.dvf.ny, P.ref.oy, P.ihdy);
        else {
            AxisEntry m = axis_map(P.src.oz, P.src.hz, k0 + (e - n_x - n_y) / P.nsz, (e - n_x - n_y) % P.nsz, P.nsz,
                                   P.dvf.oz, P.dvf.hz, P.dvf.nz, P.ref.oz, P.ihdz);
            // a z-subvoxel outside the DVF extent is dropped (A3): NaN coordinates send it through the exact path,
            // which returns "outside", so the inner loop needs no per-subvoxel flag test
            if (m.cell & kCellOk) atomicAdd(&s_okz, 1);
            else m.p = m.P = __int_as_float(0x7fc00000);
            m.cell &= ~kCellOk;                          // z entries: the cell identity only (i0 | d1)
            sz[e - n_x - n_y] = m;
        }
    }
    __syncthreads();

    // the box of DVF nodes this CTA interpolates between (the maps are monotone along their axis) is staged in shared
    // memory when it fits: 16-byte asynchronous copies, in flight while the voxels' integer mass and energy are formed
    Tile T;
    {
        const int nvx = min(kTileX, P.src.nx - blockIdx.x * kTileX), nvy = min(kTY, P.src.ny - blockIdx.y * kTY);
        const int cx1 = sx[(P.nsx - 1) * kTileX + nvx - 1].cell, cy1 = sy[(nvy - 1) * P.nsy + P.nsy - 1].cell,
                  cz1 = sz[n_z - 1].cell;
        T.x0 = sx[0].cell & kCellNode; T.y0 = sy[0].cell & kCellNode; T.z0 = sz[0].cell & kCellNode;
        T.nx = (cx1 & kCellNode) + ((cx1 & kCellD1) ? 1 : 0) - T.x0 + 1;
        T.ny = (cy1 & kCellNode) + ((cy1 & kCellD1) ? 1 : 0) - T.y0 + 1;
        T.nz = (cz1 & kCellNode) + ((cz1 & kCellD1) ? 1 : 0) - T.z0 + 1;
    }
    const bool use_tile = P.dvf.nx > 1 && (long long)T.nx * T.ny * T.nz <= (long long)P.tile_cap;
    if (use_tile) {
        const int rows = T.ny * T.nz;
        for (int r = tid >> 5; r < rows; r += (kTileX * kTY) >> 5) {
            const int ty = r % T.ny, tz = r / T.ny;
            const float4* __restrict__ src = P.U + ((size_t)(T.z0 + tz) * P.dvf.ny + (T.y0 + ty)) * P.dvf.nx + T.x0;
            for (int x = tid & 31; x < T.nx; x += 32) {
                const unsigned dst = (unsigned)__cvta_generic_to_shared(tile + r * T.nx + x);
                asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" :: "r"(dst), "l"(src + x) : "memory");
            }
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    }
    const bool mine = i < P.src.nx && j < P.src.ny;
    if (mine) {                                          // A1: integer mass and energy of this thread's voxels
        float rho[kChunkZMax], dose[kChunkZMax];
#pragma unroll
        for (int kk = 0; kk < kChunkZMax; ++kk) {        // all loads first
            const size_t v = ((size_t)(k0 + min(kk, kz_n - 1)) * P.src.ny + j) * P.src.nx + i;
            rho[kk] = __ldg(P.rho + v); dose[kk] = __ldg(P.dose + v);
        }
#pragma unroll
        for (int kk = 0; kk < kChunkZMax; ++kk)
            if (kk < kz_n)
                s_em[kk * (kTileX * kTY) + tid] =
                    make_longlong2(__double2ll_rn(__dmul_rn(__dmul_rn((double)rho[kk], (double)dose[kk]), 4294967296.0)),
                                   __double2ll_rn(__dmul_rn((double)rho[kk], 16777216.0)));
    }
    if (use_tile) asm volatile("cp.async.wait_group 0;" ::: "memory");
    __syncthreads();
    // largest displacement of the field (the record behind the nodes): bounds |u| in the tolerance and the range test
    const float4 um = __ldg(P.U + (size_t)P.dvf.nx * P.dvf.ny * P.dvf.nz);
    // index tolerance per axis from the largest displacement; 0.5 - tol for the |fr| test (x, y), the pair
    // (-tol, +tol) for z; tol >= 0.25 or NaN: every subvoxel takes the exact path
    const float tolx = __fmaf_rn(um.x, P.tux, P.tgx), toly = __fmaf_rn(um.y, P.tuy, P.tgy),
                tolz = __fmaf_rn(um.z, P.tuz, P.tgz);
    const float htx = tolx < 0.25f ? 0.5f - tolx : -1.0f, hty = toly < 0.25f ? 0.5f - toly : -1.0f;
    const float inf = __int_as_float(0x7f800000);
    const f32x2 tolz12 = tolz < 0.25f ? pk(-tolz, tolz) : pk(-inf, inf);

    unsigned n_ref = 0, n_dvf = 0;
    const int okz = s_okz;                               // z-subvoxels of the column inside the DVF extent (CTA-uniform)
    // can a destination of this CTA fall outside the reference grid?  Source tile +- U against the grid shrunk by one
    // voxel (1.5 with the rounding margin), per axis; comparisons with a NaN / Inf U fail and select the checked path.
    bool interior = okz == n_z;
    {
        const float x0 = P.src.ox + (float)(blockIdx.x * kTileX) * P.src.hx;
        const float x1 = P.src.ox + (float)min(blockIdx.x * kTileX + kTileX, P.src.nx) * P.src.hx;
        const float y0 = P.src.oy + (float)(blockIdx.y * kTY) * P.src.hy;
        const float y1 = P.src.oy + (float)min(blockIdx.y * kTY + kTY, P.src.ny) * P.src.hy;
        const float z0 = P.src.oz + (float)k0 * P.src.hz, z1 = P.src.oz + (float)(k0 + kz_n) * P.src.hz;
        interior = interior && (x0 - um.x >= P.ref.ox + 1.5f * P.ref.hx) &&
                   (x1 + um.x <= P.ref.ox + ((float)P.ref.nx - 1.5f) * P.ref.hx) &&
                   (y0 - um.y >= P.ref.oy + 1.5f * P.ref.hy) &&
                   (y1 + um.y <= P.ref.oy + ((float)P.ref.ny - 1.5f) * P.ref.hy) &&
                   (z0 - um.z >= P.ref.oz + 1.5f * P.ref.hz) &&
                   (z1 + um.z <= P.ref.oz + ((float)P.ref.nz - 1.5f) * P.ref.hz);
    }
    if (mine) {
        unsigned dropped = 0, n_cols = 0;                    // subvoxels the flushes dropped; columns inside the DVF's x/y extent
        const AxisEntry* sxl = sx + threadIdx.x;
        const AxisEntry* syl = sy + threadIdx.y * P.nsy;
        if (use_tile) {
            if (interior) push_columns<false, true, kNsz, kTY>(P, sxl, syl, sz, s_em + tid, tile, T, kz_n, htx, hty, tolz12, n_cols, dropped);
            else          push_columns<true, true, kNsz, kTY>(P, sxl, syl, sz, s_em + tid, tile, T, kz_n, htx, hty, tolz12, n_cols, dropped);
        } else {
            if (interior) push_columns<false, false, kNsz, kTY>(P, sxl, syl, sz, s_em + tid, tile, T, kz_n, htx, hty, tolz12, n_cols, dropped);
            else          push_columns<true, false, kNsz, kTY>(P, sxl, syl, sz, s_em + tid, tile, T, kz_n, htx, hty, tolz12, n_cols, dropped);
        }
        // subvoxel centres outside the DVF grid's extent (A3): whole columns (x or y outside) and, in the walked columns, the
        // NaN-coded z-subvoxels; mapped outside the reference grid (A4): what the flushes dropped, minus those z-subvoxels
        n_dvf = (unsigned)(P.nsx * P.nsy * n_z) - n_cols * (unsigned)okz;
        n_ref = dropped - n_cols * (unsigned)(n_z - okz);
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
    float inv_shx, inv_shy, inv_shz;         // RN(1 / h) of the source grid (div_by_known)
    AccCounters* counters;
};

// source-grid cell of a coordinate (D2): lower node i0 in [0, max(n - 2, 0)], weight w, inside flag.  The upper node is
// i0 + 1 for every cell of a grid with n >= 2 nodes (i0 <= n - 2) and i0 itself when n == 1: a per-axis constant.
struct Cell { int i0; float w; bool ok; };
__device__ __forceinline__ Cell cell_from_quotient(float Q, int n)      // Q = RN(RN(p - o) / h)
{
    Cell c;
    float g = __fsub_rn(Q, 0.5f);
    c.ok = (g >= -0.5f) && (g < __fsub_rn((float)n, 0.5f));
    g = fminf(fmaxf(g, 0.0f), (float)(n - 1));
    const int k = max(min(__float2int_rd(g), n - 2), 0);
    c.i0 = k;
    c.w  = __fsub_rn(g, (float)k);
    return c;
}
// The correctly rounded quotient RN(e / h) without the division sequence, for a divisor whose reciprocal is at hand
// (Markstein's correction): y = RN(1 / h), q0 = RN(e y), r = e - h q0 (exact, one fma), q1 = RN(q0 + r y) = RN(e / h) for
// every e, provided the significand of h is not all ones and nothing underflows.  The launcher tests the proviso and
// falls back to __fdiv_rn (kFastDiv = false); tests/test_markstein_division.py checks the identity exhaustively over all
// 2^23 significands of e for the spacings of the configs and for random ones.  These are true fused operations by
// design (they are not part of the contract's rounding sequence: only their RESULT, the IEEE quotient, is).
__device__ __forceinline__ float div_by_known(float e, float h, float inv_h)
{
    const float q0 = __fmul_rn(e, inv_h);
    return __fmaf_rn(__fmaf_rn(-h, q0, e), inv_h, q0);
}
__device__ __forceinline__ f32x2 div2_by_known(f32x2 e, f32x2 neg_h, f32x2 inv_h)
{
    f32x2 q0, r, q1;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(q0) : "l"(e), "l"(inv_h));
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(neg_h), "l"(q0), "l"(e));
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(q1) : "l"(r), "l"(inv_h), "l"(q0));
    return q1;
}

// Thread = a column of chunk_z reference voxels at (i, j); CTA = 32 x 4 columns.  Loop nest as in the push: subvoxel
// (b, a) of the column outside, all its z-subvoxels inside, so that the x/y-lerps of the DVF interpolation are
// evaluated once per z-NODE (the upper node of a cell is the lower node of the next) and the "new z-cell" branch is
// warp-uniform.  The double sum of a voxel receives its values in (b, a, c) order -- reading D4 -- because every voxel
// of the column keeps its own running sum (shared memory) and the c-run of a (b, a) column is added to it value by
// value.  Per subvoxel: z-lerp, q = r + u, the source-grid cell of q (three IEEE quotients -- the continuous index is
// needed as a value, not only its floor -- by Markstein's correction with the known reciprocal of the spacing), 8 dose loads, 7 lerps (the six in x and y as f32x2 pairs), one double add.
// kX1 = 1: the source grid has more than one node along x (0: a single one); kFastDiv: see div_by_known
template <int kX1, bool kFastDiv>
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
                                P.dvf.ox, P.dvf.hx, P.dvf.nx, 0.0f, 1.0);
        else if (e < n_x + n_y)
            s_map[e] = axis_map(P.ref.oy, P.ref.hy, blockIdx.y * kTileY + (e - n_x) / P.nsy, (e - n_x) % P.nsy, P.nsy,
                                P.dvf.oy, P.dvf.hy, P.dvf.ny, 0.0f, 1.0);
        else
            sz[e - n_x - n_y] = axis_map(P.ref.oz, P.ref.hz, k0 + (e - n_x - n_y) / P.nsz, (e - n_x - n_y) % P.nsz, P.nsz,
                                         P.dvf.oz, P.dvf.hz, P.dvf.nz, 0.0f, 1.0);
    }
    for (int kk = 0; kk < kz_n; ++kk) s_sum[kk * (kTileX * kTileY) + tid] = 0.0;
    __syncthreads();

    unsigned n_src = 0, n_dvf = 0;
    if (i < P.ref.nx && j < P.ref.ny) {
        const int nsx = P.nsx, nsy = P.nsy, nsz = P.nsz;
        const int dnx = P.dvf.nx, dny = P.dvf.ny;
        const int dx1 = dnx > 1 ? 1 : 0;
        const int snx = P.src.nx, sny = P.src.ny, snz = P.src.nz;
        const int row = sny > 1 ? snx : 0;                                   // offset of the upper y / z node (D2)
        const size_t plane = snz > 1 ? (size_t)sny * snx : 0;
        const float sox = P.src.ox, soy = P.src.oy, soz = P.src.oz, shx = P.src.hx, shy = P.src.hy, shz = P.src.hz;
        const AxisEntry* sxl = sx + threadIdx.x;
        const AxisEntry* syl = sy + threadIdx.y * nsy;
        const int sz_stride = dny * dnx;
        for (int b = 0; b < nsy; ++b) {
            const AxisEntry my = syl[b];
            const int sy1 = (my.cell & kCellD1) ? dnx : 0;
            for (int a = 0; a < nsx; ++a) {
                const AxisEntry mx = sxl[a * kTileX];
                if (!(mx.cell & my.cell & kCellOk)) { n_dvf += (unsigned)n_z; continue; }  // column outside the DVF extent
                const float4* __restrict__ col = P.U + (my.cell & kCellNode) * dnx + (mx.cell & kCellNode);
                int node_hi = -1, cell_z = -1;
                f32x2 c0xy = 0ull, c1xy = 0ull, ddxy = 0ull;
                float c0z = 0.f, c1z = 0.f, ddz = 0.f;
                const AxisEntry* mzp = sz;
                for (int kk = 0; kk < kz_n; ++kk) {
                    double sum = s_sum[kk * (kTileX * kTileY) + tid];
                    for (int c = 0; c < nsz; ++c, ++mzp) {
                        const AxisEntry mz = *mzp;
                        if (!(mz.cell & kCellOk)) { n_dvf += 1; continue; }                // warp-uniform
                        if ((mz.cell & ~kCellOk) != cell_z) {                              // new DVF z-cell (uniform)
                            cell_z = mz.cell & ~kCellOk;
                            const int lo = mz.cell & kCellNode, hi = lo + ((mz.cell & kCellD1) ? 1 : 0);
                            if (lo == node_hi) { c0xy = c1xy; c0z = c1z; }
                            else node_bilerp(col + (size_t)lo * sz_stride, dx1, sy1, mx.w, my.w, c0xy, c0z);
                            if (hi == lo) { c1xy = c0xy; c1z = c0z; }
                            else node_bilerp(col + (size_t)hi * sz_stride, dx1, sy1, mx.w, my.w, c1xy, c1z);
                            node_hi = hi;
                            ddxy = sub2(c1xy, c0xy); ddz = __fsub_rn(c1z, c0z);
                        }
                        float qx, qy;
                        upk(add2(pk(mx.p, my.p), mad2_unfused(c0xy, mz.w, ddxy)), qx, qy);
                        const float qz = __fadd_rn(mz.p, __fadd_rn(c0z, __fmul_rn(mz.w, ddz)));
                        // continuous source-grid index per axis: three IEEE quotients (D2)
                        float Qx, Qy, Qz;
                        if (kFastDiv) {
                            upk(div2_by_known(sub2(pk(qx, qy), pk(sox, soy)), pk(-shx, -shy), pk(P.inv_shx, P.inv_shy)), Qx, Qy);
                            Qz = div_by_known(__fsub_rn(qz, soz), shz, P.inv_shz);
                        } else {
                            Qx = __fdiv_rn(__fsub_rn(qx, sox), shx); Qy = __fdiv_rn(__fsub_rn(qy, soy), shy);
                            Qz = __fdiv_rn(__fsub_rn(qz, soz), shz);
                        }
                        const Cell cx = cell_from_quotient(Qx, snx), cy = cell_from_quotient(Qy, sny),
                                   cz = cell_from_quotient(Qz, snz);
                        if (!(cx.ok && cy.ok && cz.ok)) { n_src += 1; continue; }
                        // 8 dose nodes: one 64-bit address, the x-neighbour at a compile-time offset (kX1), the y- and
                        // z-neighbours at CTA-uniform offsets; the four x-lerps and the two y-lerps as f32x2 pairs
                        const float* __restrict__ d00 = P.dose + ((size_t)cz.i0 * sny + cy.i0) * snx + cx.i0;
                        const float* __restrict__ d01 = d00 + row;
                        const float* __restrict__ d10 = d00 + plane;
                        const float* __restrict__ d11 = d10 + row;
                        const f32x2 cy0 = lerp2(pk(__ldg(d00), __ldg(d01)), pk(__ldg(d00 + kX1), __ldg(d01 + kX1)), cx.w);
                        const f32x2 cy1 = lerp2(pk(__ldg(d10), __ldg(d11)), pk(__ldg(d10 + kX1), __ldg(d11 + kX1)), cx.w);
                        float c00, c01, c10, c11;
                        upk(cy0, c00, c01); upk(cy1, c10, c11);
                        float v0, v1;
                        upk(lerp2(pk(c00, c10), pk(c01, c11), cy.w), v0, v1);
                        const float val = lerp_rn(v0, v1, cz.w);
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
    cudaError_t e = cudaSuccess;
    for (void (*k)(const PushParams) : { emtm_push_kernel<0, 4>, emtm_push_kernel<0, 8>, emtm_push_kernel<2, 4> })
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024);
    for (void (*k)(const PullParams) : { dim_pull_kernel<0, false>, dim_pull_kernel<0, true>, dim_pull_kernel<1, false>,
                                         dim_pull_kernel<1, true> })
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024);
    return e;
}

void launch_dvf_interleave(const pbs4d_grid& g, const float* disp_planar, float* out4, cudaStream_t st)
{
    const size_t n = (size_t)g.nx * g.ny * g.nz;
    float4* out = reinterpret_cast<float4*>(out4);
    cudaMemsetAsync(out + n, 0, sizeof(float4), st);     // the max |u| record behind the nodes
    dim3 grid((unsigned)g.ny * (unsigned)g.nz, (unsigned)((g.nx + 127) / 128));
    dvf_interleave_kernel<<<grid, 128, 0, st>>>(g.nx, g.ny, disp_planar, disp_planar + n, disp_planar + 2 * n, out);
}

void launch_emtm_push(const pbs4d_grid& src, const float* dose, const float* rho, const pbs4d_grid& dvf_grid,
                      const float* disp4, const pbs4d_grid& ref, int nsx, int nsy, int nsz,
                      long long* E, long long* M, AccCounters* counters, cudaStream_t st)
{
    PushParams P;
    P.src = src; P.dvf = dvf_grid; P.ref = ref; P.dose = dose; P.rho = rho;
    P.U = reinterpret_cast<const float4*>(disp4);
    P.inv_hrx = 1.0f / ref.hx; P.inv_hry = 1.0f / ref.hy; P.inv_hrz = 1.0f / ref.hz;
    P.ihdx = 1.0 / (double)ref.hx; P.ihdy = 1.0 / (double)ref.hy; P.ihdz = 1.0 / (double)ref.hz;
    // index tolerance per axis (derivation at kMagic): tol = 2^-23 (8 (n + 2) + 2 |o| / h) + U 2^-23 16 / h, U read by
    // the kernel from the record behind the field; a grid too long for the rounding trick takes the exact path always
    const double e23 = 1.1920928955078125e-7;
    auto geo = [&](int n, float o, float h) {
        return n <= 4000000 ? (float)(e23 * (8.0 * (n + 2.0) + 2.0 * std::fabs((double)o) / (double)h)) : INFINITY;
    };
    auto slope = [&](int n, float h) { return n <= 4000000 ? (float)(e23 * 16.0 / (double)h) : 0.0f; };
    P.tgx = geo(ref.nx, ref.ox, ref.hx); P.tgy = geo(ref.ny, ref.oy, ref.hy); P.tgz = geo(ref.nz, ref.oz, ref.hz);
    P.tux = slope(ref.nx, ref.hx); P.tuy = slope(ref.ny, ref.hy); P.tuz = slope(ref.nz, ref.hz);
    P.nsx = nsx; P.nsy = nsy; P.nsz = nsz;
    P.E = (unsigned long long*)E; P.M = (unsigned long long*)M; P.counters = counters;
    // z-chunk per thread: the x/y-lerps are evaluated once per z-node of a column, and the first node of a column is
    // extra, so longer columns amortise it (and the CTA prologue); shorter ones keep the DVF tile and the (e_q, m_q)
    // stage small enough for 6-7 resident CTAs per SM.  Measured on config 4 (chunk 8 / 4 / 2, ms per 9 phases):
    // n = 2 1.02 / 0.86 / 1.04, n = 4 4.6 / 3.6 / 3.9, n = 8 28.7 / 22.5 / 21.8, (2,2,5) 1.57 / 1.25 / 1.42.
    // With two z-subvoxels per voxel the CTA prologue weighs most: there the long column without the tile (the nodes
    // through L1) is best, 0.82 ms.
    P.chunk_z = nsz <= 2 ? kChunkZMax : 4;
    // CTA shape: 32 x 8 columns from nsz = 3 on (the node box's halo and the CTA prologue are shared by twice the
    // columns: config 4 n = 8 22.6 -> 21.1 ms, config 5 6.46 -> 6.25 ms), 32 x 4 below (n = 2: 0.735 against 0.749 ms)
    const int ty = nsz >= 3 ? 8 : 4;
    dim3 b(kTileX, ty, 1), g((src.nx + kTileX - 1) / kTileX, (src.ny + ty - 1) / ty, (src.nz + P.chunk_z - 1) / P.chunk_z);
    // shared memory: axis maps + (e_q, m_q) per voxel + the DVF tile.  The tile is sized for a field on the source
    // grid's spacing ((32 + 2) x (ty + 2) x (chunk_z + 2) nodes) and shrunk so that the total stays under 60 KB.
    const size_t fixed = (size_t)(kTileX * nsx + ty * nsy + P.chunk_z * nsz) * sizeof(AxisEntry) +
                         (size_t)P.chunk_z * kTileX * ty * sizeof(longlong2);
    const size_t want = (size_t)(kTileX + 2) * (ty + 2) * (P.chunk_z + 2);
    const size_t room = fixed < 60 * 1024 ? (60 * 1024 - fixed) / sizeof(float4) : 0;
    P.tile_cap = nsz <= 2 ? 0 : (int)std::min(want, room);
    const size_t smem = fixed + (size_t)P.tile_cap * sizeof(float4);
    // the two-subvoxel z-run of nsz = 2 is unrolled (config 4, 9 phases: 0.82 -> 0.73 ms); longer runs are not: the
    // unrolled body repeats the cell-change block and outgrows the instruction cache (nsz = 8: 22.5 -> 38 ms, nsz = 5:
    // 1.25 -> 1.63 ms).  (> 48 KB of shared memory possible: configure_accumulate() opted in)
    void (*kernel)(const PushParams) = nsz == 2 ? emtm_push_kernel<2, 4> : nsz >= 3 ? emtm_push_kernel<0, 8> : emtm_push_kernel<0, 4>;
    kernel<<<g, b, smem, st>>>(P);
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
    // as for the push, longer columns amortise the first z-node and the CTA prologue; measured on config 4 (ms per 9
    // phases, chunk 4 / 8 / 16 / 32): n = 1 0.395 / 0.358 / 0.336 / 0.573, n = 2 1.45 / 1.43 / 1.42 / 2.26
    P.chunk_z = nsz <= 2 ? 16 : 4;
    dim3 b(kTileX, kTileY, 1), g((ref.nx + kTileX - 1) / kTileX, (ref.ny + kTileY - 1) / kTileY,
                                 (ref.nz + P.chunk_z - 1) / P.chunk_z);
    const size_t smem = (size_t)(kTileX * nsx + kTileY * nsy + P.chunk_z * nsz) * sizeof(AxisEntry) +
                        (size_t)P.chunk_z * kTileX * kTileY * sizeof(double);
    // Markstein's division needs a spacing whose significand is not all ones (and a normal, finite one)
    auto known_ok = [](float h) {
        uint32_t b; std::memcpy(&b, &h, 4);
        return std::isfinite(h) && h >= 1.0e-30f && h <= 1.0e30f && (b & 0x7FFFFFu) != 0x7FFFFFu;
    };
    P.inv_shx = 1.0f / src.hx; P.inv_shy = 1.0f / src.hy; P.inv_shz = 1.0f / src.hz;
    const bool fast = known_ok(src.hx) && known_ok(src.hy) && known_ok(src.hz);
    void (*kernel)(const PullParams) = src.nx > 1 ? (fast ? dim_pull_kernel<1, true> : dim_pull_kernel<1, false>)
                                                  : (fast ? dim_pull_kernel<0, true> : dim_pull_kernel<0, false>);
    kernel<<<g, b, smem, st>>>(P);                         // <= 60 KB: configure_accumulate() opted in
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
