// History-parallel proton transport + dose scoring for sm_100a (Sec. 2.C names
// the engine -- "class II condensed-history proton transport" -- the model itself is BASELINE.json north_star +
// config 1: Philox-counter-seeded histories, step = min(voxel boundary, 1 mm, 2 % of residual range), Bethe-Bloch
// CSDA loss (midpoint rule), Bohr straggling, Highland deflection without log term, 0.5 MeV cutoff deposited
// locally, 64-bit fixed-point atomic scoring).
//
// Layout of the computation (B200-first, not the paper's Titan-X design):
//  * one persistent thread per lane slot; a lane whose history ends refills itself with the next history of the
//    launch (static stride), so warps stay full through the step loop -- the Philox counter is (step, history),
//    never the lane, which makes any lane/history assignment give the same integers;
//  * all arithmetic fp32 on the FP32/MUFU pipes; position is kept in voxel-local coordinates so boundary
//    distances keep full fp32 resolution;
//  * log2-spaced CSDA range table staged in shared memory; stopping power analytic (one MUFU.LG2 each);
//  * deposits are converted to int64 quanta of 2^-k MeV and accumulated in a register while the history stays in
//    one voxel; one red.global.add.u64 per voxel visit, resolved in the L2 (the int64 grid + density grid of a phase
//    is L2-resident for the paper-shaped phantoms);
//  * per-launch tallies (incident/deposited/escaped quanta, steps) are block-reduced, one atomic per block.
#include "internal.h"
#include "physics_tables.h"

#include <cuda_runtime.h>

namespace pbs4d {

namespace {

constexpr int   kThreads   = 128;
constexpr float kInvMp     = 1.0f / 938.27208816f;
constexpr float kMp        = 938.27208816f;
constexpr float kMe        = 0.51099895f;
constexpr float kRatio     = 0.51099895f / 938.27208816f;          // me / Mp
constexpr float kKZA       = 0.307075f * (10.0f / 18.01528f);        // K Z/A, MeV cm2/g
constexpr float kLogArg    = 2.0f * 0.51099895f / 75.0e-6f;          // 2 me c2 / I
constexpr float kInvX0     = 1.0f / 36.08f;
constexpr float kEs        = 13.6f;
constexpr float kEcut      = 0.5f;
constexpr float kSmax      = 1.0f;
constexpr float kFrac      = 0.02f;
constexpr float kTie       = 1.0f + 1.0f / 1024.0f;                  // boundary/step-limit tie tolerance (DESIGN A22)
constexpr float kLn2       = 0.6931471805599453f;
constexpr float kTwoPi     = 6.283185307179586f;
constexpr float kU01       = 1.0f / 8388608.0f;

struct Params {
    pbs4d_grid g;
    const float* __restrict__ rho;
    const DevSegment* __restrict__ segs;
    const float* __restrict__ range_tab;      // kRangeNodes log2(R_w[g/cm2]) values
    int32_t n_segs;
    long long n_hist;
    uint32_t seed_lo, seed_hi, flags;
    unsigned long long* Q;
    TransportCounters* counters;
};

// ---- Philox4x32-10, counter = (block, 0, g_lo, g_hi), key = seed ----
__device__ __forceinline__ void philox(uint32_t block, uint32_t g_lo, uint32_t g_hi, uint32_t k0, uint32_t k1,
                                       uint32_t& o0, uint32_t& o1, uint32_t& o2, uint32_t& o3)
{
    uint32_t c0 = block, c1 = 0u, c2 = g_lo, c3 = g_hi;
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const unsigned long long pa = (unsigned long long)0xD2511F53u * c0;
        const unsigned long long pb = (unsigned long long)0xCD9E8D57u * c2;
        const uint32_t n0 = (uint32_t)(pb >> 32) ^ c1 ^ k0;
        const uint32_t n2 = (uint32_t)(pa >> 32) ^ c3 ^ k1;
        c1 = (uint32_t)pb; c3 = (uint32_t)pa; c0 = n0; c2 = n2;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    o0 = c0; o1 = c1; o2 = c2; o3 = c3;
}

__device__ __forceinline__ float u01(uint32_t x) { return ((float)(x >> 9) + 0.5f) * kU01; }

// kinematics at kinetic energy E: a = beta^2 gamma^2 = tau (tau + 2), gam = gamma
struct Kin { float a, gam, inv_beta2, x; };
__device__ __forceinline__ Kin kinematics(float E)
{
    Kin k;
    const float tau = E * kInvMp;
    k.a   = tau * (tau + 2.0f);
    k.gam = 1.0f + tau;
    k.inv_beta2 = __fdividef(k.gam * k.gam, k.a);
    k.x   = 2.0f * kRatio * k.gam + kRatio * kRatio;                 // T_max = 2 me a / (1 + x)
    return k;
}

// Bethe mass stopping power of water [MeV cm2/g]:
//   K Z/A / beta2 [ 1/2 ln(2 me a Tmax / I^2) - beta2 ] with 1/2 ln(..) = ln(2 me a / I) - 1/2 ln(1 + x)
__device__ __forceinline__ float bethe(const Kin& k)
{
    const float l1  = __log2f(kLogArg * k.a) * kLn2;
    const float l2  = 0.5f * k.x * (1.0f - 0.5f * k.x);              // 1/2 ln(1+x), x ~ 1e-3
    const float b2  = __fdividef(1.0f, k.inv_beta2);
    return kKZA * k.inv_beta2 * (l1 - l2 - b2);
}

// CSDA range in water [g/cm2] from the shared-memory table (log2-log2 linear interpolation)
__device__ __forceinline__ float range_water(float E, const float* tab)
{
    float x = (__log2f(E) - kRangeLog2E0) * kRangeInvStep;
    x = fminf(fmaxf(x, 0.0f), (float)(kRangeNodes - 1) - 0.001f);
    const int   i = (int)x;
    const float f = x - (float)i;
    const float a = tab[i], b = tab[i + 1];
    return exp2f(a + f * (b - a));
}

}  // namespace

namespace {

// Per-lane history state.  Position p* is voxel-local: 0 <= p <= h on each axis.
struct Lane {
    float px, py, pz, dx, dy, dz, E, wq;      // wq = weight * 2^k (deposit -> quanta)
    double wq_d;
    int ix, iy, iz;
    uint32_t g_lo, g_hi, m;
    long long vox;                             // linear voxel index of the pending deposit
    long long pend;                            // quanta deposited in vox and not yet flushed
    float dens;
};

// T3: sample history j of the launch.  Returns false if the ray misses the grid (all energy escapes).
__device__ __forceinline__ bool start_history(const Params& P, long long j, Lane& L, long long& q_inc,
                                              long long& q_esc)
{
    // segment lookup: last segment with local_begin <= j
    int lo = 0, hi = P.n_segs - 1;
    while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (P.segs[mid].local_begin <= j) lo = mid; else hi = mid - 1;
    }
    const DevSegment& S = P.segs[lo];
    const unsigned long long g = (unsigned long long)(S.first_history + (j - S.local_begin));
    L.g_lo = (uint32_t)g; L.g_hi = (uint32_t)(g >> 32); L.m = 0u;
    L.wq = S.weight_scaled; L.wq_d = S.weight_scaled_d;

    uint32_t r0, r1, r2, r3;
    philox(0u, L.g_lo, L.g_hi, P.seed_lo, P.seed_hi, r0, r1, r2, r3);
    const float rad = sqrtf(-2.0f * logf(u01(r0)));
    float sn, cs;
    sincospif(2.0f * u01(r1), &sn, &cs);
    float gx = rad * cs, gy = rad * sn;
    float gE = sqrtf(-2.0f * logf(u01(r2))) * cospif(2.0f * u01(r3));
    if (P.flags & PBS4D_NO_SPOTSIZE) { gx = 0.0f; gy = 0.0f; }
    if (P.flags & PBS4D_NO_ESPREAD)  gE = 0.0f;
    L.E = S.energy_mev * (1.0f + 0.01f * gE);
    const float a = S.x_mm + S.sigma_mm * gx, b = S.y_mm + S.sigma_mm * gy;
    float r[3], d[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) { r[k] = S.ref[k] + a * S.eu[k] + b * S.ev[k]; d[k] = S.dir[k]; }
    const long long qi = __double2ll_rn((double)L.E * L.wq_d);
    q_inc += qi;

    // slab-method ray/box intersection over t in (-inf, inf)
    const float o[3] = { P.g.ox, P.g.oy, P.g.oz }, h[3] = { P.g.hx, P.g.hy, P.g.hz };
    const int   n[3] = { P.g.nx, P.g.ny, P.g.nz };
    float t_in = -INFINITY, t_out = INFINITY; int ax = -1; bool miss = false;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const float lo_k = o[k], hi_k = o[k] + (float)n[k] * h[k];
        if (d[k] == 0.0f) { if (r[k] < lo_k || r[k] >= hi_k) miss = true; continue; }
        float t1 = (lo_k - r[k]) / d[k], t2 = (hi_k - r[k]) / d[k];
        if (t1 > t2) { const float tt = t1; t1 = t2; t2 = tt; }
        if (t1 > t_in) { t_in = t1; ax = k; }
        if (t2 < t_out) t_out = t2;
    }
    if (miss || ax < 0 || !(t_in < t_out)) { q_esc += qi; return false; }
    int idx[3]; float pl[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const float rk = r[k] + t_in * d[k];
        int i = (int)floorf((rk - o[k]) / h[k]);
        i = max(0, min(i, n[k] - 1));
        idx[k] = i;
        pl[k] = fminf(fmaxf(rk - (o[k] + (float)i * h[k]), 0.0f), h[k]);
        if (k == ax) {
            if (d[k] > 0.0f) { idx[k] = 0;        pl[k] = 0.0f; }
            else             { idx[k] = n[k] - 1; pl[k] = h[k]; }
        }
    }
    L.px = pl[0]; L.py = pl[1]; L.pz = pl[2];
    L.dx = d[0];  L.dy = d[1];  L.dz = d[2];
    L.ix = idx[0]; L.iy = idx[1]; L.iz = idx[2];
    L.vox = ((long long)L.iz * P.g.ny + L.iy) * P.g.nx + L.ix;
    L.pend = 0;
    L.dens = __ldg(P.rho + L.vox);
    return true;
}

__device__ __forceinline__ void flush(const Params& P, Lane& L)
{
    if (L.pend != 0) {
        atomicAdd(P.Q + L.vox, (unsigned long long)L.pend);
        L.pend = 0;
    }
}

__global__ void __launch_bounds__(kThreads)
transport_kernel(const Params P)
{
    __shared__ float s_range[kRangeNodes];
    __shared__ long long s_tally[5];
    for (int i = threadIdx.x; i < kRangeNodes; i += kThreads) s_range[i] = P.range_tab[i];
    if (threadIdx.x < 5) s_tally[threadIdx.x] = 0;
    __syncthreads();

    const long long stride = (long long)gridDim.x * kThreads;
    long long next = (long long)blockIdx.x * kThreads + threadIdx.x;
    long long q_inc = 0, q_dep = 0, q_esc = 0;
    unsigned long long n_steps = 0, n_hist = 0;
    const float hx = P.g.hx, hy = P.g.hy, hz = P.g.hz;
    const int   nx = P.g.nx, ny = P.g.ny, nz = P.g.nz;
    const bool do_mcs = !(P.flags & PBS4D_NO_MCS), do_strag = !(P.flags & PBS4D_NO_STRAGGLE);

    Lane L;
    bool alive = false;
    for (;;) {
        if (!alive) {
            // refill this lane with its next history (T3); a lane with none left leaves the loop
            if (next >= P.n_hist) break;
            alive = start_history(P, next, L, q_inc, q_esc);
            next += stride;
            n_hist += 1;
            if (!alive) continue;
        }
        // ---------------- one condensed-history step (T5-T10) ----------------
        L.m += 1u;
        const float dens = L.dens;
        const Kin   k0 = kinematics(L.E);
        const float S0 = bethe(k0);
        const float R  = __fdividef(10.0f * range_water(L.E, s_range), dens);           // mm, local medium

        // T6: distance to the voxel faces (voxel-local coordinates)
        const float idx_ = __frcp_rn(L.dx), idy_ = __frcp_rn(L.dy), idz_ = __frcp_rn(L.dz);
        float sax = L.dx > 0.0f ? (hx - L.px) * idx_ : (L.dx < 0.0f ? -L.px * idx_ : INFINITY);
        float say = L.dy > 0.0f ? (hy - L.py) * idy_ : (L.dy < 0.0f ? -L.py * idy_ : INFINITY);
        float saz = L.dz > 0.0f ? (hz - L.pz) * idz_ : (L.dz < 0.0f ? -L.pz * idz_ : INFINITY);
        sax = fmaxf(sax, 0.0f); say = fmaxf(say, 0.0f); saz = fmaxf(saz, 0.0f);
        const float s_b   = fminf(sax, fminf(say, saz));
        const float s_lim = fminf(kSmax, kFrac * R);
        const bool  crossing = s_b <= s_lim * kTie;
        const float s = crossing ? s_b : s_lim;

        // T7: midpoint-rule mean loss
        const float t   = dens * s * 0.1f;                                               // g/cm2
        const float Em  = fmaxf(L.E - 0.5f * S0 * t, 1.0e-3f);
        const Kin   km  = kinematics(Em);
        const float dEm = bethe(km) * t;

        // T8: straggling (Philox block m)
        uint32_t r0, r1, r2, r3;
        philox(L.m, L.g_lo, L.g_hi, P.seed_lo, P.seed_hi, r0, r1, r2, r3);
        float dE = dEm;
        if (do_strag) {
            const float tmax = __fdividef(2.0f * kMe * km.a, 1.0f + km.x);
            const float b2   = __fdividef(1.0f, km.inv_beta2);
            const float var  = 0.5f * kKZA * km.inv_beta2 * tmax * (1.0f - 0.5f * b2) * t;
            const float gg   = sqrtf(-2.0f * logf(u01(r2))) * cospif(2.0f * u01(r3));
            dE = dEm + sqrtf(var) * gg;
        }
        dE = fminf(fmaxf(dE, 0.0f), L.E);
        if (L.E - dE <= kEcut) { dE = L.E; alive = false; }

        // T9/T11: score into the voxel the step lay in (register accumulation, flushed on voxel change)
        const long long q = __float2ll_rn(dE * L.wq);
        L.pend += q; q_dep += q; n_steps += 1;

        L.px += s * L.dx; L.py += s * L.dy; L.pz += s * L.dz;

        // T10: boundary-limited step -> snap every axis attaining the minimum onto its face
        bool moved = false;
        if (crossing) {
            if (sax == s_b) { if (L.dx > 0.0f) { L.ix += 1; L.px = 0.0f; } else { L.ix -= 1; L.px = hx; } moved = true; }
            if (say == s_b) { if (L.dy > 0.0f) { L.iy += 1; L.py = 0.0f; } else { L.iy -= 1; L.py = hy; } moved = true; }
            if (saz == s_b) { if (L.dz > 0.0f) { L.iz += 1; L.pz = 0.0f; } else { L.iz -= 1; L.pz = hz; } moved = true; }
        }

        // T9: Highland deflection at the end of the step (kinematics at Em), branch-free orthonormal basis
        if (do_mcs) {
            const float pv  = kMp * __fdividef(km.a, km.gam);
            const float th0 = __fdividef(kEs, pv) * sqrtf(t * kInvX0);
            const float th  = th0 * sqrtf(-2.0f * logf(u01(r0)));
            float sp, cp, st, ct;
            sincospif(2.0f * u01(r1), &sp, &cp);
            sincosf(th, &st, &ct);
            const float sw = copysignf(1.0f, L.dz);
            const float aa = -__frcp_rn(sw + L.dz);
            const float bb = L.dx * L.dy * aa;
            const float e1x = 1.0f + sw * L.dx * L.dx * aa, e1y = sw * bb, e1z = -sw * L.dx;
            const float e2x = bb, e2y = sw + L.dy * L.dy * aa, e2z = -L.dy;
            const float ux = cp * e1x + sp * e2x, uy = cp * e1y + sp * e2y, uz = cp * e1z + sp * e2z;
            const float nxd = ct * L.dx + st * ux, nyd = ct * L.dy + st * uy, nzd = ct * L.dz + st * uz;
            const float inv = rsqrtf(nxd * nxd + nyd * nyd + nzd * nzd);
            L.dx = nxd * inv; L.dy = nyd * inv; L.dz = nzd * inv;
        }
        L.E -= dE;

        if (!alive) { flush(P, L); continue; }
        if (moved) {
            flush(P, L);
            if ((unsigned)L.ix >= (unsigned)nx || (unsigned)L.iy >= (unsigned)ny || (unsigned)L.iz >= (unsigned)nz) {
                q_esc += __double2ll_rn((double)L.E * L.wq_d);                           // left the grid
                alive = false;
                continue;
            }
            L.vox  = ((long long)L.iz * ny + L.iy) * nx + L.ix;
            L.dens = __ldg(P.rho + L.vox);
        }
    }

    // block-level tally reduction: warp shuffle, shared atomics, one global atomic per block and counter
    long long v[5] = { (long long)n_hist, (long long)n_steps, q_inc, q_dep, q_esc };
#pragma unroll
    for (int c = 0; c < 5; ++c) {
        long long x = v[c];
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) x += __shfl_xor_sync(0xffffffffu, x, off);
        if ((threadIdx.x & 31) == 0) atomicAdd((unsigned long long*)&s_tally[c], (unsigned long long)x);
    }
    __syncthreads();
    if (threadIdx.x < 5) {
        unsigned long long* dst = threadIdx.x == 0 ? &P.counters->histories
                                : threadIdx.x == 1 ? &P.counters->steps
                                : threadIdx.x == 2 ? (unsigned long long*)&P.counters->q_incident
                                : threadIdx.x == 3 ? (unsigned long long*)&P.counters->q_deposited
                                                   : (unsigned long long*)&P.counters->q_escaped;
        atomicAdd(dst, (unsigned long long)s_tally[threadIdx.x]);
    }
}

}  // namespace

const void* transport_kernel_symbol() { return (const void*)transport_kernel; }

static float* g_range_tab_dev[16] = { nullptr };   // one table per device, built on first use

void launch_transport(const pbs4d_grid& g, const float* rho, const DevSegment* segs, int32_t n_segs,
                      int64_t n_hist, uint64_t seed, uint32_t flags, long long* Q, TransportCounters* counters,
                      int sm_count, cudaStream_t st)
{
    int dev = 0;
    cudaGetDevice(&dev);
    if (dev >= 0 && dev < 16 && !g_range_tab_dev[dev]) {
        float host_tab[kRangeNodes];
        build_range_table(host_tab);
        cudaMalloc(&g_range_tab_dev[dev], sizeof(host_tab));
        cudaMemcpy(g_range_tab_dev[dev], host_tab, sizeof(host_tab), cudaMemcpyHostToDevice);
    }
    Params P;
    P.g = g; P.rho = rho; P.segs = segs; P.range_tab = g_range_tab_dev[dev];
    P.n_segs = n_segs; P.n_hist = n_hist;
    P.seed_lo = (uint32_t)seed; P.seed_hi = (uint32_t)(seed >> 32); P.flags = flags;
    P.Q = (unsigned long long*)Q; P.counters = counters;
    int per_sm = 1;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, transport_kernel, kThreads, 0);
    if (per_sm < 1) per_sm = 1;
    long long want = (n_hist + kThreads - 1) / kThreads;
    long long cap  = (long long)sm_count * per_sm;
    int blocks = (int)(want < cap ? want : cap);
    if (blocks < 1) blocks = 1;
    transport_kernel<<<blocks, kThreads, 0, st>>>(P);
}

}  // namespace pbs4d
