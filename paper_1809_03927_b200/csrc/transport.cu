// History-parallel proton transport + dose scoring for sm_100a (Sec. 2.C names
// the engine -- "class II condensed-history proton transport" -- the model itself is BASELINE.json north_star +
// config 1: Philox-counter-seeded histories, step = min(voxel boundary, 1 mm, 2 % of residual range), Bethe-Bloch
// CSDA loss (midpoint rule), Bohr straggling, Highland deflection without log term, 0.5 MeV cutoff deposited
// locally, 64-bit fixed-point atomic scoring).
//
// Layout of the computation (B200-first, not the paper's Titan-X design).  The kernel is bound by instruction
// issue and by the XU (MUFU/conversion) pipe, never by HBM, so everything below is about instructions per step:
//  * persistent warps (4 CTAs x 256 threads per SM, 64 registers).  Every warp keeps a pool of 32 pre-sampled
//    histories in shared memory: when it is empty the whole warp takes 32 history indices from a global counter
//    (one atomicAdd) and samples them together, and a lane whose history ends pops the next entry.  The Philox
//    counter is (step, history), never the lane, so any lane/history assignment gives the same integers;
//  * the step loop is warp-uniform (refill phase, then one predicated, branch-free step for every live lane): the
//    warp reconverges every iteration;
//  * S(E), 2 % of the CSDA range, the Bohr variance and the Highland theta0^2 come from ONE float4 table in shared
//    memory, indexed by integer operations on the bit pattern of E (no logarithm), linear in E inside an interval;
//    the values at the midpoint energy are read off the same pair of nodes (one lookup per step);
//  * one reciprocal per step for the voxel-face distance (the nearest face is found by cross-multiplication),
//    1/density cached per voxel visit, Gaussian factors folded under one square root each, small-angle polynomial
//    for the polar deflection, uniform floats built with bit operations: 10 MUFU per step instead of ~27;
//  * Philox round keys are kernel parameters (constant bank operands);
//  * position is voxel-local (0 <= p <= h) so face distances keep full fp32 resolution;
//  * deposits are converted to int64 quanta of 2^-k MeV and summed in a register while the history stays in one
//    voxel; one red.global.add.u64 per voxel visit, resolved in the L2.
#include "internal.h"
#include "physics_tables.h"

#include <cuda_runtime.h>

namespace pbs4d {

namespace {

constexpr int   kThreads   = 256;
constexpr int   kWarps     = kThreads / 32;
constexpr int   kPoolWords = 10;                                     // words per pre-sampled history in the warp's pool
constexpr float kEcut      = 0.5f;
constexpr float kSmax      = 1.0f;
constexpr float kTie       = 1.0f + 1.0f / 1024.0f;                  // boundary/step-limit tie tolerance (DESIGN A22)
constexpr float kTwoPi     = 6.283185307179586f;
constexpr float kPi        = 3.14159265358979f;
constexpr float kNeg2Ln2   = -1.3862943611198906f;                  // -2 ln 2
constexpr float kTinyDir   = 1.0e-20f;                              // stands in for an exactly-zero direction component

struct Params {
    pbs4d_grid g;
    const float* __restrict__ rho;
    const DevSegment* __restrict__ segs;
    const long long* __restrict__ seg_begin;  // [n_segs] local index of each segment's first history (ascending)
    const float4* __restrict__ tab;           // kTabNodes physics nodes
    int32_t n_segs;
    long long hist_begin, n_hist;             // this launch transports local histories hist_begin .. hist_begin + n_hist - 1
    uint32_t flags;
    uint32_t max_steps;                       // hang guard: a history that reaches this many steps is absorbed where it is
    uint32_t k0[10], k1[10];                  // Philox round keys
    unsigned long long* Q;
    TransportCounters* counters;
};

// ---- Philox4x32-10, counter = (block, 0, g_lo, g_hi) ----
__device__ __forceinline__ void philox(const Params& P, uint32_t block, uint32_t g_lo, uint32_t g_hi,
                                       uint32_t& o0, uint32_t& o1, uint32_t& o2, uint32_t& o3)
{
    uint32_t c0 = block, c1 = 0u, c2 = g_lo, c3 = g_hi;
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t h0 = __umulhi(0xD2511F53u, c0), l0 = 0xD2511F53u * c0;
        const uint32_t h1 = __umulhi(0xCD9E8D57u, c2), l1 = 0xCD9E8D57u * c2;
        c0 = h1 ^ c1 ^ P.k0[r];
        c2 = h0 ^ c3 ^ P.k1[r];
        c1 = l1; c3 = l0;
    }
    o0 = c0; o1 = c1; o2 = c2; o3 = c3;
}

// u = ((x >> 9) + 0.5) 2^-23, built without an integer->float conversion: (1 + m 2^-23) - (1 - 2^-24).  The
// subtrahend 0x3F7FFFFF is a float and the difference (2 m + 1) 2^-24 has 24 significant bits: one exact FADD.
constexpr float kOneMinusEps = 0.99999994039535522461f;             // 1 - 2^-24
__device__ __forceinline__ float u01(uint32_t x)
{
    return __uint_as_float(0x3F800000u | (x >> 9)) - kOneMinusEps;
}
__device__ __forceinline__ float unit_float(uint32_t x) { return __uint_as_float(0x3F800000u | (x >> 9)); }   // in [1, 2)

__device__ __forceinline__ float fast_sqrt(float x)
{
    float y;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float fast_log2(float x)       // x >= 2^-24 here: no denormal pre-scaling needed
{
    float y;
    asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float fast_rcp(float x)
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// cos(2 pi u), sin(2 pi u) for u in (0,1): the MUFU argument is moved to (-pi, pi), where sin/cos.approx are
// accurate to ~2^-21 absolute; cos(x + pi) = -cos x
__device__ __forceinline__ void sincos_2pi(float u, float& s, float& c)
{
    const float a = fmaf(u, kTwoPi, -kPi);
    s = -__sinf(a); c = -__cosf(a);
}

// the same angle 2 pi u - pi straight from the random word x, u = ((x >> 9) + 0.5) 2^-23: with f = 1 + (x >> 9) 2^-23
// (built by bit operations) it is 2 pi f - 3 pi + pi 2^-23, one FMA
__device__ __forceinline__ float angle_from_word(uint32_t x)
{
    return fmaf(__uint_as_float(0x3F800000u | (x >> 9)), kTwoPi, -9.42477758f);      // -3 pi + pi 2^-23
}

// table interval and fraction of an energy (integer operations on the bit pattern; see physics_tables.h)
struct Lookup { int i; float f, inv_w; };
__device__ __forceinline__ Lookup locate(float E)
{
    const uint32_t b = __float_as_uint(E);
    Lookup L;
    L.i = min(max((int)(b >> 16) - (int)(kTabBits0 >> 16), 0), kTabNodes - 2);
    const float e_node = __uint_as_float(b & 0xFFFF0000u);
    const float inv_w  = __uint_as_float(0x82800000u - (b & 0x7F800000u));          // 2^(7 - exponent)
    L.f = (E - e_node) * inv_w;
    L.inv_w = inv_w;
    return L;
}

// ---- packed fp32 pairs (sm_100 f32x2: one issue slot for two operations; each half rounds as the scalar op) ----
// The kernel is bound by instruction issue, so the (x, y) halves of position and direction and the pairs of table
// columns that are interpolated together go through FFMA2 / FMUL2 / FADD2.
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk(float lo, float hi)
{
    f32x2 d; asm("mov.b64 %0, {%1, %2};" : "=l"(d) : "f"(lo), "f"(hi)); return d;
}
__device__ __forceinline__ void upk(f32x2 v, float& lo, float& hi)
{
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
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

// one table node from shared memory at a 32-bit shared address (the compiler otherwise rebuilds the generic address of
// the table -- S2R SR_CgaCtaId, MOV, LEA -- in every iteration of the step loop)
__device__ __forceinline__ float4 lds_node(unsigned addr)
{
    float4 v;
    asm("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
    return v;
}

// Per-lane history state.  Position p* is voxel-local: 0 <= p <= h on each axis.
struct Lane {
    float px, py, pz, dx, dy, dz, E, wq;      // wq = weight * 2^k (deposit -> quanta)
    int ix, iy, iz;
    uint32_t g_lo, g_hi, m;
    int vox;                                   // linear voxel index of the pending deposit (< 2^31 voxels)
    long long pend;                            // quanta deposited in vox and not yet flushed
    float rho;                                 // density of the current voxel; 0.1 rho and 1 / rho are formed at the top
                                               // of every step, a table lookup away from the load that produced rho
    int seg;                                   // index of the history's segment in the launch table
};

// T3: sample history j of the launch.  Returns false if the ray misses the grid (all energy escapes).
__device__ __noinline__ bool start_history(const Params& P, long long j, Lane& L, long long& q_inc, long long& q_esc)
{
    // segment lookup: last segment with seg_begin <= j
    int lo = 0, hi = P.n_segs - 1;
    while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (__ldg(P.seg_begin + mid) <= j) lo = mid; else hi = mid - 1;
    }
    const DevSegment& S = P.segs[lo];
    L.seg = lo;
    const unsigned long long g = (unsigned long long)(S.first_history + (j - S.local_begin));
    L.g_lo = (uint32_t)g; L.g_hi = (uint32_t)(g >> 32); L.m = 0u;
    L.wq = S.weight_scaled;

    uint32_t r0, r1, r2, r3;
    philox(P, 0u, L.g_lo, L.g_hi, r0, r1, r2, r3);
    const float rad = fast_sqrt(kNeg2Ln2 * fast_log2(u01(r0)));
    float sn, cs, snE, csE;
    sincos_2pi(u01(r1), sn, cs);
    sincos_2pi(u01(r3), snE, csE);
    float gx = rad * cs, gy = rad * sn;
    float gE = fast_sqrt(kNeg2Ln2 * fast_log2(u01(r2))) * csE;
    if (P.flags & PBS4D_NO_SPOTSIZE) { gx = 0.0f; gy = 0.0f; }
    if (P.flags & PBS4D_NO_ESPREAD)  gE = 0.0f;
    L.E = S.energy_mev * (1.0f + 0.01f * gE);
    const float a = S.x_mm + S.sigma_mm * gx, b = S.y_mm + S.sigma_mm * gy;
    float r[3], d[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) { r[k] = S.ref[k] + a * S.eu[k] + b * S.ev[k]; d[k] = S.dir[k]; }
    const long long qi = __double2ll_rn((double)L.E * S.weight_scaled_d);
    q_inc += qi;

    // slab-method ray/box intersection over t in (-inf, inf)
    const float o[3] = { P.g.ox, P.g.oy, P.g.oz }, h[3] = { P.g.hx, P.g.hy, P.g.hz };
    const int   n[3] = { P.g.nx, P.g.ny, P.g.nz };
    float t_in = -INFINITY, t_out = INFINITY; int ax = -1; bool miss = false;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const float lo_k = o[k], hi_k = o[k] + (float)n[k] * h[k];
        if (d[k] == 0.0f) { if (r[k] < lo_k || r[k] >= hi_k) miss = true; continue; }
        const float inv_d = fast_rcp(d[k]);
        float t1 = (lo_k - r[k]) * inv_d, t2 = (hi_k - r[k]) * inv_d;
        if (t1 > t2) { const float tt = t1; t1 = t2; t2 = tt; }
        if (t1 > t_in) { t_in = t1; ax = k; }
        if (t2 < t_out) t_out = t2;
    }
    if (miss || ax < 0 || !(t_in < t_out)) { q_esc += qi; return false; }
    int idx[3]; float pl[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const float rk = r[k] + t_in * d[k];
        int i = (int)floorf(__fdividef(rk - o[k], h[k]));
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
    L.vox = (L.iz * P.g.ny + L.iy) * P.g.nx + L.ix;
    L.pend = 0;
    return true;
}

__device__ __forceinline__ void flush(const Params& P, Lane& L, long long& q_dep, uint32_t& n_red)
{
    n_red += 1u;
    atomicAdd(P.Q + L.vox, (unsigned long long)L.pend);
    q_dep += L.pend;
    L.pend = 0;
}

// kMcs / kStrag: Highland deflection / Bohr straggling compiled in (the production kernel has both; the other three
// instantiations serve the test switches PBS4D_NO_MCS / PBS4D_NO_STRAGGLE without flag tests in the step loop)
template <bool kMcs, bool kStrag>
__global__ void __launch_bounds__(kThreads, 4)
transport_kernel(const __grid_constant__ Params P)
{
    __shared__ float4 s_tab[kTabNodes];
    __shared__ long long s_tally[7];                    // [6]: histories stopped by the step cap
    __shared__ uint32_t s_pool[kWarps][kPoolWords][32];
    for (int i = threadIdx.x; i < kTabNodes; i += kThreads) s_tab[i] = P.tab[i];
    unsigned tab_addr;                                  // laundered through asm: kept in a register, not rebuilt per step
    asm volatile("mov.u32 %0, %1;" : "=r"(tab_addr) : "r"((unsigned)__cvta_generic_to_shared(s_tab)));
    if (threadIdx.x < 7) s_tally[threadIdx.x] = 0;
    __syncthreads();

    const unsigned lane = threadIdx.x & 31u;
    long long q_dep = 0;                                // rare tallies (incident, escaped, histories) go straight to
    uint32_t n_red = 0;                                 // shared memory; per-step ones stay in registers
    // two per-thread values that are touched once per history live in shared memory, not in registers (the step loop sits
    // at its register budget: one state register less was worth 1.4 %): the step count and the history's segment
    __shared__ uint32_t s_nsteps[kThreads];
    __shared__ int s_seg[kThreads];
    s_nsteps[threadIdx.x] = 0u;
    const float hx = P.g.hx, hy = P.g.hy, hz = P.g.hz;
    const int   nx = P.g.nx, ny = P.g.ny, nz = P.g.nz;

    // Per-warp pool of 32 pre-sampled histories (T3 done by the whole warp at once, at full lane efficiency); a lane
    // whose history ends pops the next one instead of sampling it alone while 31 lanes wait.
    uint32_t (*pool)[32] = s_pool[threadIdx.x >> 5];
    int  avail = 0;                                     // warp-uniform: unconsumed pool entries (32-avail .. 31)
    bool drained = false;                               // warp-uniform: the launch has no histories left to fetch

    Lane L;
    bool alive = false, exhausted = false;
    for (;;) {
        // ---------------- refill phase: dead lanes pop pre-sampled histories ----------------
        const bool dead = !alive && !exhausted;
        const unsigned need = __ballot_sync(0xffffffffu, dead);
        if (need) {
            if (avail == 0 && !drained) {
                unsigned long long base = 0;
                if (lane == 0) base = atomicAdd(&P.counters->next_history, 32ull);
                base = __shfl_sync(0xffffffffu, base, 0);
                const long long j = (long long)base + lane;
                int tag = -1;                           // -1: no such history, -2: the ray misses the grid
                if (j < P.n_hist) {
                    Lane T;
                    long long qi = 0, qe = 0;
                    const bool ok = start_history(P, P.hist_begin + j, T, qi, qe);
                    atomicAdd((unsigned long long*)&s_tally[0], 1ull);
                    atomicAdd((unsigned long long*)&s_tally[2], (unsigned long long)qi);
                    if (qe) atomicAdd((unsigned long long*)&s_tally[4], (unsigned long long)qe);
                    tag = ok ? T.seg : -2;
                    pool[0][lane] = __float_as_uint(T.px); pool[1][lane] = __float_as_uint(T.py);
                    pool[2][lane] = __float_as_uint(T.pz); pool[3][lane] = __float_as_uint(T.E);
                    pool[4][lane] = (uint32_t)T.ix; pool[5][lane] = (uint32_t)T.iy; pool[6][lane] = (uint32_t)T.iz;
                    pool[7][lane] = T.g_lo; pool[8][lane] = T.g_hi;
                }
                pool[9][lane] = (uint32_t)tag;
                drained = (long long)base + 32 >= P.n_hist;
                avail = 32;
                __syncwarp();
            }
            if (avail > 0) {
                const int rank = __popc(need & ((1u << lane) - 1u));
                if (dead && rank < avail) {
                    const int sl = 32 - avail + rank;
                    const int tag = (int)pool[9][sl];
                    if (tag == -1) exhausted = true;
                    else if (tag >= 0) {
                        const DevSegment& S = P.segs[tag];
                        L.px = __uint_as_float(pool[0][sl]); L.py = __uint_as_float(pool[1][sl]);
                        L.pz = __uint_as_float(pool[2][sl]); L.E  = __uint_as_float(pool[3][sl]);
                        L.ix = (int)pool[4][sl]; L.iy = (int)pool[5][sl]; L.iz = (int)pool[6][sl];
                        L.g_lo = pool[7][sl]; L.g_hi = pool[8][sl]; L.m = 0u;
                        L.dx = S.dir[0] == 0.0f ? kTinyDir : S.dir[0];
                        L.dy = S.dir[1] == 0.0f ? kTinyDir : S.dir[1];
                        L.dz = S.dir[2] == 0.0f ? kTinyDir : S.dir[2];
                        L.wq = S.weight_scaled; s_seg[threadIdx.x] = tag;
                        L.vox = (L.iz * ny + L.iy) * nx + L.ix;
                        L.pend = 0;
                        L.rho = __ldg(P.rho + L.vox);
                        alive = true;
                    }
                }
                avail = max(avail - __popc(need), 0);
                __syncwarp();
            } else if (dead) {
                exhausted = true;                       // pool empty and nothing left to fetch
            }
        }
        const unsigned live = __ballot_sync(0xffffffffu, alive);
        if (live == 0u) {
            if (__all_sync(0xffffffffu, exhausted)) break;
            continue;
        }
        // step loop: one vote per iteration; it is left as soon as a lane's history ends (back to the refill phase)
        do {
        if (alive) {
            // ---------------- one condensed-history step (T5-T10) ----------------
            L.m += 1u;
            const Lookup k0 = locate(L.E);
            const float4 A0 = lds_node(tab_addr + (unsigned)k0.i * 16u), B0 = lds_node(tab_addr + (unsigned)k0.i * 16u + 16u);
            float rs, S0;                                                     // 0.2 R_w(E), S(E): one packed interpolation
            {
                const f32x2 a = pk(A0.x, A0.y);
                upk(fma2(pk(k0.f, k0.f), sub2(pk(B0.x, B0.y), a), a), rs, S0);
            }
            // the density was loaded when the history entered the voxel (end of the previous iteration): its reciprocal
            // is taken here, after the table lookup, so that the load's latency hides behind the lookup instead of
            // stalling the warp in the voxel-change block
            const float dens = 0.1f * L.rho;                                  // t [g/cm2] = dens x s [mm]
            const float s_lim = fminf(kSmax, rs * fast_rcp(L.rho));

            // T6: nearest voxel face.  Per axis: numerator = distance to the face ahead, denominator = |d|;
            // the smallest quotient is found by cross-multiplication, then one reciprocal.
            // (direction components are never exactly zero: a zero component of the field direction is replaced by
            // +1e-20 when the history starts, which keeps that axis' quotient astronomically large, as 1/0 would)
            const float denx = fabsf(L.dx), deny = fabsf(L.dy), denz = fabsf(L.dz);
            float hpx, hpy;
            upk(sub2(pk(hx, hy), pk(L.px, L.py)), hpx, hpy);
            const float numx = fmaxf(L.dx > 0.0f ? hpx : L.px, 0.0f);
            const float numy = fmaxf(L.dy > 0.0f ? hpy : L.py, 0.0f);
            const float numz = fmaxf(L.dz > 0.0f ? hz - L.pz : L.pz, 0.0f);
            // x against z, then y against the winner; equal cross products mark axes that attain the minimum together
            const float cxz = numx * denz, czx = numz * denx;
            const bool  x_lt = cxz < czx;
            float num = x_lt ? numx : numz, den = x_lt ? denx : denz;
            bool  mx = cxz <= czx, mz = !x_lt;
            const float cy = numy * den, cw = num * deny;
            const bool  y_lt = cy < cw;
            num = y_lt ? numy : num; den = y_lt ? deny : den;
            bool  my = cy <= cw;
            mx = mx && !y_lt; mz = mz && !y_lt;
            const float s_b = num * fast_rcp(den);
            const bool  crossing = s_b <= s_lim * kTie;
            const float s = crossing ? s_b : s_lim;

            // T7: midpoint-rule mean loss
            const float t   = dens * s;                                       // g/cm2 (dens = 0.1 rho)
            // E_m = E - S(E) t / 2 lies at most about one and a half table intervals below E, in ANY medium: the step
            // is at most 2 % of the range at the voxel's density, so t <= 0.02 R_w(E) [g/cm2] whatever rho is, and with
            // S R_w ~ E / p (p ~ 1.77) the half-step loss is <= 0.01 E / p ~ 0.6 % of E, an interval being 0.4-0.8 % of
            // E.  S, V, T at E_m are therefore read off the SAME pair of nodes, extrapolating linearly below the
            // interval (error <= p(p-1)/2 (dE/E)^2 ~ 4e-5).  (Until round 3 a second lookup stood here for losses of
            // more than 4 intervals; the bound shows it could not be reached, and no test ever took it.)
            const float half = fminf(0.5f * S0 * t, L.E - 0.25f);
            const float  fm = fmaf(-half, k0.inv_w, k0.f);
            const float4 Am = A0, Bm = B0;
            const float Sm  = fmaf(fm, Bm.y - Am.y, Am.y);
            const float dEm = Sm * t;

            // T8: straggling (Philox block m): sigma g = sqrt(V t (-2 ln u2)) cos(2 pi u3)
            uint32_t r0, r1, r2, r3;
            philox(P, L.m, L.g_lo, L.g_hi, r0, r1, r2, r3);
            // Bohr variance and theta0^2 at E_m (one packed interpolation), both uniforms of the Gaussian magnitudes
            // (one packed subtraction), and the two products -V t lg u2, -T t lg u0 (two packed multiplications)
            float varg, th2;
            {
                const f32x2 a  = pk(Am.z, Am.w);
                const f32x2 vt = fma2(pk(fm, fm), sub2(pk(Bm.z, Bm.w), a), a);                       // (V, T)
                float u2, u0;
                upk(sub2(pk(unit_float(r2), unit_float(r0)), pk(kOneMinusEps, kOneMinusEps)), u2, u0);
                upk(mul2(mul2(vt, pk(-t, -t)), pk(fast_log2(u2), fast_log2(u0))), varg, th2);
            }
            float dE = dEm;
            if (kStrag) {
                const float a3 = angle_from_word(r3);
                dE = fmaf(fast_sqrt(varg), -__cosf(a3), dEm);
            }
            dE = fminf(fmaxf(dE, 0.0f), L.E);
            // below the cutoff the rest is deposited on the spot (T10).  The same exit serves as the hang guard of this
            // persistent kernel: a history that has taken P.max_steps steps (2^20; a 250 MeV proton in air-filled
            // lung needs a few thousand) is absorbed where it stands and counted in `aborted` -- never expected with
            // inputs that passed validation, but a history that cannot end would otherwise hold the GPU for ever
            if (L.E - dE <= kEcut || L.m >= P.max_steps) { dE = L.E; alive = false; }

            // T9/T11: score into the voxel the step lay in (register accumulation, flushed on voxel change)
            L.pend += __float2ll_rn(dE * L.wq);

            upk(fma2(pk(s, s), pk(L.dx, L.dy), pk(L.px, L.py)), L.px, L.py);
            L.pz = fmaf(s, L.dz, L.pz);

            // T10: boundary-limited step -> snap every axis attaining the minimum onto its face (branch-free)
            mx = mx && crossing; my = my && crossing; mz = mz && crossing;
            {
                const bool fx = L.dx > 0.0f, fy = L.dy > 0.0f, fz = L.dz > 0.0f;
                L.ix += mx ? (fx ? 1 : -1) : 0; L.px = mx ? (fx ? 0.0f : hx) : L.px;
                L.iy += my ? (fy ? 1 : -1) : 0; L.py = my ? (fy ? 0.0f : hy) : L.py;
                L.iz += mz ? (fz ? 1 : -1) : 0; L.pz = mz ? (fz ? 0.0f : hz) : L.pz;
            }
            // T9: Highland deflection at the end of the step (kinematics at Em), branch-free orthonormal basis;
            // theta^2 = T t (-2 ln u0); sin and cos of the (small) polar angle by their Taylor polynomials
            if (kMcs) {
                const float th  = fast_sqrt(th2);
                // sin(th) / th = 1 + th2 (-1/6 + th2 / 120) and cos(th) = 1 + th2 (-1/2 + th2 (1/24 - th2 / 720)): the two
                // Horner chains advance together, two packed fmas
                float ps, pc;
                {
                    const f32x2 t2 = pk(th2, th2);
                    const f32x2 h1 = fma2(t2, pk(1.0f / 120.0f, -1.0f / 720.0f), pk(-1.0f / 6.0f, 1.0f / 24.0f));
                    upk(fma2(t2, h1, pk(1.0f, -0.5f)), ps, pc);
                }
                const float st  = th * ps;
                const float ct  = fmaf(th2, pc, 1.0f);
                float sp, cp;
                const float a1 = angle_from_word(r1);
                sp = -__sinf(a1); cp = -__cosf(a1);
                const float sw = copysignf(1.0f, L.dz);
                const float aa = -fast_rcp(sw + L.dz);
                const float bb = L.dx * L.dy * aa;
                float dxa, dya;
                upk(mul2(pk(L.dx, L.dy), pk(aa, aa)), dxa, dya);
                const float e1x = fmaf(sw * L.dx, dxa, 1.0f), e1y = sw * bb, e1z = -sw * L.dx;
                const float e2x = bb, e2y = fmaf(L.dy, dya, sw), e2z = -L.dy;
                const f32x2 uxy = fma2(pk(cp, cp), pk(e1x, e1y), mul2(pk(sp, sp), pk(e2x, e2y)));
                const float uz  = fmaf(cp, e1z, sp * e2z);
                const f32x2 nxy = fma2(pk(ct, ct), pk(L.dx, L.dy), mul2(pk(st, st), uxy));
                const float nzd = fmaf(ct, L.dz, st * uz);
                float nxd, nyd;
                upk(nxy, nxd, nyd);
                const float n2  = fmaf(nxd, nxd, fmaf(nyd, nyd, nzd * nzd));
                const float inv = fmaf(-0.5f, n2, 1.5f);                      // 1/sqrt(n2) to first order, n2 = 1 + O(1e-6)
                upk(mul2(nxy, pk(inv, inv)), L.dx, L.dy); L.dz = nzd * inv;
            }
            L.E -= dE;

            if (crossing || !alive) {
                flush(P, L, q_dep, n_red);
                if (!alive) {
                    s_nsteps[threadIdx.x] += L.m;                             // history absorbed: L.m = its step count
                    if (L.m >= P.max_steps) atomicAdd((unsigned long long*)&s_tally[6], 1ull);
                }
                if (alive) {
                    if ((unsigned)L.ix >= (unsigned)nx || (unsigned)L.iy >= (unsigned)ny || (unsigned)L.iz >= (unsigned)nz) {
                        atomicAdd((unsigned long long*)&s_tally[4],                            // left the grid
                                  (unsigned long long)__double2ll_rn((double)L.E * P.segs[s_seg[threadIdx.x]].weight_scaled_d));
                        alive = false;
                        s_nsteps[threadIdx.x] += L.m;
                    } else {
                        L.vox = (L.iz * ny + L.iy) * nx + L.ix;
                        L.rho = __ldg(P.rho + L.vox);
                    }
                }
            }
        }
        } while (__ballot_sync(0xffffffffu, alive) == live);
    }

    // block-level tally reduction: warp shuffle, shared atomics, one global atomic per block and counter
    long long v[6] = { 0, (long long)s_nsteps[threadIdx.x], 0, q_dep, 0, (long long)n_red };
#pragma unroll
    for (int c = 0; c < 6; ++c) {
        long long x = v[c];
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) x += __shfl_xor_sync(0xffffffffu, x, off);
        if (lane == 0) atomicAdd((unsigned long long*)&s_tally[c], (unsigned long long)x);
    }
    __syncthreads();
    if (threadIdx.x == 6 && s_tally[6]) atomicAdd(&P.counters->aborted, (unsigned long long)s_tally[6]);
    if (threadIdx.x < 6) {
        unsigned long long* dst = threadIdx.x == 5 ? &P.counters->reds
                                : threadIdx.x == 0 ? &P.counters->histories
                                : threadIdx.x == 1 ? &P.counters->steps
                                : threadIdx.x == 2 ? (unsigned long long*)&P.counters->q_incident
                                : threadIdx.x == 3 ? (unsigned long long*)&P.counters->q_deposited
                                                   : (unsigned long long*)&P.counters->q_escaped;
        atomicAdd(dst, (unsigned long long)s_tally[threadIdx.x]);
    }
}

}  // namespace

const void* transport_kernel_symbol() { return (const void*)transport_kernel<true, true>; }

cudaError_t configure_transport(void)
{
    // 22.5 KB table + 10 KB history pools per CTA: ask for a shared-memory carve-out that keeps 4 CTAs resident.
    // A per-device attribute: pbs4d_create calls this once for every context (any device).
    cudaError_t e = cudaFuncSetAttribute(transport_kernel<true, true>, cudaFuncAttributePreferredSharedMemoryCarveout, 75);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(transport_kernel<true, false>, cudaFuncAttributePreferredSharedMemoryCarveout, 75);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(transport_kernel<false, true>, cudaFuncAttributePreferredSharedMemoryCarveout, 75);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(transport_kernel<false, false>, cudaFuncAttributePreferredSharedMemoryCarveout, 75);
    return e;
}

size_t physics_table_bytes(void) { return sizeof(TabNode) * kTabNodes; }

void launch_transport(const pbs4d_grid& g, const float* rho, const DevSegment* segs, const long long* seg_begin,
                      int32_t n_segs, int64_t hist_begin, int64_t n_hist, uint64_t seed, uint32_t flags,
                      const void* phys_tab_dev, long long* Q, TransportCounters* counters, int sm_count, cudaStream_t st)
{
    Params P;
    P.g = g; P.rho = rho; P.segs = segs; P.seg_begin = seg_begin; P.tab = static_cast<const float4*>(phys_tab_dev);
    P.n_segs = n_segs; P.hist_begin = hist_begin; P.n_hist = n_hist; P.flags = flags;
    P.max_steps = (flags & PBS4D_TEST_STEP_CAP_64) ? 64u : (1u << 20);
    uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
    for (int r = 0; r < 10; ++r) { P.k0[r] = k0; P.k1[r] = k1; k0 += 0x9E3779B9u; k1 += 0xBB67AE85u; }
    P.Q = (unsigned long long*)Q; P.counters = counters;
    const bool mcs = !(flags & PBS4D_NO_MCS), strag = !(flags & PBS4D_NO_STRAGGLE);
    void (*kernel)(const Params) = mcs ? (strag ? transport_kernel<true, true> : transport_kernel<true, false>)
                                       : (strag ? transport_kernel<false, true> : transport_kernel<false, false>);
    int per_sm = 1;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, kThreads, 0);
    if (per_sm < 1) per_sm = 1;
    long long want = (n_hist + kThreads - 1) / kThreads;
    long long cap  = (long long)sm_count * per_sm;
    int blocks = (int)(want < cap ? want : cap);
    if (blocks < 1) blocks = 1;
    kernel<<<blocks, kThreads, 0, st>>>(P);
}

}  // namespace pbs4d
