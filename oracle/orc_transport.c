/* oracle/orc_transport.c -- CPU ORACLE (test infrastructure only; see orc.h).
 * Per-history condensed-history proton transport, double precision.
 * Model: BASELINE.json north_star + config 1 (step = min(voxel boundary, 1 mm, 2 % of residual range),
 * Bethe CSDA loss, Bohr straggling, Highland deflection, 0.5 MeV cutoff deposited locally, no nuclear
 * interactions).  PAPER.md:69-71 (Sec. 2.C) names the engine but gives no physics.
 * Readings: A5 midpoint loss, A6 range to rest in local medium, A8 no log term, A9 deflection at
 * end of step, A12 residual into the voxel of the last step, A22 boundary/step-limit tie tolerance 2^-10. */
#include "orc.h"
#include <math.h>
#include <string.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

static const double E_CUT_ = 0.5;
static const double S_MAX_ = 1.0;          /* mm */
static const double F_RNG_ = 0.02;         /* 2 % of residual range */
static const double TIE_   = 1.0 / 1024.0; /* reading A22 */
static const double TWO_PI = 6.283185307179586476925286766559;

/* T2: u = ((x >> 9) + 0.5) 2^-23 in (0,1) */
static double u01(uint32_t x) { return ((double)(x >> 9) + 0.5) * (1.0 / 8388608.0); }

static void philox_block(uint64_t seed, uint64_t g, uint32_t block, double u[4])
{
    uint32_t ctr[4] = { block, 0u, (uint32_t)g, (uint32_t)(g >> 32) };
    uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    uint32_t o[4];
    orc_philox4x32_10(ctr, key, o);
    for (int i = 0; i < 4; ++i) u[i] = u01(o[i]);
}

int32_t orc_fixed_shift(int64_t n_segs, const orc_segment* segs, const orc_spot* spots)
{
    double tot = 0.0;
    for (int64_t s = 0; s < n_segs; ++s)
        tot += (double)segs[s].protons * (double)spots[segs[s].spot].energy_mev;
    tot *= 1.1;
    if (!(tot > 0.0)) return 40;
    int32_t k = (int32_t)floor(log2(4611686018427387904.0 / tot));
    if (k > 40) k = 40;                    /* LSB never below 2^-40 MeV */
    return k;
}

typedef struct { int64_t inc, dep, esc; uint64_t steps; } tally;

static void one_history(const orc_grid* G, const float* rho, const orc_field* F, const orc_spot* sp,
                        double w, uint64_t seed, uint64_t g, double scale, uint32_t flags,
                        int64_t* Q, tally* T, int n_probe, const int32_t* probe_faces,
                        double* probe_xy, int64_t H, int64_t gl, double* stop_xyz)
{
    const double h[3] = { G->hx, G->hy, G->hz }, o[3] = { G->ox, G->oy, G->oz };
    const int    n[3] = { G->nx, G->ny, G->nz };
    double u[4];

    /* ---- T3: source, Philox block 0 ---- */
    philox_block(seed, g, 0u, u);
    double rr = sqrt(-2.0 * log(u[0]));
    double gx = rr * cos(TWO_PI * u[1]), gy = rr * sin(TWO_PI * u[1]);
    double gE = sqrt(-2.0 * log(u[2])) * cos(TWO_PI * u[3]);
    if (flags & ORC_NO_SPOTSIZE) { gx = 0.0; gy = 0.0; }
    if (flags & ORC_NO_ESPREAD)  gE = 0.0;
    double E = (double)sp->energy_mev * (1.0 + 0.01 * gE);
    double a = (double)sp->x_mm + (double)sp->sigma_mm * gx;
    double b = (double)sp->y_mm + (double)sp->sigma_mm * gy;
    double r[3], d[3];
    for (int k = 0; k < 3; ++k) {
        r[k] = (double)F->ref[k] + a * (double)F->eu[k] + b * (double)F->ev[k];
        d[k] = (double)F->dir[k];
    }
    int64_t q_inc = llrint(E * w * scale);
    T->inc += q_inc;

    /* slab-method ray/box intersection over t in (-inf, inf) */
    double t_in = -INFINITY, t_out = INFINITY; int ax_in = -1, miss = 0;
    for (int k = 0; k < 3; ++k) {
        double lo = o[k], hi = o[k] + n[k] * h[k];
        if (d[k] == 0.0) { if (r[k] < lo || r[k] >= hi) miss = 1; continue; }
        double t1 = (lo - r[k]) / d[k], t2 = (hi - r[k]) / d[k];
        if (t1 > t2) { double tt = t1; t1 = t2; t2 = tt; }
        if (t1 > t_in) { t_in = t1; ax_in = k; }
        if (t2 < t_out) t_out = t2;
    }
    if (miss || ax_in < 0 || !(t_in < t_out)) { T->esc += q_inc; if (stop_xyz) stop_xyz[gl*3] = stop_xyz[gl*3+1] = stop_xyz[gl*3+2] = NAN; return; }
    int idx[3];
    for (int k = 0; k < 3; ++k) {
        r[k] += t_in * d[k];
        int i = (int)floor((r[k] - o[k]) / h[k]);
        if (i < 0) i = 0;
        if (i > n[k] - 1) i = n[k] - 1;
        idx[k] = i;
    }
    if (d[ax_in] > 0.0) { idx[ax_in] = 0;            r[ax_in] = o[ax_in]; }
    else                { idx[ax_in] = n[ax_in] - 1; r[ax_in] = o[ax_in] + n[ax_in] * h[ax_in]; }

    /* ---- T4: step loop ---- */
    int alive = 1;
    for (uint32_t m = 1; alive; ++m) {
        size_t vox = ((size_t)idx[2] * n[1] + idx[1]) * n[0] + idx[0];
        double dens = (double)rho[vox];

        /* T5: residual range in the local medium, mm */
        double R = 10.0 * orc_range_water(E) / dens;

        /* T6: distance to the voxel boundary per axis */
        double sa[3], s_b = INFINITY;
        for (int k = 0; k < 3; ++k) {
            if (d[k] > 0.0)      sa[k] = ((idx[k] + 1) * h[k] + o[k] - r[k]) / d[k];
            else if (d[k] < 0.0) sa[k] = (idx[k] * h[k] + o[k] - r[k]) / d[k];
            else                 sa[k] = INFINITY;
            if (sa[k] < 0.0) sa[k] = 0.0;
            if (sa[k] < s_b) s_b = sa[k];
        }
        double s_lim = fmin(S_MAX_, F_RNG_ * R);
        int crossing = (s_b <= s_lim * (1.0 + TIE_));     /* reading A22 */
        double s = crossing ? s_b : s_lim;

        /* T7: midpoint-rule mean loss */
        double t   = dens * s / 10.0;                     /* g/cm2 */
        double dE1 = orc_bethe_S(E) * t;
        double Em  = fmax(E - 0.5 * dE1, 1.0e-3);
        double dEm = orc_bethe_S(Em) * t;

        /* T8: straggling, Philox block m */
        philox_block(seed, g, m, u);
        double dE = dEm;
        if (!(flags & ORC_NO_STRAGGLE)) {
            double sig = sqrt(orc_bohr_var_per_t(Em) * t);
            double gg  = sqrt(-2.0 * log(u[2])) * cos(TWO_PI * u[3]);
            dE = dEm + sig * gg;
        }
        if (dE < 0.0) dE = 0.0;
        if (dE > E)   dE = E;
        if (E - dE <= E_CUT_) { dE = E; alive = 0; }      /* A12: residual deposited in this voxel */

        /* T9 / T11: score into the voxel the step lay in */
        int64_t q = llrint(dE * w * scale);
        #pragma omp atomic
        Q[vox] += q;
        T->dep += q;
        T->steps += 1;

        for (int k = 0; k < 3; ++k) r[k] += s * d[k];

        /* T10: boundary-limited step: every axis attaining the minimum is put exactly on its face */
        if (crossing) {
            for (int k = 0; k < 3; ++k) if (sa[k] == s_b) {
                if (d[k] > 0.0) { idx[k] += 1; r[k] = idx[k] * h[k] + o[k]; }
                else            { r[k] = idx[k] * h[k] + o[k]; idx[k] -= 1; }
            }
        }

        /* T9: Highland deflection at the end of the step, kinematics at Em, branch-free basis (A20) */
        if (!(flags & ORC_NO_MCS)) {
            double th0 = sqrt(orc_theta0_sq_per_t(Em) * t);
            double th  = th0 * sqrt(-2.0 * log(u[0]));
            double ph  = TWO_PI * u[1];
            double sw = copysign(1.0, d[2]);
            double aa = -1.0 / (sw + d[2]);
            double bb = d[0] * d[1] * aa;
            double e1[3] = { 1.0 + sw * d[0] * d[0] * aa, sw * bb, -sw * d[0] };
            double e2[3] = { bb, sw + d[1] * d[1] * aa, -d[1] };
            double ct = cos(th), st = sin(th), cp = cos(ph), spn = sin(ph);
            double nd[3], nn = 0.0;
            for (int k = 0; k < 3; ++k) { nd[k] = ct * d[k] + st * (cp * e1[k] + spn * e2[k]); nn += nd[k] * nd[k]; }
            nn = 1.0 / sqrt(nn);
            for (int k = 0; k < 3; ++k) d[k] = nd[k] * nn;
        }
        E -= dE;

        if (crossing && alive) {
            /* probes: first +z crossing of listed faces */
            for (int p = 0; p < n_probe; ++p)
                if (sa[2] == s_b && idx[2] == probe_faces[p] && isnan(probe_xy[((int64_t)p * H + gl) * 2])) {
                    probe_xy[((int64_t)p * H + gl) * 2]     = r[0];
                    probe_xy[((int64_t)p * H + gl) * 2 + 1] = r[1];
                }
            /* T10: left the grid -> remaining kinetic energy escapes */
            if (idx[0] < 0 || idx[0] >= n[0] || idx[1] < 0 || idx[1] >= n[1] || idx[2] < 0 || idx[2] >= n[2]) {
                T->esc += llrint(E * w * scale);
                if (stop_xyz) stop_xyz[gl*3] = stop_xyz[gl*3+1] = stop_xyz[gl*3+2] = NAN;
                return;
            }
        }
    }
    if (stop_xyz) { stop_xyz[gl*3] = r[0]; stop_xyz[gl*3+1] = r[1]; stop_xyz[gl*3+2] = r[2]; }
}

/* threads the parallel loops of this library run on (for the benchmark's "cores" field; no arithmetic) */
int orc_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

int orc_transport(const orc_grid* grid, const float* rho,
                  int32_t n_fields, const orc_field* fields, const orc_spot* spots,
                  int64_t n_segs, const orc_segment* segs,
                  uint64_t seed, int32_t fixed_shift, uint32_t flags,
                  int64_t* Q, orc_mc_stats* stats,
                  int32_t n_probe, const int32_t* probe_faces, int64_t hist_base, int64_t hist_count,
                  double* probe_xy, double* stop_xyz)
{
    if (!grid || !rho || !fields || !spots || (!segs && n_segs) || !Q) return -1;
    (void)n_fields;
    (void)orc_range_water(1.0);                      /* build the range table before the parallel region */
    const double scale = ldexp(1.0, fixed_shift);
    if (probe_xy) for (int64_t i = 0; i < (int64_t)n_probe * hist_count * 2; ++i) probe_xy[i] = NAN;
    int64_t inc = 0, dep = 0, esc = 0; uint64_t steps = 0, hist = 0;
    /* Histories are independent (T1: one Philox stream each) and every tally is an integer sum, so the order in which
     * they run changes nothing.  They are numbered 0 .. total-1 across the segments (begin[s] = histories of the
     * segments before s) and handed to the threads from ONE parallel loop: a loop per segment left the threads idle
     * on plans with thousands of segments of a few histories each. */
    int64_t* begin = (int64_t*)malloc((size_t)(n_segs + 1) * sizeof(int64_t));
    if (!begin) return -2;
    begin[0] = 0;
    for (int64_t s = 0; s < n_segs; ++s) begin[s + 1] = begin[s] + (segs[s].n_hist > 0 ? segs[s].n_hist : 0);
    const int64_t total = begin[n_segs];
    #pragma omp parallel for schedule(dynamic, 256) reduction(+:inc,dep,esc,steps,hist)
    for (int64_t i = 0; i < total; ++i) {
        int64_t lo = 0, hi = n_segs;                 /* the segment s with begin[s] <= i < begin[s + 1] */
        while (hi - lo > 1) { int64_t mid = lo + (hi - lo) / 2; if (begin[mid] <= i) lo = mid; else hi = mid; }
        const orc_segment* sg = &segs[lo];
        const orc_spot*  sp = &spots[sg->spot];
        const orc_field* F  = &fields[sg->field];
        uint64_t g = (uint64_t)(sg->first_history + (i - begin[lo]));
        tally T = { 0, 0, 0, 0 };
        int64_t gl = (int64_t)g - hist_base;
        int traced = (probe_xy || stop_xyz) && gl >= 0 && gl < hist_count;
        one_history(grid, rho, F, sp, sg->weight, seed, g, scale, flags, Q, &T,
                    traced && probe_xy ? n_probe : 0, probe_faces, probe_xy, hist_count, gl,
                    traced ? stop_xyz : 0);
        inc += T.inc; dep += T.dep; esc += T.esc; steps += T.steps; hist += 1;
    }
    free(begin);
    if (stats) {
        stats->histories = hist; stats->steps = steps;
        stats->q_incident = inc; stats->q_deposited = dep; stats->q_escaped = esc;
        stats->fixed_shift = fixed_shift; stats->pad = 0;
    }
    return 0;
}

/* T12 (the MC outputs dose and density per voxel) */
void orc_finalize_dose(const orc_grid* G, const float* rho, const int64_t* Q, int32_t fixed_shift,
                       double per_protons, float* dose)
{
    const double vol_cm3 = (double)G->hx * (double)G->hy * (double)G->hz * 1.0e-3;
    const double inv = ldexp(1.0, -fixed_shift);
    const size_t nvox = (size_t)G->nx * G->ny * G->nz;
    for (size_t i = 0; i < nvox; ++i) {
        double D = (double)Q[i] * inv * 1.602176634e-10 / ((double)rho[i] * vol_cm3);
        if (per_protons > 0.0) D /= per_protons;
        dose[i] = (float)D;
    }
}

/* a1: piecewise-linear HU -> density, clamped to the table ends (reading A4); optional overlap-volume-weighted
 * resampling onto the dose grid (reading A19).  BASELINE.json config 2: (-1000,0.001), (0,1.0), (1000,1.6). */
static double hu2rho(double hu, int n, const float* hp, const float* rp)
{
    if (hu <= hp[0]) return rp[0];
    if (hu >= hp[n - 1]) return rp[n - 1];
    int k = 0;
    while (k < n - 2 && hu >= hp[k + 1]) ++k;
    double f = (hu - (double)hp[k]) / ((double)hp[k + 1] - (double)hp[k]);
    return (double)rp[k] + f * ((double)rp[k + 1] - (double)rp[k]);
}

int orc_hu_to_density(const orc_grid* ct, const int16_t* hu, const orc_grid* dg,
                      int32_t n_pts, const float* hp, const float* rp, float* out)
{
    if (!ct || !hu || n_pts < 2 || !hp || !rp || !out) return -1;
    if (!dg) {
        size_t nv = (size_t)ct->nx * ct->ny * ct->nz;
        for (size_t i = 0; i < nv; ++i) out[i] = (float)hu2rho((double)hu[i], n_pts, hp, rp);
        return 0;
    }
    const double ch[3] = { ct->hx, ct->hy, ct->hz }, co[3] = { ct->ox, ct->oy, ct->oz };
    const int    cn[3] = { ct->nx, ct->ny, ct->nz };
    const double dh[3] = { dg->hx, dg->hy, dg->hz }, d0[3] = { dg->ox, dg->oy, dg->oz };
    #pragma omp parallel for schedule(static)
    for (int z = 0; z < dg->nz; ++z)
    for (int y = 0; y < dg->ny; ++y)
    for (int x = 0; x < dg->nx; ++x) {
        int id[3] = { x, y, z };
        int lo[3], hi[3];
        for (int k = 0; k < 3; ++k) {
            double a = d0[k] + id[k] * dh[k], b = a + dh[k];
            lo[k] = (int)floor((a - co[k]) / ch[k]); if (lo[k] < 0) lo[k] = 0;
            hi[k] = (int)ceil((b - co[k]) / ch[k]);  if (hi[k] > cn[k]) hi[k] = cn[k];
        }
        double acc = 0.0, wsum = 0.0;
        for (int kz = lo[2]; kz < hi[2]; ++kz)
        for (int ky = lo[1]; ky < hi[1]; ++ky)
        for (int kx = lo[0]; kx < hi[0]; ++kx) {
            int ic[3] = { kx, ky, kz };
            double wv = 1.0;
            for (int k = 0; k < 3; ++k) {
                double a = d0[k] + id[k] * dh[k], b = a + dh[k];
                double ca = co[k] + ic[k] * ch[k], cb = ca + ch[k];
                double ov = fmin(b, cb) - fmax(a, ca);
                wv *= ov > 0.0 ? ov : 0.0;
            }
            if (wv > 0.0) {
                acc  += wv * hu2rho((double)hu[((size_t)kz * cn[1] + ky) * cn[0] + kx], n_pts, hp, rp);
                wsum += wv;
            }
        }
        /* a dose voxel not overlapping the CT at all is vacuum-like air: first table density */
        out[((size_t)z * dg->ny + y) * dg->nx + x] = (float)(wsum > 0.0 ? acc / wsum : (double)rp[0]);
    }
    return 0;
}
