/* oracle/orc.h -- CPU ORACLE for the pbs4d hot path.  TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, double-precision C restatement of what the path computes, written from
 * /root/reference/PAPER.md (arxiv 1809.03927) and BASELINE.json's north_star / configs, following the
 * step lists D1-D7, T1-T12, A1-A6 of SURVEY.md section 8(c) with the readings listed in DESIGN.md.
 * It shares NO code with the CUDA path (paper_1809_03927_b200/csrc) and is never called by it.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may use it.
 *
 * Conventions: grids are C-order [z][y][x] (x fastest); o = corner of voxel (0,0,0); lengths mm,
 * energies MeV, density g/cm3.  All pointers are HOST pointers owned by the caller.
 */
#ifndef ORC_H
#define ORC_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct { int32_t nx, ny, nz; float hx, hy, hz, ox, oy, oz; } orc_grid;

/* PAPER.md:239 "spots which each have a specific (x,y) position and energy"; PAPER.md:45 (location, energy, weight) */
typedef struct { float dir[3], eu[3], ev[3], ref[3]; int32_t start_phase; } orc_field;
typedef struct { int32_t field, layer; float x_mm, y_mm, energy_mev, sigma_mm, weight; } orc_spot;

/* BASELINE.json:9,11 delivery model (spot time ~ weight at protons_per_s, scan speed, energy switch,
 * breathing period, repainting, gating) */
typedef struct {
    int32_t n_phases; int64_t period_ns; int64_t protons_per_weight; int64_t protons_per_s;
    int32_t ns_per_um; int64_t layer_switch_ns; int32_t repaints; uint32_t gate_mask;
} orc_delivery_params;

/* one (field, phase, spot) entry of the sub-plans of PAPER.md:49, after history allocation (D7) */
typedef struct {
    int32_t field, phase, spot; int32_t pad;
    int64_t protons;        /* protons delivered to this spot in this phase */
    int64_t first_history;  /* global history index of the first history of the segment */
    int64_t n_hist;         /* histories simulated for it (0: segment dropped) */
    double  weight;         /* protons / n_hist */
} orc_segment;

/* ---- Philox4x32-10 (T1) ---- */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);

/* ---- physics closed forms (T5, T8, T9) ---- */
double orc_bethe_S(double E_mev);            /* mass stopping power of water, MeV cm2/g */
double orc_range_water(double E_mev);        /* CSDA range incl. closure R_c, g/cm2 (table, log-log interp.) */
double orc_bohr_var_per_t(double E_mev);     /* straggling variance per mass thickness, MeV2 cm2/g */
double orc_theta0_sq_per_t(double E_mev);    /* Highland theta0^2 per mass thickness (no log term), cm2/g */

/* ---- delivery (D1-D7) ----
 * Two-call protocol: call with segs == NULL to get the number of segments, then with a buffer.
 * Returns number of segments (>=0) or <0 on bad arguments.  total_histories == 0: skip D7 (n_hist = 0).
 * total_time_ns (optional) receives each field's end-of-delivery time [n_fields]. */
int64_t orc_simulate_delivery(int32_t n_fields, const orc_field* fields, int64_t n_spots, const orc_spot* spots,
                              const orc_delivery_params* prm, uint64_t total_histories,
                              orc_segment* segs, int64_t max_segs, int64_t* total_time_ns,
                              int64_t* dropped_protons);

/* Extended delivery model (steps E1-E5 in orc_delivery.c): all zero / NULL = base model. */
typedef struct {
    int32_t n_cycles; const int64_t* cycle_period_ns;   /* irregular breathing: period of cycle c (last one repeats) */
    int64_t discard_ns;                                 /* beam discarded when extraction (re)starts (70 ms) */
    int64_t spill_protons_max;                          /* charge capacity of one synchrotron fill; 0 = unlimited */
    int64_t flat_top_ns;                                /* flat-top / extraction time limit of a fill; 0 = unlimited */
    int64_t spot_switch_fixed_ns;                       /* fixed prepare/verify part of the spot-switch time */
    int32_t n_layer_switch; const int64_t* layer_switch_ns;   /* energy-dependent reset time per layer id */
    int64_t max_protons_per_paint;                      /* iso-layered repainting: max protons per spot delivery */
} orc_delivery_ext;

int64_t orc_simulate_delivery_ext(int32_t n_fields, const orc_field* fields, int64_t n_spots, const orc_spot* spots,
                                  const orc_delivery_params* prm, const orc_delivery_ext* ext, uint64_t total_histories,
                                  orc_segment* segs, int64_t max_segs, int64_t* total_time_ns,
                                  int64_t* dropped_protons, int64_t* n_fills);

/* ---- uncertainty trials (steps U0-U5 in orc_trials.c) ---- */
typedef struct {
    uint64_t seed;
    int32_t  n_trials, n_cycles;                  /* trials; breathing cycles sampled per trial (the last repeats) */
    int64_t  period_lo_ns, period_hi_ns, period_step_ns;   /* mean period ~ U{lo, lo + step, ... <= hi}; lo = 0: fixed */
    int64_t  period_sigma_ns;                     /* per-cycle period ~ N(mean, sigma) */
    int64_t  discard_sigma_ns, flat_top_sigma_ns, spot_switch_sigma_ns, layer_switch_sigma_ns;
    int64_t  spill_protons_sigma, protons_per_s_sigma;     /* 1-sigma of the synchrotron parameters; 0 = fixed */
} orc_trial_spec;

/* Sample trial `trial`: start_phase[n_fields], cycle_period_ns[spec->n_cycles], layer_switch_ns[ext->n_layer_switch]
 * (caller's arrays); prm_out / ext_out = copies of prm / ext with the sampled values, pointing into those arrays. */
int orc_sample_trial(const orc_trial_spec* spec, int32_t trial, int32_t n_fields,
                     const orc_delivery_params* prm, const orc_delivery_ext* ext,
                     int32_t* start_phase, int64_t* cycle_period_ns, int64_t* layer_switch_ns,
                     orc_delivery_params* prm_out, orc_delivery_ext* ext_out);

/* ---- transport (T1-T12) ---- */
#define ORC_NO_MCS       1u   /* pin switch: no Highland deflection        */
#define ORC_NO_STRAGGLE  2u   /* pin switch: no Bohr straggling            */
#define ORC_NO_ESPREAD   4u   /* pin switch: mono-energetic source         */
#define ORC_NO_SPOTSIZE  8u   /* pin switch: zero-width spot               */

typedef struct {
    uint64_t histories, steps;
    int64_t  q_incident, q_deposited, q_escaped;   /* fixed point, quantum 2^-fixed_shift MeV */
    int32_t  fixed_shift; int32_t pad;
} orc_mc_stats;

/* T11: k = floor(log2(2^62 / (1.1 * sum protons*E_spot))) */
int32_t orc_fixed_shift(int64_t n_segs, const orc_segment* segs, const orc_spot* spots);

/* Transport the histories of the given segments on one density grid.
 * Q [nz*ny*nx] int64 is ADDED to (caller zeroes).  probe_faces: optional list of z-face indices k (face between
 * voxel k-1 and k); probe_xy[(p*H + g_local)*2 + {0,1}] receives x,y of history g_local = g - hist_base at its first +z crossing
 * of that face (NaN if never).  stop_xyz[g_local*3..] (optional) receives the position where the history ended
 * (absorbed) or NaN if it escaped. */
/* number of threads orc_transport's history loop runs on (OpenMP; OMP_NUM_THREADS) */
int orc_threads(void);

int orc_transport(const orc_grid* grid, const float* rho,
                  int32_t n_fields, const orc_field* fields, const orc_spot* spots,
                  int64_t n_segs, const orc_segment* segs,
                  uint64_t seed, int32_t fixed_shift, uint32_t flags,
                  int64_t* Q, orc_mc_stats* stats,
                  int32_t n_probe, const int32_t* probe_faces, int64_t hist_base, int64_t hist_count,
                  double* probe_xy, double* stop_xyz);

/* T12: D = Q 2^-k 1.602176634e-10 / (rho V[cm3] 1e-3 kg/g) -> fp32 Gy;  per_protons > 0 divides by it */
void orc_finalize_dose(const orc_grid* grid, const float* rho, const int64_t* Q, int32_t fixed_shift,
                       double per_protons, float* dose);

/* a1: HU -> rho piecewise linear (clamped), optional overlap-volume-weighted resample to dose grid (A19) */
int orc_hu_to_density(const orc_grid* ct, const int16_t* hu, const orc_grid* dose_grid /*NULL: == ct*/,
                      int32_t n_pts, const float* hu_pts, const float* rho_pts, float* rho_out);

/* ---- accumulation (A1-A6), strict fp32 + int64 ---- */
typedef struct { uint64_t subvoxels, dropped_outside_ref, dropped_outside_dvf; } orc_acc_stats;

/* Push one source phase (A1-A5): adds into E, M [ref grid] (caller zeroes). */
int orc_emtm_push(const orc_grid* src, const float* dose, const float* rho,
                  const orc_grid* dvf_grid, const float* disp /*[3][z][y][x]*/,
                  const orc_grid* ref, int32_t nsx, int32_t nsy, int32_t nsz,
                  int64_t* E, int64_t* M, orc_acc_stats* stats);

/* A6 for n_src pushed phases: out = (float)(D_ref + sum_S E_S/M_S 2^-8), masked by DVF coverage.
 * E, M: [n_src][ref voxels]; dvf_grids: [n_src]. */
int orc_emtm_finalize(const orc_grid* ref, const float* dose_ref, int32_t n_src,
                      const int64_t* E, const int64_t* M, const orc_grid* dvf_grids, float* out);

/* ---- dose-interpolation method (DIM), Eq. 3; steps P1-P5 in orc_dim.c ----
 * Pull one source phase: dose_pulled[i] = D_i^S (double) for every reference voxel.  disp = T^{R->S} as displacements
 * [3][z][y][x] mm on grid Dg in the REFERENCE frame; dose_src on grid S.  stats: subvoxels, dropped_outside_ref =
 * mapped points outside the source grid, dropped_outside_dvf = subvoxel centres outside the DVF grid. */
int orc_dim_pull(const orc_grid* R, int32_t nsx, int32_t nsy, int32_t nsz,
                 const orc_grid* Dg, const float* disp, const orc_grid* S, const float* dose_src,
                 double* dose_pulled, orc_acc_stats* stats);

/* Eq. 2 + mask for n_src pulled phases: out = (float)(D_ref + sum_S pulled[S]) in ascending order, 0 where the voxel
 * centre is outside any DVF's extent.  pulled: [n_src][R voxels]. */
int orc_dim_finalize(const orc_grid* R, const float* dose_ref, int32_t n_src, const double* pulled,
                     const orc_grid* dvf_grids, float* out);

/* ---- DVF construction from DICOM minimal grid information, PAPER.md:251-259 (App. B, Eq. 7-8) ---- */
typedef struct {
    int32_t nx, ny, nz, pad;                 /* N_X (row direction), N_Y (column direction), N_Z (depth direction) */
    double start[3];                         /* centre of the starting voxel, mm */
    double delta[3];                         /* deformation-grid resolutions */
    double row_cos[3], col_cos[3];           /* U, V; W = U x V */
    double pre[16], post[16];                /* M_Pre, M_Post, row-major 4x4 */
} orc_dicom_dvf;

/* delta: translations [3][k][j][i] (fp32); rf / disp (either may be NULL): r_f and r_f - r_0, fp32 [3][k][j][i] */
int orc_build_dvf(const orc_dicom_dvf* grid, const float* delta, float* rf, float* disp);

#ifdef __cplusplus
}
#endif
#endif
