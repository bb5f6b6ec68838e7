/* pbs4d.h -- C-ABI boundary of the B200-native 4D proton dose hot path (arxiv 1809.03927, Pepin et al.).
 *
 * The calls follow the paper's statement of the problem (inputs are N_g CT series, N_g-1 deformation
 * fields and one plan; PAPER.md:53-55 delivery options; PAPER.md:122 accumulation method and subdivision n; output
 * is one dose on the reference phase) and the names fixed by BASELINE.json north_star:
 *   set_ct_phases, set_plan_spots, simulate_delivery -> per-phase spot/proton lists, mc_dose_phase,
 *   accumulate_subvoxel -> 4D dose.
 *
 * Conventions.  Grids are C-order [z][y][x] (x fastest); o = corner of voxel (0,0,0), voxel centre = o + (i+1/2) h.
 * Lengths mm, energies MeV, densities g/cm3, dose Gy.  Pointers named *_dev are DEVICE pointers on the context's
 * device; everything else is a HOST pointer.  The caller owns every buffer it passes; it must stay valid until the
 * call returns.  All calls enqueue on the context's stream and synchronise it before returning.
 * Every function returns PBS4D_OK (0) or a negative error code; nothing throws across the boundary; the message of
 * the last error is available from pbs4d_last_error().  There is NO CPU fallback: without a CUDA device
 * pbs4d_create fails with PBS4D_ERR_CUDA.
 */
#ifndef PBS4D_H
#define PBS4D_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PBS4D_OK             0
#define PBS4D_ERR_ARG       (-1)   /* bad argument                         */
#define PBS4D_ERR_ORDER     (-2)   /* call-order violation                 */
#define PBS4D_ERR_CUDA      (-3)   /* CUDA runtime error / no device       */
#define PBS4D_ERR_NOMEM     (-4)   /* out of host or device memory         */
#define PBS4D_ERR_OVERFLOW  (-5)   /* fixed-point overflow guard tripped   */

typedef struct pbs4d_ctx pbs4d_ctx;      /* opaque; owns all internal host/device memory */

/* at most 4 000 000 x 262 140 x 65 535 voxels (x, y, z: kernel launch geometry) and fewer than 2e9 in total;
 * anything else is refused with PBS4D_ERR_ARG by the call that receives the grid */
typedef struct { int32_t nx, ny, nz; float hx, hy, hz, ox, oy, oz; } pbs4d_grid;

/* A treatment field: parallel beam along dir; (eu, ev) span the beam's-eye-view plane through ref.
 * start_phase = breathing phase in which delivery of this field commences. */
typedef struct { float dir[3], eu[3], ev[3], ref[3]; int32_t start_phase; } pbs4d_field;

/* A spot = (x, y) position, energy, weight; all spots of one energy form a layer. */
typedef struct { int32_t field, layer; float x_mm, y_mm, energy_mev, sigma_mm, weight; } pbs4d_spot;

/* Delivery timing model (App. A; values as BASELINE.json configs 3, 5). */
typedef struct {
    int32_t  n_phases;             /* N_g breathing phases                                          */
    int64_t  period_ns;            /* breathing period; phase length = period_ns / n_phases         */
    int64_t  protons_per_weight;   /* protons of a spot = llround(weight * protons_per_weight)      */
    int64_t  protons_per_s;        /* spill rate ("spot-spill time")                  */
    int32_t  ns_per_um;            /* scan speed ("spot-switch time"); 10 m/s -> 100                */
    int64_t  layer_switch_ns;      /* "layer-switch time"                            */
    int32_t  repaints;             /* N x layer repainting (BASELINE.json config 5); >= 1           */
    uint32_t gate_mask;            /* bit p set = beam allowed in phase p (gating)     */
} pbs4d_delivery_params;

/* Extended delivery model: the synchrotron behaviour the paper describes beyond the constants of BASELINE.json's
 * configs (Sec. 2.B; App. A).  The paper takes its values from its Ref. 45, which is
 * not available: every value is an input, and the sampled breathing periods (t_ph ~ N(mu, sigma)/N) are
 * passed in rather than drawn inside.  All zero / NULL = the base model of pbs4d_delivery_params. */
typedef struct {
    int32_t n_cycles; const int64_t* cycle_period_ns;  /* irregular breathing: period of breathing cycle c, ns; the
                                                          last entry repeats; NULL: period_ns for every cycle        */
    int64_t discard_ns;             /* beam discarded whenever extraction (re)starts: after every synchrotron reset and
                                       after every wait for gate-on (70 ms); must be < one phase        */
    int64_t spill_protons_max;      /* charge capacity of one synchrotron fill (~2 nC); 0 = unlimited   */
    int64_t flat_top_ns;            /* flat-top / extraction time limit of a fill, counted from the end of the reset
                                       (~8 s); 0 = unlimited; must exceed discard_ns + longest period  */
    int64_t spot_switch_fixed_ns;   /* fixed prepare/verify part of the spot-switch time               */
    int32_t n_layer_switch; const int64_t* layer_switch_ns;   /* energy-dependent reset ("layer-switch") time per layer
                                       id; NULL or id out of range: layer_switch_ns of the base struct */
    int64_t max_protons_per_paint;  /* iso-layered repainting with a maximum MU per spot delivery: every
                                       painting delivers at most this many protons of each spot until none is left;
                                       0: the base N x repainting                                                      */
} pbs4d_delivery_ext;

/* One entry of the sub-plans after history allocation. */
typedef struct {
    int32_t field, phase, spot, pad;
    int64_t protons;               /* protons of this spot delivered in this phase by this field    */
    int64_t first_history;         /* global history index (Philox counter) of its first history    */
    int64_t n_hist;                /* histories simulated for it (0: dropped)                       */
    double  weight;                /* protons / n_hist                                              */
} pbs4d_segment;

/* Result of simulate_delivery; arrays are owned by the context, valid until the next simulate_delivery/destroy.
 * Segments are sorted by (field, phase, spot). */
typedef struct {
    int64_t n_segments; const pbs4d_segment* segments;
    int32_t n_fields;   const int64_t* field_time_ns;   /* end-of-delivery time per field */
    int64_t dropped_protons;                            /* protons of segments that got 0 histories */
    int32_t fixed_shift;                                /* k: dose quantum = 2^-k MeV */
} pbs4d_phase_lists;

#define PBS4D_NO_MCS       1u      /* test switches: disable Highland deflection / Bohr straggling /       */
#define PBS4D_NO_STRAGGLE  2u      /* source energy spread / spot size                                      */
#define PBS4D_NO_ESPREAD   4u
#define PBS4D_NO_SPOTSIZE  8u
#define PBS4D_TEST_STEP_CAP_64 16u /* test switch: the transport's step cap (hang guard) at 64 steps instead of 2^20 */

typedef struct {
    uint64_t histories, steps;
    int64_t  q_incident, q_deposited, q_escaped;        /* fixed point, quantum 2^-fixed_shift MeV */
    int32_t  fixed_shift; int32_t pad;
    float    kernel_ms;                                 /* device time of the transport kernel (CUDA events) */
    int32_t  aborted;                                   /* histories stopped by the step cap (2^20 steps; their energy
                                                           is deposited where they stood): 0 for any valid input */
    uint64_t scoring_atomics;                           /* red.global.add.u64 issued by the scoring (one per voxel visit) */
} pbs4d_mc_stats;

typedef struct {
    uint64_t subvoxels, dropped_outside_ref, dropped_outside_dvf;
    float    push_ms, finalize_ms;                      /* device times (CUDA events) */
} pbs4d_acc_stats;

/* Create a context on CUDA device `device`; cuda_stream is a cudaStream_t (e.g. torch's current stream) or NULL. */
int  pbs4d_create(pbs4d_ctx** out, int device, void* cuda_stream);
void pbs4d_destroy(pbs4d_ctx* ctx);
const char* pbs4d_last_error(const pbs4d_ctx* ctx);

/* a1 (the MC converts Hounsfield units to material density).  hu_dev[p] -> int16 [z][y][x] on grid ct.
 * Density = piecewise-linear table (hu_pts ascending, n_pts >= 2, clamped at the ends), resampled by overlap-volume
 * weighted mean onto dose_grid (NULL: dose grid == ct grid).  The context keeps fp32 densities. */
int pbs4d_set_ct_phases(pbs4d_ctx* ctx, int32_t n_phases, const pbs4d_grid* ct, const int16_t* const* hu_dev,
                        const pbs4d_grid* dose_grid, int32_t n_pts, const float* hu_pts, const float* rho_pts);

/* Alternative to set_ct_phases: densities given directly on the dose grid (rho_dev[p] -> fp32 [z][y][x]); copied.
 * Every density must be finite and within [1e-6, 100] g/cm3 (checked on the device; PBS4D_ERR_ARG otherwise): a zero
 * density has no dose (0/0), an infinite one a zero step limit. */
int pbs4d_set_density_phases(pbs4d_ctx* ctx, int32_t n_phases, const pbs4d_grid* dose_grid,
                             const float* const* rho_dev);

/* Deformation vector field T^{S->R} (Eq. 1; App. B) as displacements [3][z][y][x] (x,y,z components,
 * mm) at the centres of an axis-aligned grid in the SOURCE phase frame; trilinear in between.
 * Copied into the context.  Requires set_ct_phases/set_density_phases first. */
int pbs4d_set_dvf(pbs4d_ctx* ctx, int32_t src_phase, int32_t ref_phase, const pbs4d_grid* dvf_grid,
                  const float* disp_dev);

/* Fields and spots in delivery order (copied). */
int pbs4d_set_plan_spots(pbs4d_ctx* ctx, int32_t n_fields, const pbs4d_field* fields,
                         int64_t n_spots, const pbs4d_spot* spots);

/* Optional physics switches for tests (default 0 = full model). */
int pbs4d_set_mc_flags(pbs4d_ctx* ctx, uint32_t flags);

/* a3: beam-delivery simulation on the host in int64 arithmetic; splits every spot's protons over
 * the phases it is delivered in and allocates total_histories over the resulting segments. */
int pbs4d_simulate_delivery(pbs4d_ctx* ctx, const pbs4d_delivery_params* prm, uint64_t total_histories,
                            pbs4d_phase_lists* out);

/* The same simulation without a context or a device (host only; used by CPU tests and tools).  Writes at most
 * max_segs segments to segs_out (may be NULL to query), the segment count to *n_segs_out, per-field end times to
 * field_time_ns[n_fields] (optional), dropped protons and the fixed-point shift (optional). */
int pbs4d_simulate_delivery_host(int32_t n_fields, const pbs4d_field* fields, int64_t n_spots,
                                 const pbs4d_spot* spots, const pbs4d_delivery_params* prm, uint64_t total_histories,
                                 pbs4d_segment* segs_out, int64_t max_segs, int64_t* n_segs_out,
                                 int64_t* field_time_ns, int64_t* dropped_protons, int32_t* fixed_shift);

/* The same with the extended model; *n_fills (optional) receives the number of synchrotron fills of all fields. */
int pbs4d_simulate_delivery_ext(pbs4d_ctx* ctx, const pbs4d_delivery_params* prm, const pbs4d_delivery_ext* ext,
                                uint64_t total_histories, pbs4d_phase_lists* out, int64_t* n_fills);
int pbs4d_simulate_delivery_ext_host(int32_t n_fields, const pbs4d_field* fields, int64_t n_spots,
                                     const pbs4d_spot* spots, const pbs4d_delivery_params* prm,
                                     const pbs4d_delivery_ext* ext, uint64_t total_histories,
                                     pbs4d_segment* segs_out, int64_t max_segs, int64_t* n_segs_out,
                                     int64_t* field_time_ns, int64_t* dropped_protons, int32_t* fixed_shift,
                                     int64_t* n_fills);

/* ---- uncertainty trials ----
 * "The effect of these uncertainties was considered by running 25 trials of the 4DDC where, for each trial, the
 * initial-breathing phase, breathing period, and synchrotron delivery parameters were simultaneously varied according
 * to their statistical distributions ...: starting phase ~ U(CT_0, CT_90), synchrotron parameters ~ N(mu, sigma), and
 * breathing period ~ U(3,7) s" (discrete uniforms, inclusive); "t_ph ~ N(mu, sigma)/N" per breathing cycle
 * (PAPER.md:55).  Ref. 45's central values and uncertainties are not available: they are inputs.  Every draw is one
 * Philox4x32-10 block addressed by (what, which, trial) under `seed`, so a trial can be sampled on its own. */
typedef struct {
    uint64_t seed;
    int32_t  n_trials;              /* T (25 in the paper)                                                    */
    int32_t  n_cycles;              /* breathing cycles sampled per trial (the last one repeats); 0: regular   */
    int64_t  period_lo_ns, period_hi_ns, period_step_ns;   /* mean period ~ U{lo, lo + step, ... <= hi}; lo = 0: the
                                                              plan's period_ns, not sampled                     */
    int64_t  period_sigma_ns;       /* per-cycle period ~ N(mean period, sigma), floored at a quarter of the mean */
    int64_t  discard_sigma_ns, flat_top_sigma_ns, spot_switch_sigma_ns, layer_switch_sigma_ns;
    int64_t  spill_protons_sigma, protons_per_s_sigma;     /* 1-sigma uncertainties of the parameters; 0 = fixed */
} pbs4d_trial_spec;

/* Device-free: sample trial `trial` (0 <= trial < n_trials) around the central values prm / ext.  The caller's arrays
 * start_phase[n_fields], cycle_period_ns[spec->n_cycles], layer_switch_ns[ext->n_layer_switch] receive the draws;
 * *prm_out / *ext_out are copies of prm / ext with the sampled values whose pointers refer to those arrays.  Sampled
 * values are clamped so that every trial can be delivered (discard < shortest phase, flat-top > longest period). */
int pbs4d_sample_delivery_trial(const pbs4d_trial_spec* spec, int32_t trial, int32_t n_fields,
                                const pbs4d_delivery_params* prm, const pbs4d_delivery_ext* ext,
                                int32_t* start_phase, int64_t* cycle_period_ns, int64_t* layer_switch_ns,
                                pbs4d_delivery_params* prm_out, pbs4d_delivery_ext* ext_out);

/* a3 for one trial: sample it, start every field in its sampled phase and run the extended delivery simulation (always
 * the extended one: with ext == NULL the central values are the base model's, which the extended simulator reproduces).
 * The plan kept by the context is not changed: the planned starting phases are back when the call returns, also after
 * an error; only the segment lists in the context are the trial's. */
int pbs4d_simulate_delivery_trial(pbs4d_ctx* ctx, const pbs4d_trial_spec* spec, int32_t trial,
                                  const pbs4d_delivery_params* prm, const pbs4d_delivery_ext* ext,
                                  uint64_t total_histories, pbs4d_phase_lists* out, int64_t* n_fills);

typedef struct {
    uint64_t histories;             /* histories transported in this trial                                    */
    int64_t  delivery_ns;           /* end of delivery of the slowest field                                   */
    int64_t  fills;                 /* synchrotron fills of all fields                                        */
    int32_t  phases_run, pad;       /* phases that received beam                                              */
    float    transport_ms, accumulate_ms;   /* device times                                                   */
} pbs4d_trial_result;

/* The trial loop: for trial = first .. first + count - 1: simulate_delivery_trial, mc_dose_phases (Philox key
 * seed + trial) on every phase that receives beam plus ref_phase, accumulate_subvoxel onto ref_phase; the 4D dose of
 * trial t goes to dose4d_dev[t - first] (fp32 [z][y][x], caller's buffers).  Densities, DVFs and the plan must have
 * been set; the context is re-used across trials (no allocation after the first).  results (optional) -> [count]. */
int pbs4d_run_trials(pbs4d_ctx* ctx, const pbs4d_trial_spec* spec, int32_t first, int32_t count,
                     const pbs4d_delivery_params* prm, const pbs4d_delivery_ext* ext, uint64_t total_histories,
                     uint64_t seed, int32_t ref_phase, int32_t nsx, int32_t nsy, int32_t nsz,
                     float* const* dose4d_dev, pbs4d_trial_result* results);

/* a4-a7: Monte Carlo transport of all segments of `phase` on that phase's density grid.
 * dose_dev (optional) receives fp32 Gy [z][y][x] on the dose grid for the delivered protons (divided by
 * per_protons if > 0, e.g. "Gy per proton"); rho_dev (optional) receives the density grid (dose and
 * density are the MC's outputs).  The context keeps the phase dose for accumulate_subvoxel. */
int pbs4d_mc_dose_phase(pbs4d_ctx* ctx, int32_t phase, uint64_t seed, double per_protons,
                        float* dose_dev, float* rho_dev, pbs4d_mc_stats* stats);

/* The same for n distinct phases at once ("N_g simulations per field", one per breathing phase; the
 * paper spread them over its 8 cards, here they share one device): the n transport kernels are enqueued on internal
 * streams between a fork and a join on the context's stream, so the drain of one persistent kernel overlaps the next.
 * stats (optional) -> [n], in the order of `phases`; kernel_ms of overlapping launches overlap too, so *elapsed_ms
 * (optional) receives the device time from fork to join.  Results are identical to n mc_dose_phase calls. */
int pbs4d_mc_dose_phases(pbs4d_ctx* ctx, int32_t n, const int32_t* phases, uint64_t seed, double per_protons,
                         pbs4d_mc_stats* stats, float* elapsed_ms);

/* Fixed-point energy grid of the last mc_dose_phase call for `phase`, copied to q_dev (int64 [z][y][x]). */
int pbs4d_get_phase_energy(pbs4d_ctx* ctx, int32_t phase, int64_t* q_dev);

/* a8-a9 (Eq. 2, 4-6): energy-/mass-transfer accumulation with nsx*nsy*nsz subvoxels per voxel of
 * every source phase that has a DVF to ref_phase, onto ref_phase; masked to the volume covered by all DVFs.
 * phase_dose_dev: [n_phases] device pointers to fp32 doses on the dose grid, or NULL to use the doses kept by
 * mc_dose_phase.  dose4d_dev: fp32 [z][y][x] out. */
int pbs4d_accumulate_subvoxel(pbs4d_ctx* ctx, int32_t ref_phase, int32_t nsx, int32_t nsy, int32_t nsz,
                              const float* const* phase_dose_dev, float* dose4d_dev, pbs4d_acc_stats* stats);

/* Integer energy/mass sums of the last accumulate_subvoxel for one source phase (int64 [z][y][x] each). */
int pbs4d_get_accumulators(pbs4d_ctx* ctx, int32_t src_phase, int64_t* e_dev, int64_t* m_dev);

/* ---- multi-GPU sharding ("N_g simulations per field", "the MC was distributed amongst eight
 * GPUs").  One process per GPU, each with its own context holding the whole plan.  Histories are
 * independent units (one Philox counter each), so rank r of w transports the contiguous slice
 * [floor(n r / w), floor(n (r+1) / w)) of every phase's n local histories; the int64 energy grids of the ranks then
 * add up to the unsharded grid BIT FOR BIT.  The caller sums them in place (an integer all-reduce over
 * pbs4d_phase_energy_ptr, e.g. NCCL through torch.distributed) and re-derives the dose with
 * pbs4d_finalize_phase_dose.  Accumulation shards by source phase: pbs4d_accumulate_push with the rank's src_mask,
 * exchange of the int64 sums (pbs4d_accumulator_ptrs: broadcast from the owner or all-reduce, the other ranks hold
 * zeros), then pbs4d_accumulate_finalize on every rank. */

/* Device-free partition arithmetic: *begin, *count of rank's slice of n_hist histories (every history exactly once
 * over the ranks; empty slices when world > n_hist). */
int pbs4d_shard_window(int64_t n_hist, int32_t rank, int32_t world, int64_t* begin, int64_t* count);

/* Subsequent mc_dose_phase(s) transport only this rank's slice of every phase (default rank 0 of 1 = everything).
 * Stats then count the slice; doses kept by the context are partial until the grids have been summed.  The setting
 * stays until changed; pbs4d_run_plan_host and pbs4d_run_trials, which contain no exchange step, return
 * PBS4D_ERR_ORDER while world > 1. */
int pbs4d_set_shard(pbs4d_ctx* ctx, int32_t rank, int32_t world);

/* Device pointer to the context's own int64 energy grid [z][y][x] of `phase` (valid until the next set_ct_phases /
 * set_density_phases / destroy) for an in-place integer sum over ranks. */
int pbs4d_phase_energy_ptr(pbs4d_ctx* ctx, int32_t phase, int64_t** q_dev);

/* a7 again, from the (now summed) energy grid: refreshes the phase dose kept by the context. */
int pbs4d_finalize_phase_dose(pbs4d_ctx* ctx, int32_t phase, double per_protons);

/* a8 alone: zero the accumulators of every eligible source phase (DVF to ref_phase + a dose) and push those whose
 * bit is set in src_mask.  stats->subvoxels counts the pushed phases only. */
int pbs4d_accumulate_push(pbs4d_ctx* ctx, int32_t ref_phase, int32_t nsx, int32_t nsy, int32_t nsz,
                          const float* const* phase_dose_dev, uint32_t src_mask, pbs4d_acc_stats* stats);

/* Device pointers to the context's own int64 E and M sums [z][y][x] of one eligible source phase (valid as above). */
int pbs4d_accumulator_ptrs(pbs4d_ctx* ctx, int32_t src_phase, int64_t** e_dev, int64_t** m_dev);

/* a9 alone over every eligible source phase (all of them must have been pushed or received). */
int pbs4d_accumulate_finalize(pbs4d_ctx* ctx, int32_t ref_phase, const float* const* phase_dose_dev,
                              float* dose4d_dev, pbs4d_acc_stats* stats);

/* Whole path with HOST buffers (copies inside): set_plan_spots + simulate_delivery first (host, milliseconds) -- the
 * sub-plans say which breathing phases receive beam; then, for those phases and the reference phase only, CT upload +
 * HU -> density, DVF upload (on a copy stream, underneath the transport), mc_dose_phases, accumulate_subvoxel and
 * the copy of the 4D dose to dose4d_host.  CTs and DVFs of phases that receive no beam (gating) are never touched.
 * hu_host[p] (all non-NULL), disp_host[p] (NULL = no DVF for p).  histories_run, h2d_bytes (bytes actually copied host ->
 * device), seconds ([4]: delivery simulation, upload + density enqueue, transport, accumulate + D2H; wall times) are
 * optional.  Afterwards the context holds densities and doses of the active phases only. */
int pbs4d_run_plan_host(pbs4d_ctx* ctx, int32_t n_phases, const pbs4d_grid* ct, const int16_t* const* hu_host,
                        const pbs4d_grid* dose_grid, int32_t n_pts, const float* hu_pts, const float* rho_pts,
                        const pbs4d_grid* dvf_grid, const float* const* disp_host, int32_t ref_phase,
                        int32_t n_fields, const pbs4d_field* fields, int64_t n_spots, const pbs4d_spot* spots,
                        const pbs4d_delivery_params* prm, uint64_t total_histories, uint64_t seed,
                        int32_t nsx, int32_t nsy, int32_t nsz, float* dose4d_host, uint64_t* histories_run,
                        uint64_t* h2d_bytes, double* seconds);

/* ---- dose-interpolation method (DIM), the paper's second accumulation method (Eq. 3; "Input
 * options allowed the user to choose both the accumulation method and the voxel-subdivision scale n").
 * DIMs use deformation fields of the opposite direction: T^{R->S} as displacements [3][z][y][x] (mm)
 * at the centres of an axis-aligned grid in the REFERENCE phase frame; copied.  Requires set_ct_phases /
 * set_density_phases first (they define the dose grid). */
int pbs4d_set_dvf_pull(pbs4d_ctx* ctx, int32_t src_phase, int32_t ref_phase, const pbs4d_grid* dvf_grid,
                       const float* disp_dev);

/* Eq. 3 for every source phase that has a T^{R->S} field to ref_phase: each reference voxel is split into
 * nsx*nsy*nsz subvoxels, each centre is mapped to the source phase, the trilinearly interpolated source dose there
 * (0 outside the source grid) is averaged over the subvoxels; then Eq. 2 (sum over phases in ascending order, in
 * double) and the DVF-coverage mask.  Arguments as for accumulate_subvoxel; in stats,
 * dropped_outside_ref counts mapped points outside the source grid, push_ms is the device time of the pull kernels. */
int pbs4d_accumulate_dim(pbs4d_ctx* ctx, int32_t ref_phase, int32_t nsx, int32_t nsy, int32_t nsz,
                         const float* const* phase_dose_dev, float* dose4d_dev, pbs4d_acc_stats* stats);

/* ---- DVF construction (Sec. 2.D.1, App. B, Eq. 7-8) ----
 * The minimal grid information a DICOM deformable spatial registration stores: starting voxel centre, resolutions,
 * row/column direction cosines (depth = row x column), voxel counts, and the rigid pre-/post-deformation matrices
 * (row-major 4x4; identity for registration between 4DCT phases). */
typedef struct {
    int32_t nx, ny, nz, pad;                 /* N_X along the row direction (fastest index), N_Y, N_Z */
    double start[3], delta[3];               /* mm */
    double row_cos[3], col_cos[3];
    double pre[16], post[16];
} pbs4d_dicom_dvf;

/* One thread per deformation-grid voxel: r_0 by Eq. 8, r_f = M_Post (M_Pre r_0 + Delta) by Eq. 7, in double.
 * delta_dev: stored translations [3][k][j][i] fp32.  rf_dev (optional): r_f; disp_dev (optional): r_f - r_0, both fp32
 * [3][k][j][i].  grid_out (optional): when the direction cosines are the coordinate axes (row = +x, column = +y) the
 * axis-aligned grid on which disp_dev can be passed to set_dvf / set_dvf_pull; otherwise PBS4D_ERR_ARG is returned
 * if grid_out is requested (an oblique grid has no pbs4d_grid). */
int pbs4d_build_dvf(pbs4d_ctx* ctx, const pbs4d_dicom_dvf* info, const float* delta_dev, float* rf_dev, float* disp_dev,
                    pbs4d_grid* grid_out);

/* ---- a1 without any allocation ("converting Hounsfield Units to material density") ----
 * For callers that cannot call cudaMalloc: a process whose own memory pool already owns almost all of the GPU (a
 * planning server's caching allocator, PyTorch) has nothing left for an allocation made by a library, and a loop with a
 * latency budget cannot take the driver locks of cudaMalloc or the device-wide wait of cudaFree.  This call needs no
 * context (pbs4d_create allocates) and makes no cudaMalloc, cudaFree or other allocating call, on any invocation.
 *
 *   rho_dev[i] = (float) table(hu_dev[i]),  i < n_voxels;  table = the piecewise-linear function through
 *   (hu_pts[k], rho_pts[k]), clamped at its ends, evaluated in double -- bit for bit what pbs4d_set_ct_phases computes
 *   when dose_grid == NULL (no resampling here).
 *
 * hu_dev (int16, n_voxels), rho_dev (fp32, n_voxels): DEVICE pointers on the calling thread's CURRENT device, caller's
 * buffers, any alignment (16-byte aligned pointers take the vector path).  hu_pts, rho_pts: HOST, n_pts entries, HU
 * strictly ascending, densities > 0; read before the call returns.  cuda_stream: cudaStream_t or NULL.
 * Limits: 2 <= n_pts <= PBS4D_NOALLOC_MAX_TABLE_PTS, 0 <= n_voxels <= PBS4D_NOALLOC_MAX_VOXELS; anything beyond is
 * refused with PBS4D_ERR_ARG before any work is queued (nothing can grow).
 * Scratch: PBS4D_NOALLOC_SCRATCH_BYTES (512 KiB: the table function at each of the 65536 int16 values) in a static
 * device array inside the library; every GPU that loads the library holds it until the process exits.  All calls on a
 * device share it.  Each call rewrites the whole array before reading it, so nothing is carried from call to call and
 * calls queued on ONE stream may follow each other freely; calls that can overlap on the GPU (different streams without
 * an event between them, or several host threads on one device) race on it and give undefined densities.
 * The first call on each device also looks up the scratch's device address (cudaGetSymbolAddress, which loads the
 * module): make that first call before starting any stream capture on that device, e.g. once at start-up with
 * n_voxels = 0.
 * Unlike the context calls this one only ENQUEUES (two kernels on cuda_stream) and returns: the caller synchronises.
 * Errors: the return code, and a message in err[err_cap] (caller's buffer, optional; always terminated, "" on
 * success).  PBS4D_ERR_CUDA without a device -- there is no CPU fallback. */
#define PBS4D_NOALLOC_MAX_TABLE_PTS   64
#define PBS4D_NOALLOC_MAX_VOXELS      2000000000LL
#define PBS4D_NOALLOC_SCRATCH_BYTES   524288
int pbs4d_hu_to_density_noalloc(const int16_t* hu_dev, int64_t n_voxels, int32_t n_pts, const float* hu_pts,
                                const float* rho_pts, float* rho_dev, void* cuda_stream, char* err, int32_t err_cap);

/* In-run roofline probes (BASELINE.json north_star: throughput is reported "as achieved fraction of the FP32-issue,
 * L2-atomic and HBM roofline measured by in-run microbenchmarks").  Each probe launches a small kernel of its own on
 * the context's stream, times it with CUDA events (best of 3-5 after a warm-up) and writes one number to *value:
 *   PBS4D_PROBE_FP32_ISSUE   fp32 FFMA lane-instructions per second (8 independent chains per thread)
 *   PBS4D_PROBE_RED_RANDOM   red.global.add.u64 lane-atomics per second, random addresses in a 32 MB (L2) window
 *   PBS4D_PROBE_RED_HOT      the same with one address per warp (the pencil-beam-core case)
 *   PBS4D_PROBE_HBM_COPY     bytes per second (read + written) of a 1 GiB float4 copy
 * Temporary device memory (up to 2 GiB for the copy) is allocated and freed inside the call. */
#define PBS4D_PROBE_FP32_ISSUE  0
#define PBS4D_PROBE_RED_RANDOM  1
#define PBS4D_PROBE_RED_HOT     2
#define PBS4D_PROBE_HBM_COPY    3
int pbs4d_roofline_probe(pbs4d_ctx* ctx, int32_t kind, double* value);

#ifdef __cplusplus
}
#endif
#endif
