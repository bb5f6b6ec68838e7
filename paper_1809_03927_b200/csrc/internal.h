// Internal declarations shared by the translation units of libpbs4d (not part of the public boundary).
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "pbs4d.h"

#ifdef __CUDACC__
#include <cuda_runtime.h>
#else
typedef struct CUstream_st* cudaStream_t;
#endif

namespace pbs4d {

// ---- host delivery simulator (delivery.cpp) ----
int simulate_delivery_host(const std::vector<pbs4d_field>& fields, const std::vector<pbs4d_spot>& spots,
                           const pbs4d_delivery_params& prm, uint64_t total_histories,
                           std::vector<pbs4d_segment>& segments, std::vector<int64_t>& field_time_ns,
                           int64_t& dropped_protons, std::string& err);
int simulate_delivery_ext_host(const std::vector<pbs4d_field>& fields, const std::vector<pbs4d_spot>& spots,
                               const pbs4d_delivery_params& prm, const pbs4d_delivery_ext& ext,
                               uint64_t total_histories, std::vector<pbs4d_segment>& segments,
                               std::vector<int64_t>& field_time_ns, int64_t& dropped_protons, int64_t& n_fills,
                               std::string& err);
int sample_trial_host(const pbs4d_trial_spec& spec, int32_t trial, int32_t n_fields, const pbs4d_delivery_params& prm,
                      const pbs4d_delivery_ext& ext, int32_t* start_phase, int64_t* cycle_period_ns,
                      int64_t* layer_switch_ns, pbs4d_delivery_params& prm_out, pbs4d_delivery_ext& ext_out);
int32_t fixed_shift_for(const std::vector<pbs4d_segment>& segments, const std::vector<pbs4d_spot>& spots);

// ---- device-side segment record (transport.cu): everything a history needs from its (field, spot) ----
struct DevSegment {
    float dir[3], eu[3], ev[3], ref[3];
    float x_mm, y_mm, energy_mev, sigma_mm;
    float weight_scaled;          // weight * 2^k as float (deposit -> quanta)
    float pad0;
    double weight_scaled_d;       // same in double, for the incident/escaped tallies
    int64_t first_history;        // global Philox history index of local history 0
    int64_t local_begin;          // index of its first history within the phase launch
};

struct TransportCounters {       // device tallies of one launch (zeroed before it)
    unsigned long long histories, steps;
    long long q_incident, q_deposited, q_escaped;
    unsigned long long next_history;      // work counter: next local history index to hand out
    unsigned long long reds;              // scoring atomics issued
    unsigned long long aborted;           // histories stopped by the step cap (hang guard)
};

// Launchers (all asynchronous on `st`).
// hist_begin / n_hist: window of the phase's local history range this launch transports (sharding); phys_tab_dev: the
// context's copy of the physics table (physics_tables.h), physics_table_bytes() bytes.
void launch_transport(const pbs4d_grid& g, const float* rho, const DevSegment* segs, const long long* seg_begin,
                      int32_t n_segs, int64_t hist_begin, int64_t n_hist, uint64_t seed, uint32_t flags,
                      const void* phys_tab_dev, long long* Q, TransportCounters* counters, int sm_count, cudaStream_t st);
const void* transport_kernel_symbol();
size_t physics_table_bytes(void);
void build_physics_table_host(void* nodes /* physics_table_bytes() */);
#ifdef __CUDACC__
cudaError_t configure_transport(void);            // per-device kernel attributes (current device)
cudaError_t configure_accumulate(void);
int launch_validate_density(const float* rho, size_t n, int* flag_dev, cudaStream_t st);
#endif

// lut: 65536 doubles of scratch owned by the caller (the table function per possible HU value; rebuilt by every call);
// rho_first: rho_pts[0], the density of a dose voxel that overlaps no CT voxel
void launch_hu_to_density(const pbs4d_grid& ct, const int16_t* hu, const pbs4d_grid* dose_grid, int32_t n_pts,
                          const float* hu_pts_dev, const float* rho_pts_dev, float rho_first, double* lut,
                          float* rho_out, cudaStream_t st);
void launch_finalize_dose(const pbs4d_grid& g, const float* rho, const long long* Q, int32_t fixed_shift,
                          double per_protons, float* dose, cudaStream_t st);

struct AccCounters { unsigned long long subvoxels, dropped_ref, dropped_dvf; };
// planar [3][z][y][x] displacements -> interleaved float4 {ux, uy, uz, uz of the y-neighbour} per node, followed by one
// float4 record {max|ux|, max|uy|, max|uz|, 0}: out4 holds 4 * nodes + 4 floats (the layout the accumulation kernels read)
void launch_dvf_interleave(const pbs4d_grid& dvf_grid, const float* disp_planar, float* out4, cudaStream_t st);
void launch_emtm_push(const pbs4d_grid& src, const float* dose, const float* rho, const pbs4d_grid& dvf_grid,
                      const float* disp4, const pbs4d_grid& ref, int nsx, int nsy, int nsz,
                      long long* E, long long* M, AccCounters* counters, cudaStream_t st);
// out = (first ? dose_ref : out_acc) ... see accumulate.cu: ratio-and-add over all pushed phases, then mask.
int sm_count_of_current_device(void);
void launch_emtm_finalize(const pbs4d_grid& ref, const float* dose_ref, int n_src, const long long* const* E_dev,
                          const long long* const* M_dev, const pbs4d_grid* dvf_grids_dev,
                          unsigned char* flags_dev /*[nx+ny+nz] scratch*/, float* out, cudaStream_t st);

void launch_dvf_build(const pbs4d_dicom_dvf& g, const float* delta_dev, float* rf_dev, float* disp_dev, cudaStream_t st);

// ---- dose-interpolation method (accumulate.cu) ----
void launch_dim_init(const pbs4d_grid& ref, const float* dose_ref, double* acc, cudaStream_t st);
void launch_dim_pull(const pbs4d_grid& ref, int nsx, int nsy, int nsz, const pbs4d_grid& dvf_grid, const float* disp4,
                     const pbs4d_grid& src, const float* dose_src, double* acc, AccCounters* counters, cudaStream_t st);
void launch_dim_final(const pbs4d_grid& ref, int n_src, const pbs4d_grid* dvf_grids_host, const double* acc,
                      unsigned char* flags_dev, float* out, cudaStream_t st);

// ---- in-run roofline probes (roofline.cu) ----
#ifdef __CUDACC__
cudaError_t probe_fp32_issue(int sm_count, cudaStream_t st, double* lane_inst_per_s);
cudaError_t probe_l2_atomic(int sm_count, int hot, cudaStream_t st, double* lane_atomics_per_s);
cudaError_t probe_hbm_copy(int sm_count, cudaStream_t st, double* bytes_per_s);
#endif

}  // namespace pbs4d
