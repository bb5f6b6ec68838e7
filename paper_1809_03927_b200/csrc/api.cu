// C-ABI boundary of libpbs4d (include/pbs4d.h): context, argument checks, device memory, launch sequencing.
// No arithmetic of the method lives here -- it is in delivery.cpp (host, int64), transport.cu, grids.cu and
// accumulate.cu (device).
#include "internal.h"

#include <cuda_runtime.h>
#include <nvtx3/nvToolsExt.h>

#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <memory>
#include <new>

using namespace pbs4d;

namespace {

struct DevBuf {                          // RAII device allocation
    void* p = nullptr; size_t bytes = 0;
    DevBuf() = default;
    DevBuf(const DevBuf&) = delete; DevBuf& operator=(const DevBuf&) = delete;
    ~DevBuf() { release(); }
    void release() { if (p) cudaFree(p); p = nullptr; bytes = 0; }
    cudaError_t ensure(size_t n) {
        if (n <= bytes && p) return cudaSuccess;
        release();
        cudaError_t e = cudaMalloc(&p, n ? n : 1);
        if (e == cudaSuccess) bytes = n;
        return e;
    }
    template <class T> T* as() const { return static_cast<T*>(p); }
};

struct EventTrio {                       // RAII: three timing events
    cudaEvent_t e[3] = { nullptr, nullptr, nullptr };
    EventTrio() = default;
    EventTrio(const EventTrio&) = delete; EventTrio& operator=(const EventTrio&) = delete;
    cudaError_t create() {
        for (auto& x : e) { cudaError_t rc = cudaEventCreate(&x); if (rc != cudaSuccess) return rc; }
        return cudaSuccess;
    }
    ~EventTrio() { for (auto x : e) if (x) cudaEventDestroy(x); }
};

struct PhaseLaunch {                     // per-phase segment table for the transport kernel
    std::vector<DevSegment> segs;
    std::vector<long long> seg_begin;    // segs[i].local_begin, contiguous for the kernel's binary search
    int64_t n_hist = 0;
    double protons = 0.0;
};

}  // namespace

// layout of pbs4d_ctx::table: hu_pts | rho_pts (at most 64 floats each), then the 65536-double density LUT
constexpr size_t kTableLutOffset = 2 * 64 * sizeof(float);
constexpr size_t kTableBytes = kTableLutOffset + 65536 * sizeof(double);

struct pbs4d_ctx {
    int device = 0;
    int sm_count = 148;
    cudaStream_t stream = nullptr;
    std::string err;

    // geometry + densities (a1)
    bool have_density = false;
    int32_t n_phases = 0;
    pbs4d_grid dose_grid{};
    std::vector<std::unique_ptr<DevBuf>> rho;            // [phase] fp32 on dose grid
    std::vector<bool> rho_valid;                         // [phase] density grid filled (run_plan_host fills active phases only)
    std::vector<cudaEvent_t> rho_ready;                  // [phase] density grid complete on the copy stream (run_plan_host)
    std::vector<bool> rho_pending;                       // [phase] the next transport launch must wait for rho_ready
    DevBuf table;                                        // hu_pts | rho_pts (<= 64 each) | 65536-entry density LUT

    // DVFs (a2)
    struct Dvf { bool set = false; int32_t ref = -1; pbs4d_grid grid{}; std::unique_ptr<DevBuf> disp; };
    std::vector<Dvf> dvf;                                // [src phase] T^{S->R} (push, EMTM)
    std::vector<Dvf> dvf_pull;                           // [src phase] T^{R->S} (pull, DIM)
    DevBuf dim_acc;                                      // double accumulator of the DIM [ref voxels]

    // plan (a2) and delivery (a3)
    std::vector<pbs4d_field> fields;
    std::vector<pbs4d_spot> spots;
    bool have_delivery = false;
    std::vector<pbs4d_segment> segments;
    std::vector<int64_t> field_time;
    int64_t dropped = 0;
    int32_t fixed_shift = 40;
    int32_t deliv_phases = 0;
    std::vector<PhaseLaunch> launches;                   // [phase]
    uint32_t mc_flags = 0;

    // transport state (a4-a7)
    std::vector<std::unique_ptr<DevBuf>> q;              // [phase] int64 energy grid
    std::vector<std::unique_ptr<DevBuf>> dose;           // [phase] fp32 Gy
    std::vector<bool> have_dose;
    DevBuf counters;
    DevBuf phys_tab;                                     // per-energy physics table of the transport kernel (per context)
    int32_t shard_rank = 0, shard_world = 1;             // history sharding (pbs4d_set_shard)
    std::vector<std::unique_ptr<DevBuf>> seg_phase;      // [phase] launch table (DevSegment[] | seg_begin[])
    std::vector<bool> seg_resident;                      // [phase] launch table of the current delivery is on the device
    std::vector<cudaStream_t> aux;                       // auxiliary streams for concurrent phase launches
    cudaStream_t copy_stream = nullptr;                  // uploads that overlap compute (run_plan_host): DMA only
    cudaStream_t prep_stream = nullptr;                  // HU -> density and DVF re-layout kernels behind the uploads
    std::vector<cudaEvent_t> upload_done;                // [2 * phase + {0: CT, 1: DVF}] copy finished on copy_stream

    // accumulation state (a8-a9)
    std::vector<std::unique_ptr<DevBuf>> accE, accM;     // [phase]
    std::vector<bool> have_acc;
    DevBuf acc_counters, cover_flags;
    DevBuf host_hu, host_dvf, host_out;                  // staging buffers of run_plan_host, kept across calls

    size_t nvox() const { return (size_t)dose_grid.nx * dose_grid.ny * dose_grid.nz; }
};

namespace {

int fail(pbs4d_ctx* c, int code, const std::string& msg)
{
    if (c) c->err = msg;
    return code;
}

int cuda_fail(pbs4d_ctx* c, cudaError_t e, const char* what)
{
    return fail(c, e == cudaErrorMemoryAllocation ? PBS4D_ERR_NOMEM : PBS4D_ERR_CUDA,
                std::string(what) + ": " + cudaGetErrorString(e));
}

// Nothing may throw across the C boundary: every extern "C" entry point is a function-try-block ending here.
int on_exception(pbs4d_ctx* c) noexcept
{
    try { throw; }
    catch (const std::bad_alloc&) {
        try { if (c) c->err = "out of host memory"; } catch (...) {}
        return PBS4D_ERR_NOMEM;
    }
    catch (...) {
        try { if (c) c->err = "unexpected C++ exception"; } catch (...) {}
        return PBS4D_ERR_ARG;
    }
}

#define CU(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return cuda_fail(ctx, e_, #call); } while (0)

// One NVTX range per API call (tracing): a timeline or launch list taken with Nsight tools shows
// which pbs4d_* call every kernel and copy belongs to (the paper reports its times per component, PAPER.md:187-195
// Table II).  Header-only NVTX 3: without a tool attached a push / pop is a load and a branch.
struct NvtxRange {
    explicit NvtxRange(const char* name) { nvtxRangePushA(name); }
    ~NvtxRange() { nvtxRangePop(); }
    NvtxRange(const NvtxRange&) = delete;
    NvtxRange& operator=(const NvtxRange&) = delete;
};

// nullptr for a usable grid, else what is wrong with it.  The per-axis limits are those of the launch geometry: the
// accumulation kernels put ceil(ny / 4) CTAs on grid.y and ceil(nz / 4) on grid.z, the resampling density kernel nz on
// grid.z (each at most 65535), and rows (ny * nz) go on grid.x, which the total bounds.
const char* grid_defect(const pbs4d_grid* g)
{
    if (!g) return "null grid";
    if (!(g->nx > 0 && g->ny > 0 && g->nz > 0)) return "grid needs at least one voxel per axis";
    if (!(g->hx > 0.0f && g->hy > 0.0f && g->hz > 0.0f) || !std::isfinite(g->hx) || !std::isfinite(g->hy) ||
        !std::isfinite(g->hz))
        return "grid spacings must be positive and finite";
    if (!std::isfinite(g->ox) || !std::isfinite(g->oy) || !std::isfinite(g->oz)) return "grid origin must be finite";
    if (g->nx > 4000000 || g->ny > 262140 || g->nz > 65535)
        return "grid too long: at most 4000000 x 262140 x 65535 voxels (x, y, z)";
    if (!((double)g->nx * g->ny * g->nz < 2.0e9)) return "grid too large: fewer than 2e9 voxels in total";
    return nullptr;
}

bool grid_ok(const pbs4d_grid* g) { return grid_defect(g) == nullptr; }

void reset_phase_state(pbs4d_ctx* ctx, int32_t n_phases, const pbs4d_grid& g)
{
    // device buffers are kept across calls (DevBuf::ensure reuses an allocation that is large enough): a plan that
    // is recomputed on the same grids costs no cudaMalloc/cudaFree
    ctx->n_phases = n_phases; ctx->dose_grid = g;
    auto fit = [&](std::vector<std::unique_ptr<DevBuf>>& v) {
        v.resize(n_phases);
        for (auto& b : v) if (!b) b.reset(new DevBuf);
    };
    fit(ctx->rho); fit(ctx->q); fit(ctx->dose); fit(ctx->accE); fit(ctx->accM);
    ctx->dvf.resize(n_phases);
    for (auto& d : ctx->dvf) { d.set = false; d.ref = -1; }
    ctx->dvf_pull.resize(n_phases);
    for (auto& d : ctx->dvf_pull) { d.set = false; d.ref = -1; }
    ctx->have_dose.assign(n_phases, false);
    ctx->have_acc.assign(n_phases, false);
    ctx->rho_valid.assign(n_phases, false);
    ctx->rho_pending.assign(n_phases, false);
    ctx->have_density = false;
}

}  // namespace

extern "C" {

int pbs4d_create(pbs4d_ctx** out, int device, void* cuda_stream) try
{
    const NvtxRange nvtx_range_("pbs4d_create");
    if (!out) return PBS4D_ERR_ARG;
    *out = nullptr;
    int n_dev = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || device < 0 || device >= n_dev) return PBS4D_ERR_CUDA;
    if (cudaSetDevice(device) != cudaSuccess) return PBS4D_ERR_CUDA;
    pbs4d_ctx* ctx = new (std::nothrow) pbs4d_ctx;
    if (!ctx) return PBS4D_ERR_NOMEM;
    ctx->device = device;
    ctx->stream = static_cast<cudaStream_t>(cuda_stream);
    int sms = 0;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device) == cudaSuccess && sms > 0) ctx->sm_count = sms;
    // per-context physics table and per-device kernel attributes: uploaded / set here, checked, and ordered before
    // any launch (the copy is synchronised; the launches of every stream come later)
    std::vector<char> host_tab(physics_table_bytes());
    build_physics_table_host(host_tab.data());
    cudaError_t e = ctx->phys_tab.ensure(host_tab.size());
    if (e == cudaSuccess) e = cudaMemcpy(ctx->phys_tab.p, host_tab.data(), host_tab.size(), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    if (e == cudaSuccess) e = configure_transport();
    if (e == cudaSuccess) e = configure_accumulate();
    if (e != cudaSuccess) { delete ctx; return e == cudaErrorMemoryAllocation ? PBS4D_ERR_NOMEM : PBS4D_ERR_CUDA; }
    *out = ctx;
    return PBS4D_OK;
}
catch (...) { return on_exception(nullptr); }

void pbs4d_destroy(pbs4d_ctx* ctx) try
{
    if (!ctx) return;
    cudaSetDevice(ctx->device);
    cudaStreamSynchronize(ctx->stream);
    for (auto st : ctx->aux) if (st) cudaStreamDestroy(st);
    for (auto e : ctx->rho_ready) if (e) cudaEventDestroy(e);
    if (ctx->copy_stream) { cudaStreamSynchronize(ctx->copy_stream); cudaStreamDestroy(ctx->copy_stream); }
    if (ctx->prep_stream) { cudaStreamSynchronize(ctx->prep_stream); cudaStreamDestroy(ctx->prep_stream); }
    for (auto e : ctx->upload_done) if (e) cudaEventDestroy(e);
    delete ctx;
}
catch (...) {}

const char* pbs4d_last_error(const pbs4d_ctx* ctx) { return ctx ? ctx->err.c_str() : "null context"; }

int pbs4d_set_ct_phases(pbs4d_ctx* ctx, int32_t n_phases, const pbs4d_grid* ct, const int16_t* const* hu_dev,
                        const pbs4d_grid* dose_grid, int32_t n_pts, const float* hu_pts, const float* rho_pts) try
{
    const NvtxRange nvtx_range_("pbs4d_set_ct_phases");
    if (!ctx) return PBS4D_ERR_ARG;
    if (const char* why = grid_defect(ct)) return fail(ctx, PBS4D_ERR_ARG, std::string("set_ct_phases: ct: ") + why);
    if (dose_grid) if (const char* why = grid_defect(dose_grid)) return fail(ctx, PBS4D_ERR_ARG, std::string("set_ct_phases: dose_grid: ") + why);
    if (n_phases < 1 || n_phases > 32 || !hu_dev || n_pts < 2 || n_pts > 64 || !hu_pts || !rho_pts)
        return fail(ctx, PBS4D_ERR_ARG, "set_ct_phases: bad argument");
    for (int i = 0; i < n_pts; ++i) {
        if (!(rho_pts[i] > 0.0f) || (i && !(hu_pts[i] > hu_pts[i - 1])))
            return fail(ctx, PBS4D_ERR_ARG, "set_ct_phases: table must ascend in HU with positive densities");
    }
    for (int p = 0; p < n_phases; ++p) if (!hu_dev[p]) return fail(ctx, PBS4D_ERR_ARG, "set_ct_phases: null phase");
    CU(cudaSetDevice(ctx->device));
    const pbs4d_grid& g = dose_grid ? *dose_grid : *ct;
    reset_phase_state(ctx, n_phases, g);
    CU(ctx->table.ensure(kTableBytes));
    CU(cudaMemcpyAsync(ctx->table.p, hu_pts, n_pts * sizeof(float), cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaMemcpyAsync(ctx->table.as<float>() + n_pts, rho_pts, n_pts * sizeof(float), cudaMemcpyHostToDevice,
                       ctx->stream));
    for (int p = 0; p < n_phases; ++p) {
        CU(ctx->rho[p]->ensure(ctx->nvox() * sizeof(float)));
        launch_hu_to_density(*ct, hu_dev[p], dose_grid, n_pts, ctx->table.as<float>(), ctx->table.as<float>() + n_pts,
                             rho_pts[0], reinterpret_cast<double*>(ctx->table.as<char>() + kTableLutOffset),
                             ctx->rho[p]->as<float>(), ctx->stream);
    }
    CU(cudaGetLastError());
    CU(cudaStreamSynchronize(ctx->stream));
    ctx->rho_valid.assign(n_phases, true);
    ctx->have_density = true;
    return PBS4D_OK;
}
catch (...) { return on_exception(ctx); }

int pbs4d_set_density_phases(pbs4d_ctx* ctx, int32_t n_phases, const pbs4d_grid* dose_grid,
                             const float* const* rho_dev) try
{
    const NvtxRange nvtx_range_("pbs4d_set_density_phases");
    if (!ctx) return PBS4D_ERR_ARG;
    if (const char* why = grid_defect(dose_grid)) return fail(ctx, PBS4D_ERR_ARG, std::string("set_density_phases: ") + why);
    if (n_phases < 1 || n_phases > 32 || !rho_dev)
        return fail(ctx, PBS4D_ERR_ARG, "set_density_phases: bad argument");
    for (int p = 0; p < n_phases; ++p) if (!rho_dev[p]) return fail(ctx, PBS4D_ERR_ARG, "set_density_phases: null phase");
    CU(cudaSetDevice(ctx->device));
    reset_phase_state(ctx, n_phases, *dose_grid);
    CU(ctx->counters.ensure(sizeof(TransportCounters) * 32));
    int* bad_dev = ctx->counters.as<int>();               // scratch word for the validation kernel
    CU(cudaMemsetAsync(bad_dev, 0, sizeof(int), ctx->stream));
    for (int p = 0; p < n_phases; ++p) {
        CU(ctx->rho[p]->ensure(ctx->nvox() * sizeof(float)));
        CU(cudaMemcpyAsync(ctx->rho[p]->p, rho_dev[p], ctx->nvox() * sizeof(float), cudaMemcpyDeviceToDevice,
                           ctx->stream));
        launch_validate_density(ctx->rho[p]->as<float>(), ctx->nvox(), bad_dev, ctx->stream);
    }
    int bad = 0;
    CU(cudaGetLastError());
    CU(cudaMemcpyAsync(&bad, bad_dev, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    if (bad) return fail(ctx, PBS4D_ERR_ARG, "set_density_phases: densities must be finite and within [1e-6, 100] g/cm3");
    ctx->rho_valid.assign(n_phases, true);
    ctx->have_density = true;
    return PBS4D_OK;
}
catch (...) { return on_exception(ctx); }

static int store_dvf(pbs4d_ctx* ctx, std::vector<pbs4d_ctx::Dvf>& table, const char* who, int32_t src_phase,
                     int32_t ref_phase, const pbs4d_grid* dvf_grid, const float* disp_dev)
{
    if (!ctx) return PBS4D_ERR_ARG;
    if (!ctx->have_density) return fail(ctx, PBS4D_ERR_ORDER, std::string(who) + ": call set_ct_phases/set_density_phases first");
    if (src_phase < 0 || src_phase >= ctx->n_phases || ref_phase < 0 || ref_phase >= ctx->n_phases ||
        src_phase == ref_phase || !disp_dev)
        return fail(ctx, PBS4D_ERR_ARG, std::string(who) + ": bad argument");
    if (const char* why = grid_defect(dvf_grid)) return fail(ctx, PBS4D_ERR_ARG, std::string(who) + ": dvf_grid: " + why);
    CU(cudaSetDevice(ctx->device));
    auto& d = table[src_phase];
    if (!d.disp) d.disp.reset(new DevBuf);
    const size_t bytes = ((size_t)4 * dvf_grid->nx * dvf_grid->ny * dvf_grid->nz + 4) * sizeof(float);   // + max |u| record
    CU(d.disp->ensure(bytes));
    launch_dvf_interleave(*dvf_grid, disp_dev, d.disp->as<float>(), ctx->stream);
    CU(cudaGetLastError());
    CU(cudaStreamSynchronize(ctx->stream));
    d.set = true; d.ref = ref_phase; d.grid = *dvf_grid;
    return PBS4D_OK;
}

int pbs4d_set_dvf(pbs4d_ctx* ctx, int32_t src_phase, int32_t ref_phase, const pbs4d_grid* dvf_grid,
                  const float* disp_dev) try
{
    const NvtxRange nvtx_range_("pbs4d_set_dvf");
    if (!ctx) return PBS4D_ERR_ARG;
    return store_dvf(ctx, ctx->dvf, "set_dvf", src_phase, ref_phase, dvf_grid, disp_dev);
}
catch (...) { return on_exception(ctx); }

int pbs4d_set_dvf_pull(pbs4d_ctx* ctx, int32_t src_phase, int32_t ref_phase, const pbs4d_grid* dvf_grid,
                       const float* disp_dev) try
{
    const NvtxRange nvtx_range_("pbs4d_set_dvf_pull");
    if (!ctx) return PBS4D_ERR_ARG;
    return store_dvf(ctx, ctx->dvf_pull, "set_dvf_pull", src_phase, ref_phase, dvf_grid, disp_dev);
}
catch (...) { return on_exception(ctx); }

int pbs4d_set_plan_spots(pbs4d_ctx* ctx, int32_t n_fields, const pbs4d_field* fields,
                         int64_t n_spots, const pbs4d_spot* spots) try
{
    const NvtxRange nvtx_range_("pbs4d_set_plan_spots");
    if (!ctx) return PBS4D_ERR_ARG;
    if (n_fields < 1 || !fields || n_spots < 1 || !spots) return fail(ctx, PBS4D_ERR_ARG, "set_plan_spots: bad argument");
    for (int64_t s = 0; s < n_spots; ++s) {
        const pbs4d_spot& sp = spots[s];
        if (sp.field < 0 || sp.field >= n_fields || !(sp.energy_mev > 0.5f) || !(sp.energy_mev < 500.0f) ||
            !(sp.sigma_mm >= 0.0f) || !(sp.weight >= 0.0f) || !std::isfinite(sp.x_mm) || !std::isfinite(sp.y_mm))
            return fail(ctx, PBS4D_ERR_ARG, "set_plan_spots: bad spot " + std::to_string(s));
    }
    for (int32_t f = 0; f < n_fields; ++f) {
        const float* d = fields[f].dir;
        const float n2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
        if (!(std::fabs(n2 - 1.0f) < 1e-3f) || fields[f].start_phase < 0)
            return fail(ctx, PBS4D_ERR_ARG, "set_plan_spots: field direction must be a unit vector, start_phase >= 0");
    }
    ctx->fields.assign(fields, fields + n_fields);
    ctx->spots.assign(spots, spots + n_spots);
    ctx->have_delivery = false;
    return PBS4D_OK;
}
catch (...) { return on_exception(ctx); }

int pbs4d_set_mc_flags(pbs4d_ctx* ctx, uint32_t flags) try
{
    const NvtxRange nvtx_range_("pbs4d_set_mc_flags");
    if (!ctx) return PBS4D_ERR_ARG;
    ctx->mc_flags = flags;
    return PBS4D_OK;
}
catch (...) { return on_exception(ctx); }

}  // extern "C"

// ------------------------------------------------------------------------------------------------------------------
// a3: delivery simulation (host) and per-phase launch tables
// ------------------------------------------------------------------------------------------------------------------
extern "C" int pbs4d_simulate_delivery_ext(pbs4d_ctx* ctx, const pbs4d_delivery_params* prm,
                                           const pbs4d_delivery_ext* ext, uint64_t total_histories,
                                           pbs4d_phase_lists* out, int64_t* n_fills);

extern "C" int pbs4d_simulate_delivery(pbs4d_ctx* ctx, const pbs4d_delivery_params* prm, uint64_t total_histories,
                                       pbs4d_phase_lists* out) try
{
    const NvtxRange nvtx_range_("pbs4d_simulate_delivery");
    return pbs4d_simulate_delivery_ext(ctx, prm, nullptr, total_histories, out, nullptr);
}
catch (...) { return on_exception(ctx); }

// ext == NULL: the base simulator; else the extended model.  Both end in the same per-phase launch tables.
extern "C" int pbs4d_simulate_delivery_ext(pbs4d_ctx* ctx, const pbs4d_delivery_params* prm,
                                           const pbs4d_delivery_ext* ext, uint64_t total_histories,
                                           pbs4d_phase_lists* out, int64_t* n_fills) try
{
    const NvtxRange nvtx_range_("pbs4d_simulate_delivery_ext");
    if (!ctx) return PBS4D_ERR_ARG;
    if (!prm) return fail(ctx, PBS4D_ERR_ARG, "simulate_delivery: null parameters");
    if (ctx->fields.empty()) return fail(ctx, PBS4D_ERR_ORDER, "simulate_delivery: call set_plan_spots first");
    if (total_histories > (uint64_t)1 << 62) return fail(ctx, PBS4D_ERR_ARG, "simulate_delivery: too many histories");
    std::string err;
    int rc;
    if (ext) {
        int64_t fills = 0;
        rc = simulate_delivery_ext_host(ctx->fields, ctx->spots, *prm, *ext, total_histories, ctx->segments,
                                        ctx->field_time, ctx->dropped, fills, err);
        if (n_fills) *n_fills = fills;
    } else {
        rc = simulate_delivery_host(ctx->fields, ctx->spots, *prm, total_histories, ctx->segments, ctx->field_time,
                                    ctx->dropped, err);
    }
    if (rc != PBS4D_OK) return fail(ctx, rc, "simulate_delivery: " + err);
    ctx->fixed_shift = fixed_shift_for(ctx->segments, ctx->spots);
    ctx->deliv_phases = prm->n_phases;

    // overflow guard: total quanta of the plan must stay below 2^62
    double tot = 0.0;
    for (const auto& sg : ctx->segments) tot += (double)sg.protons * (double)ctx->spots[sg.spot].energy_mev;
    if (std::ldexp(tot * 1.1, ctx->fixed_shift) > 4611686018427387904.0)
        return fail(ctx, PBS4D_ERR_OVERFLOW, "simulate_delivery: plan energy does not fit the fixed-point range");

    // per-phase launch tables: one DevSegment per segment with histories, local_begin = running history count
    ctx->launches.assign(prm->n_phases, PhaseLaunch{});
    const double scale = std::ldexp(1.0, ctx->fixed_shift);
    for (const auto& sg : ctx->segments) {
        PhaseLaunch& L = ctx->launches[sg.phase];
        L.protons += (double)sg.protons;
        if (sg.n_hist <= 0) continue;
        const pbs4d_field& f = ctx->fields[sg.field];
        const pbs4d_spot&  s = ctx->spots[sg.spot];
        DevSegment d{};
        for (int k = 0; k < 3; ++k) { d.dir[k] = f.dir[k]; d.eu[k] = f.eu[k]; d.ev[k] = f.ev[k]; d.ref[k] = f.ref[k]; }
        d.x_mm = s.x_mm; d.y_mm = s.y_mm; d.energy_mev = s.energy_mev; d.sigma_mm = s.sigma_mm;
        d.weight_scaled_d = sg.weight * scale;
        d.weight_scaled   = (float)d.weight_scaled_d;
        d.first_history   = sg.first_history;
        d.local_begin     = L.n_hist;
        L.segs.push_back(d);
        L.seg_begin.push_back(d.local_begin);
        L.n_hist += sg.n_hist;
    }
    ctx->have_delivery = true;
    std::fill(ctx->seg_resident.begin(), ctx->seg_resident.end(), false);
    std::fill(ctx->have_dose.begin(), ctx->have_dose.end(), false);
    if (out) {
        out->n_segments = (int64_t)ctx->segments.size();
        out->segments = ctx->segments.data();
        out->n_fields = (int32_t)ctx->field_time.size();
        out->field_time_ns = ctx->field_time.data();
        out->dropped_protons = ctx->dropped;
        out->fixed_shift = ctx->fixed_shift;
    }
    return PBS4D_OK;
}
catch (...) { return on_exception(ctx); }

// ------------------------------------------------------------------------------------------------------------------
// a4-a7: transport + scoring + finalize for one phase
// ------------------------------------------------------------------------------------------------------------------
namespace {
constexpr int kAuxStreams = 4;

// per-phase launch table -> device (once per delivery simulation).  The tables live in pageable host memory, so the
// copy goes through the H2D copy engine's queue: run_plan_host issues all of them BEFORE its bulk uploads, otherwise a
// few KB needed by the first transport launch would wait behind gigabytes of CT and DVF traffic.
int upload_segments(pbs4d_ctx* ctx, int phase, cudaStream_t st)
{
    const size_t np = ctx->launches.size();
    if (ctx->seg_phase.size() < np) ctx->seg_phase.resize(np);
    for (auto& b : ctx->seg_phase) if (!b) b.reset(new DevBuf);
    if (ctx->seg_resident.size() < np) ctx->seg_resident.resize(np, false);
    PhaseLaunch& L = ctx->launches[phase];
    if (ctx->seg_resident[phase] || L.n_hist <= 0) return PBS4D_OK;
    DevBuf& sb = *ctx->seg_phase[phase];
    const size_t seg_bytes = L.segs.size() * sizeof(DevSegment);
    CU(sb.ensure(seg_bytes + L.segs.size() * sizeof(long long)));
    CU(cudaMemcpyAsync(sb.p, L.segs.data(), seg_bytes, cudaMemcpyHostToDevice, st));
    CU(cudaMemcpyAsync(sb.as<char>() + seg_bytes, L.seg_begin.data(), L.segs.size() * sizeof(long long),
                       cudaMemcpyHostToDevice, st));
    ctx->seg_resident[phase] = true;
    return PBS4D_OK;
}
}

extern "C" int pbs4d_mc_dose_phases(pbs4d_ctx* ctx, int32_t n, const int32_t* phases, uint64_t seed, double per_protons,
                                    pbs4d_mc_stats* stats, float* elapsed_ms) try
{
    const NvtxRange nvtx_range_("pbs4d_mc_dose_phases");
    if (!ctx) return PBS4D_ERR_ARG;
    if (!ctx->have_density) return fail(ctx, PBS4D_ERR_ORDER, "mc_dose_phases: no densities (set_ct_phases)");
    if (!ctx->have_delivery) return fail(ctx, PBS4D_ERR_ORDER, "mc_dose_phases: call simulate_delivery first");
    if (n < 1 || n > 32 || !phases) return fail(ctx, PBS4D_ERR_ARG, "mc_dose_phases: bad argument");
    for (int a = 0; a < n; ++a) {
        if (phases[a] < 0 || phases[a] >= ctx->n_phases || phases[a] >= ctx->deliv_phases)
            return fail(ctx, PBS4D_ERR_ARG, "mc_dose_phases: phase out of range");
        if (!ctx->rho_valid[phases[a]]) return fail(ctx, PBS4D_ERR_ORDER, "mc_dose_phases: no density grid for this phase");
        for (int b = 0; b < a; ++b)
            if (phases[b] == phases[a]) return fail(ctx, PBS4D_ERR_ARG, "mc_dose_phases: phase listed twice");
    }
    CU(cudaSetDevice(ctx->device));
    const size_t nvox = ctx->nvox();
    // streams: one launch alone runs on the context's stream; several run on auxiliary streams between a fork and a
    // join event so that the tail of one phase's persistent kernel overlaps the start of the next
    const bool fan_out = n > 1;
    if (fan_out && ctx->aux.empty()) {
        ctx->aux.resize(kAuxStreams, nullptr);
        for (auto& st : ctx->aux) CU(cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking));
    }
    for (int a = 0; a < n; ++a) {                        // launch tables (no-op when run_plan_host uploaded them already)
        const int urc = upload_segments(ctx, phases[a], ctx->stream);
        if (urc != PBS4D_OK) return urc;
    }
    CU(ctx->counters.ensure(sizeof(TransportCounters) * 32));
    CU(cudaMemsetAsync(ctx->counters.p, 0, sizeof(TransportCounters) * n, ctx->stream));
    std::vector<cudaEvent_t> ev(2 * n + 2 + kAuxStreams, nullptr);
    auto destroy_events = [&] { for (auto e : ev) if (e) cudaEventDestroy(e); };
    for (auto& e : ev) {
        cudaError_t ce = cudaEventCreate(&e);
        if (ce != cudaSuccess) { destroy_events(); return cuda_fail(ctx, ce, "cudaEventCreate"); }
    }
    cudaEvent_t span0 = ev[2 * n], span1 = ev[2 * n + 1];
    int rc = PBS4D_OK;
    auto guard = [&](cudaError_t ce, const char* what) { if (ce != cudaSuccess && rc == PBS4D_OK) rc = cuda_fail(ctx, ce, what); };
    guard(cudaEventRecord(span0, ctx->stream), "record");
    if (fan_out) for (auto st : ctx->aux) guard(cudaStreamWaitEvent(st, span0, 0), "fork");
    for (int a = 0; a < n && rc == PBS4D_OK; ++a) {
        const int phase = phases[a];
        cudaStream_t st = fan_out ? ctx->aux[a % kAuxStreams] : ctx->stream;
        PhaseLaunch& L = ctx->launches[phase];
        guard(ctx->q[phase]->ensure(nvox * sizeof(long long)), "alloc energy grid");
        guard(ctx->dose[phase]->ensure(nvox * sizeof(float)), "alloc dose grid");
        if (rc != PBS4D_OK) break;
        guard(cudaMemsetAsync(ctx->q[phase]->p, 0, nvox * sizeof(long long), st), "memset");
        if (ctx->rho_pending[phase]) {                   // density still being produced on the copy stream
            guard(cudaStreamWaitEvent(st, ctx->rho_ready[phase], 0), "wait for density");
            ctx->rho_pending[phase] = false;
        }
        guard(cudaEventRecord(ev[2 * a], st), "record");
        if (L.n_hist > 0) {
            DevBuf& sb = *ctx->seg_phase[phase];          // uploaded on the context's stream before the fork
            const size_t seg_bytes = L.segs.size() * sizeof(DevSegment);
            int64_t h0 = 0, hn = 0;
            pbs4d_shard_window(L.n_hist, ctx->shard_rank, ctx->shard_world, &h0, &hn);
            if (hn > 0)
                launch_transport(ctx->dose_grid, ctx->rho[phase]->as<float>(), sb.as<DevSegment>(),
                                 reinterpret_cast<const long long*>(sb.as<char>() + seg_bytes), (int32_t)L.segs.size(),
                                 h0, hn, seed, ctx->mc_flags, ctx->phys_tab.p, ctx->q[phase]->as<long long>(),
                                 ctx->counters.as<TransportCounters>() + a, ctx->sm_count, st);
        }
        guard(cudaEventRecord(ev[2 * a + 1], st), "record");
        launch_finalize_dose(ctx->dose_grid, ctx->rho[phase]->as<float>(), ctx->q[phase]->as<long long>(),
                             ctx->fixed_shift, per_protons, ctx->dose[phase]->as<float>(), st);
        guard(cudaGetLastError(), "launch");
    }
    if (fan_out) {
        for (int k = 0; k < kAuxStreams; ++k) {
            guard(cudaEventRecord(ev[2 * n + 2 + k], ctx->aux[k]), "record");
            guard(cudaStreamWaitEvent(ctx->stream, ev[2 * n + 2 + k], 0), "join");
        }
    }
    guard(cudaEventRecord(span1, ctx->stream), "record");
    std::vector<TransportCounters> tc(n);
    guard(cudaMemcpyAsync(tc.data(), ctx->counters.p, sizeof(TransportCounters) * n, cudaMemcpyDeviceToHost, ctx->stream),
          "counters D2H");
    guard(cudaStreamSynchronize(ctx->stream), "synchronize");
    if (rc == PBS4D_OK) {
        for (int a = 0; a < n; ++a) {
            ctx->have_dose[phases[a]] = true;
            if (!stats) continue;
            pbs4d_mc_stats& s = stats[a];
            s.histories = tc[a].histories; s.steps = tc[a].steps;
            s.q_incident = tc[a].q_incident; s.q_deposited = tc[a].q_deposited; s.q_escaped = tc[a].q_escaped;
            s.fixed_shift = ctx->fixed_shift; s.pad = 0; s.scoring_atomics = tc[a].reds;
            s.aborted = (int32_t)std::min<unsigned long long>(tc[a].aborted, 0x7fffffffull);
            s.kernel_ms = 0.0f;
            cudaEventElapsedTime(&s.kernel_ms, ev[2 * a], ev[2 * a + 1]);
        }
        if (elapsed_ms) cudaEventElapsedTime(elapsed_ms, span0, span1);
    }
    destroy_events();
    return rc;
}
catch (...) { return on_exception(ctx); }

extern "C" int pbs4d_mc_dose_phase(pbs4d_ctx* ctx, int32_t phase, uint64_t seed, double per_protons,
                                   float* dose_dev, float* rho_dev, pbs4d_mc_stats* stats) try
{
    const NvtxRange nvtx_range_("pbs4d_mc_dose_phase");
    if (!ctx) return PBS4D_ERR_ARG;
    const int rc = pbs4d_mc_dose_phases(ctx, 1, &phase, seed, per_protons, stats, nullptr);
    if (rc != PBS4D_OK) return rc;
    const size_t nvox = ctx->nvox();
    if (dose_dev) CU(cudaMemcpyAsync(dose_dev, ctx->dose[phase]->p, nvox * sizeof(float), cudaMemcpyDeviceToDevice, ctx->stream));
    if (rho_dev)  CU(cudaMemcpyAsync(rho_dev, ctx->rho[phase]->p, nvox * sizeof(float), cudaMemcpyDeviceToDevice, ctx->stream));
    if (dose_dev || rho_dev) CU(cudaStreamSynchronize(ctx->stream));
    return PBS4D_OK;
}
catch (...) { return on_exception(ctx); }

extern "C" int pbs4d_get_phase_energy(pbs4d_ctx* ctx, int32_t phase, int64_t* q_dev) try
{
    const NvtxRange nvtx_range_("pbs4d_get_phase_energy");
    if (!ctx) return PBS4D_ERR_ARG;
    if (phase < 0 || phase >= ctx->n_phases || !q_dev) return fail(ctx, PBS4D_ERR_ARG, "get_phase_energy: bad argument");
    if (!ctx->have_dose[phase]) return fail(ctx, PBS4D_ERR_ORDER, "get_phase_energy: mc_dose_phase not run for this phase");
    CU(cudaSetDevice(ctx->device));
    CU(cudaMemcpyAsync(q_dev, ctx->q[phase]->p, ctx->nvox() * sizeof(long long), cudaMemcpyDeviceToDevice, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    return PBS4D_OK;
}
catch (...) { return on_exception(ctx); }

// ------------------------------------------------------------------------------------------------------------------
// multi-GPU history sharding (the MC was distributed amongst eight GPUs).
// Histories are independent units with one Philox counter each, so a rank transports a contiguous slice of every
// phase's history range; the int64 energy grids of the ranks add up to the unsharded grid bit for bit.
// ------------------------------------------------------------------------------------------------------------------
extern "C" int pbs4d_shard_window(int64_t n_hist, int32_t rank, int32_t world, int64_t* begin, int64_t* count)
{
    if (n_hist < 0 || world < 1 || rank < 0 || rank >= world || !begin || !count) return PBS4D_ERR_ARG;
    const int64_t b = (int64_t)(((__int128)n_hist * rank) / world);
    const int64_t e = (int64_t)(((__int128)n_hist * (rank + 1)) / world);
    *begin = b; *count = e - b;
    return PBS4D_OK;
}

extern "C" int pbs4d_set_shard(pbs4d_ctx* ctx, int32_t rank, int32_t world) try
{
    const NvtxRange nvtx_range_("pbs4d_set_shard");
    if (!ctx) return PBS4D_ERR_ARG;
    if (world < 1 || rank < 0 || rank >= world) return fail(ctx, PBS4D_ERR_ARG, "set_shard: need 0 <= rank < world");
    ctx->shard_rank = rank; ctx->shard_world = world;      // affects the mc_dose_phase(s) calls that follow only
    return PBS4D_OK;
}
catch (...) { return on_exception(ctx); }

extern "C" int pbs4d_phase_energy_ptr(pbs4d_ctx* ctx, int32_t phase, int64_t** q_dev) try
{
    const NvtxRange nvtx_range_("pbs4d_phase_energy_ptr");
    if (!ctx) return PBS4D_ERR_ARG;
    if (phase < 0 || phase >= ctx->n_phases || !q_dev) return fail(ctx, PBS4D_ERR_ARG, "phase_energy_ptr: bad argument");
    if (!ctx->have_dose[phase]) return fail(ctx, PBS4D_ERR_ORDER, "phase_energy_ptr: mc_dose_phase not run for this phase");
    *q_dev = ctx->q[phase]->as<int64_t>();
    return PBS4D_OK;
}
catch (...) { return on_exception(ctx); }

extern "C" int pbs4d_finalize_phase_dose(pbs4d_ctx* ctx, int32_t phase, double per_protons) try
{
    const NvtxRange nvtx_range_("pbs4d_finalize_phase_dose");
    if (!ctx) return PBS4D_ERR_ARG;
    if (phase < 0 || phase >= ctx->n_phases) return fail(ctx, PBS4D_ERR_ARG, "finalize_phase_dose: bad argument");
    if (!ctx->have_dose[phase]) return fail(ctx, PBS4D_ERR_ORDER, "finalize_phase_dose: mc_dose_phase not run for this phase");
    CU(cudaSetDevice(ctx->device));
    launch_finalize_dose(ctx->dose_grid, ctx->rho[phase]->as<float>(), ctx->q[phase]->as<long long>(), ctx->fixed_shift,
                         per_protons, ctx->dose[phase]->as<float>(), ctx->stream);
    CU(cudaGetLastError());
    CU(cudaStreamSynchronize(ctx->stream));
    return PBS4D_OK;
}
catch (...) { return on_exception(ctx); }

// ------------------------------------------------------------------------------------------------------------------
// a8-a9: subvoxel energy/mass push of every source phase with a DVF to ref_phase, then ratio + sum + mask
// ------------------------------------------------------------------------------------------------------------------
namespace {

// push (a8) of the source phases selected by src_mask and / or finalize (a9) over every eligible source phase.
// Eligible = has a DVF to ref_phase and a dose.  Eligible phases outside src_mask get zeroed accumulators (ready to
// receive another rank's sums, pbs4d_accumulator_ptrs).
int accumulate_impl(pbs4d_ctx* ctx, const char* who, int32_t ref_phase, int32_t nsx, int32_t nsy, int32_t nsz,
                    const float* const* phase_dose_dev, uint32_t src_mask, bool do_push, bool do_finalize,
                    float* dose4d_dev, pbs4d_acc_stats* stats)
{
    if (!ctx->have_density) return fail(ctx, PBS4D_ERR_ORDER, std::string(who) + ": no densities");
    if (ref_phase < 0 || ref_phase >= ctx->n_phases || (do_push && (nsx < 1 || nsy < 1 || nsz < 1 || nsx > 64 ||
        nsy > 64 || nsz > 64)) || (do_finalize && !dose4d_dev))
        return fail(ctx, PBS4D_ERR_ARG, std::string(who) + ": bad argument");
    auto dose_of = [&](int p) -> const float* {
        if (phase_dose_dev) return phase_dose_dev[p];
        return ctx->have_dose[p] ? ctx->dose[p]->as<float>() : nullptr;
    };
    if (!dose_of(ref_phase)) return fail(ctx, PBS4D_ERR_ORDER, std::string(who) + ": no dose for the reference phase");
    std::vector<int> src;
    for (int p = 0; p < ctx->n_phases; ++p)
        if (p != ref_phase && ctx->dvf[p].set && ctx->dvf[p].ref == ref_phase && dose_of(p)) src.push_back(p);
    if (src.size() > 32) return fail(ctx, PBS4D_ERR_ARG, std::string(who) + ": more than 32 source phases");
    CU(cudaSetDevice(ctx->device));
    const size_t nvox = ctx->nvox();
    EventTrio ev;                                        // destroyed on every return path
    CU(ev.create());
    cudaEvent_t e0 = ev.e[0], e1 = ev.e[1], e2 = ev.e[2];
    uint64_t pushed = 0;
    if (do_push) {
        CU(ctx->acc_counters.ensure(sizeof(AccCounters)));
        CU(cudaMemsetAsync(ctx->acc_counters.p, 0, sizeof(AccCounters), ctx->stream));
        std::fill(ctx->have_acc.begin(), ctx->have_acc.end(), false);
        for (int p : src) {
            CU(ctx->accE[p]->ensure(nvox * sizeof(long long)));
            CU(ctx->accM[p]->ensure(nvox * sizeof(long long)));
            CU(cudaMemsetAsync(ctx->accE[p]->p, 0, nvox * sizeof(long long), ctx->stream));
            CU(cudaMemsetAsync(ctx->accM[p]->p, 0, nvox * sizeof(long long), ctx->stream));
        }
    }
    CU(cudaEventRecord(e0, ctx->stream));
    if (do_push) {
        for (int p : src) {
            ctx->have_acc[p] = true;
            if (!((src_mask >> p) & 1u)) continue;
            launch_emtm_push(ctx->dose_grid, dose_of(p), ctx->rho[p]->as<float>(), ctx->dvf[p].grid,
                             ctx->dvf[p].disp->as<float>(), ctx->dose_grid, nsx, nsy, nsz,
                             ctx->accE[p]->as<long long>(), ctx->accM[p]->as<long long>(),
                             ctx->acc_counters.as<AccCounters>(), ctx->stream);
            pushed += 1;
        }
    }
    CU(cudaEventRecord(e1, ctx->stream));
    if (do_finalize) {
        std::vector<const long long*> Ep, Mp; std::vector<pbs4d_grid> dg;
        for (int p : src) {
            if (!ctx->have_acc[p]) return fail(ctx, PBS4D_ERR_ORDER, std::string(who) + ": source phase was not pushed");
            Ep.push_back(ctx->accE[p]->as<long long>()); Mp.push_back(ctx->accM[p]->as<long long>());
            dg.push_back(ctx->dvf[p].grid);
        }
        CU(ctx->cover_flags.ensure((size_t)ctx->dose_grid.nx + ctx->dose_grid.ny + ctx->dose_grid.nz));
        launch_emtm_finalize(ctx->dose_grid, dose_of(ref_phase), (int)src.size(), Ep.data(), Mp.data(), dg.data(),
                             ctx->cover_flags.as<unsigned char>(), dose4d_dev, ctx->stream);
    }
    CU(cudaEventRecord(e2, ctx->stream));
    CU(cudaGetLastError());
    AccCounters ac{};
    if (do_push) CU(cudaMemcpyAsync(&ac, ctx->acc_counters.p, sizeof(ac), cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    if (stats) {
        stats->subvoxels = pushed * nvox * (do_push ? (uint64_t)nsx * nsy * nsz : 0);
        stats->dropped_outside_ref = ac.dropped_ref; stats->dropped_outside_dvf = ac.dropped_dvf;
        cudaEventElapsedTime(&stats->push_ms, e0, e1);
        cudaEventElapsedTime(&stats->finalize_ms, e1, e2);
    }
    return PBS4D_OK;
}

}  // namespace

extern "C" int pbs4d_accumulate_subvoxel(pbs4d_ctx* ctx, int32_t ref_phase, int32_t nsx, int32_t nsy, int32_t nsz,
                                         const float* const* phase_dose_dev, float* dose4d_dev,
                                         pbs4d_acc_stats* stats) try
{
    const NvtxRange nvtx_range_("pbs4d_accumulate_subvoxel");
    if (!ctx) return PBS4D_ERR_ARG;
    return accumulate_impl(ctx, "accumulate_subvoxel", ref_phase, nsx, nsy, nsz, phase_dose_dev, 0xFFFFFFFFu, true, true,
                           dose4d_dev, stats);
}
catch (...) { return on_exception(ctx); }

// the two halves of accumulate_subvoxel, for runs sharded by source phase: every rank pushes the source
// phases of its src_mask, the int64 sums are exchanged through pbs4d_accumulator_ptrs, then a9 runs on the full set
extern "C" int pbs4d_accumulate_push(pbs4d_ctx* ctx, int32_t ref_phase, int32_t nsx, int32_t nsy, int32_t nsz,
                                     const float* const* phase_dose_dev, uint32_t src_mask, pbs4d_acc_stats* stats) try
{
    const NvtxRange nvtx_range_("pbs4d_accumulate_push");
    if (!ctx) return PBS4D_ERR_ARG;
    return accumulate_impl(ctx, "accumulate_push", ref_phase, nsx, nsy, nsz, phase_dose_dev, src_mask, true, false,
                           nullptr, stats);
}
catch (...) { return on_exception(ctx); }

extern "C" int pbs4d_accumulate_finalize(pbs4d_ctx* ctx, int32_t ref_phase, const float* const* phase_dose_dev,
                                         float* dose4d_dev, pbs4d_acc_stats* stats) try
{
    const NvtxRange nvtx_range_("pbs4d_accumulate_finalize");
    if (!ctx) return PBS4D_ERR_ARG;
    return accumulate_impl(ctx, "accumulate_finalize", ref_phase, 1, 1, 1, phase_dose_dev, 0u, false, true, dose4d_dev,
                           stats);
}
catch (...) { return on_exception(ctx); }

extern "C" int pbs4d_accumulator_ptrs(pbs4d_ctx* ctx, int32_t src_phase, int64_t** e_dev, int64_t** m_dev) try
{
    const NvtxRange nvtx_range_("pbs4d_accumulator_ptrs");
    if (!ctx) return PBS4D_ERR_ARG;
    if (src_phase < 0 || src_phase >= ctx->n_phases || !e_dev || !m_dev)
        return fail(ctx, PBS4D_ERR_ARG, "accumulator_ptrs: bad argument");
    if (!ctx->have_acc[src_phase]) return fail(ctx, PBS4D_ERR_ORDER, "accumulator_ptrs: phase has no accumulators");
    *e_dev = ctx->accE[src_phase]->as<int64_t>(); *m_dev = ctx->accM[src_phase]->as<int64_t>();
    return PBS4D_OK;
}
catch (...) { return on_exception(ctx); }

extern "C" int pbs4d_get_accumulators(pbs4d_ctx* ctx, int32_t src_phase, int64_t* e_dev, int64_t* m_dev) try
{
    const NvtxRange nvtx_range_("pbs4d_get_accumulators");
    if (!ctx) return PBS4D_ERR_ARG;
    if (src_phase < 0 || src_phase >= ctx->n_phases || !e_dev || !m_dev)
        return fail(ctx, PBS4D_ERR_ARG, "get_accumulators: bad argument");
    if (!ctx->have_acc[src_phase]) return fail(ctx, PBS4D_ERR_ORDER, "get_accumulators: phase was not pushed");
    CU(cudaSetDevice(ctx->device));
    CU(cudaMemcpyAsync(e_dev, ctx->accE[src_phase]->p, ctx->nvox() * sizeof(long long), cudaMemcpyDeviceToDevice, ctx->stream));
    CU(cudaMemcpyAsync(m_dev, ctx->accM[src_phase]->p, ctx->nvox() * sizeof(long long), cudaMemcpyDeviceToDevice, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    return PBS4D_OK;
}
catch (...) { return on_exception(ctx); }

// ------------------------------------------------------------------------------------------------------------------
// uncertainty trials: sampled delivery -> per-phase MC -> accumulation, per trial, context re-used
// ------------------------------------------------------------------------------------------------------------------
extern "C" int pbs4d_simulate_delivery_trial(pbs4d_ctx* ctx, const pbs4d_trial_spec* spec, int32_t trial,
                                             const pbs4d_delivery_params* prm, const pbs4d_delivery_ext* ext,
                                             uint64_t total_histories, pbs4d_phase_lists* out, int64_t* n_fills) try
{
    const NvtxRange nvtx_range_("pbs4d_simulate_delivery_trial");
    if (!ctx) return PBS4D_ERR_ARG;
    if (!spec || !prm) return fail(ctx, PBS4D_ERR_ARG, "simulate_delivery_trial: null argument");
    if (ctx->fields.empty()) return fail(ctx, PBS4D_ERR_ORDER, "simulate_delivery_trial: call set_plan_spots first");
    const pbs4d_delivery_ext none{};
    const pbs4d_delivery_ext& central = ext ? *ext : none;
    const int32_t nf = (int32_t)ctx->fields.size();
    std::vector<int32_t> start(nf);
    std::vector<int64_t> cycles(std::max(spec->n_cycles, 1)), resets(std::max(central.n_layer_switch, 1));
    pbs4d_delivery_params p{}; pbs4d_delivery_ext x{};
    const int rc = sample_trial_host(*spec, trial, nf, *prm, central, start.data(), cycles.data(), resets.data(), p, x);
    if (rc != PBS4D_OK) return fail(ctx, rc, "simulate_delivery_trial: bad trial specification");
    // the sampled starting phases are this trial's, not the plan's: the planned ones come back when the call ends,
    // whether or not the simulation succeeds (the segment lists it leaves in the context are the trial's)
    struct RestoreStartPhases {
        std::vector<pbs4d_field>& fields; std::vector<int32_t> planned;
        explicit RestoreStartPhases(std::vector<pbs4d_field>& f) : fields(f) { for (const auto& e : f) planned.push_back(e.start_phase); }
        ~RestoreStartPhases() { for (size_t f = 0; f < planned.size() && f < fields.size(); ++f) fields[f].start_phase = planned[f]; }
    } restore(ctx->fields);
    for (int32_t f = 0; f < nf; ++f) ctx->fields[f].start_phase = start[f];
    return pbs4d_simulate_delivery_ext(ctx, &p, &x, total_histories, out, n_fills);
}
catch (...) { return on_exception(ctx); }

extern "C" int pbs4d_run_trials(pbs4d_ctx* ctx, const pbs4d_trial_spec* spec, int32_t first, int32_t count,
                                const pbs4d_delivery_params* prm, const pbs4d_delivery_ext* ext,
                                uint64_t total_histories, uint64_t seed, int32_t ref_phase, int32_t nsx, int32_t nsy,
                                int32_t nsz, float* const* dose4d_dev, pbs4d_trial_result* results) try
{
    const NvtxRange nvtx_range_("pbs4d_run_trials");
    if (!ctx) return PBS4D_ERR_ARG;
    if (!spec || !prm || !dose4d_dev || first < 0 || count < 1 || first + count > spec->n_trials)
        return fail(ctx, PBS4D_ERR_ARG, "run_trials: bad argument");
    if (!ctx->have_density) return fail(ctx, PBS4D_ERR_ORDER, "run_trials: no densities (set_ct_phases)");
    if (ctx->shard_world != 1)                              // no exchange happens in here: the doses would be partial
        return fail(ctx, PBS4D_ERR_ORDER, "run_trials: history sharding is on (set_shard(0, 1) first); a sharded run "
                                          "needs the caller's sum over ranks between transport and accumulation");
    if (ref_phase < 0 || ref_phase >= ctx->n_phases) return fail(ctx, PBS4D_ERR_ARG, "run_trials: bad reference phase");
    for (int32_t t = 0; t < count; ++t) {
        if (!dose4d_dev[t]) return fail(ctx, PBS4D_ERR_ARG, "run_trials: null output buffer");
        int64_t fills = 0;
        int rc = pbs4d_simulate_delivery_trial(ctx, spec, first + t, prm, ext, total_histories, nullptr, &fills);
        if (rc != PBS4D_OK) return rc;
        std::vector<int32_t> todo;
        for (int p = 0; p < ctx->n_phases && p < ctx->deliv_phases; ++p)
            if (ctx->launches[p].n_hist > 0 || p == ref_phase) todo.push_back(p);
        std::vector<pbs4d_mc_stats> st(todo.size());
        float tr_ms = 0.0f;
        std::fill(ctx->have_dose.begin(), ctx->have_dose.end(), false);     // doses of the previous trial are stale
        rc = pbs4d_mc_dose_phases(ctx, (int32_t)todo.size(), todo.data(), seed + (uint64_t)(first + t), 0.0, st.data(),
                                  &tr_ms);
        if (rc != PBS4D_OK) return rc;
        pbs4d_acc_stats as{};
        rc = pbs4d_accumulate_subvoxel(ctx, ref_phase, nsx, nsy, nsz, nullptr, dose4d_dev[t], &as);
        if (rc != PBS4D_OK) return rc;
        if (results) {
            pbs4d_trial_result& r = results[t];
            r.histories = 0; for (const auto& s : st) r.histories += s.histories;
            r.delivery_ns = 0; for (int64_t v : ctx->field_time) r.delivery_ns = std::max(r.delivery_ns, v);
            r.fills = fills; r.phases_run = 0; r.pad = 0;
            for (int p = 0; p < ctx->deliv_phases; ++p) r.phases_run += ctx->launches[p].n_hist > 0 ? 1 : 0;
            r.transport_ms = tr_ms; r.accumulate_ms = as.push_ms + as.finalize_ms;
        }
    }
    return PBS4D_OK;
}
catch (...) { return on_exception(ctx); }

// ------------------------------------------------------------------------------------------------------------------
// whole path with host buffers (end-to-end entry used by bench.py's e2e leg)
// ------------------------------------------------------------------------------------------------------------------
extern "C" int pbs4d_run_plan_host(pbs4d_ctx* ctx, int32_t n_phases, const pbs4d_grid* ct, const int16_t* const* hu_host,
                                   const pbs4d_grid* dose_grid, int32_t n_pts, const float* hu_pts, const float* rho_pts,
                                   const pbs4d_grid* dvf_grid, const float* const* disp_host, int32_t ref_phase,
                                   int32_t n_fields, const pbs4d_field* fields, int64_t n_spots, const pbs4d_spot* spots,
                                   const pbs4d_delivery_params* prm, uint64_t total_histories, uint64_t seed,
                                   int32_t nsx, int32_t nsy, int32_t nsz, float* dose4d_host, uint64_t* histories_run,
                                   uint64_t* h2d_bytes, double* seconds) try
{
    const NvtxRange nvtx_range_("pbs4d_run_plan_host");
    if (!ctx) return PBS4D_ERR_ARG;
    if (const char* why = grid_defect(ct)) return fail(ctx, PBS4D_ERR_ARG, std::string("run_plan_host: ct: ") + why);
    if (dose_grid) if (const char* why = grid_defect(dose_grid)) return fail(ctx, PBS4D_ERR_ARG, std::string("run_plan_host: dose_grid: ") + why);
    if (disp_host) if (const char* why = grid_defect(dvf_grid)) return fail(ctx, PBS4D_ERR_ARG, std::string("run_plan_host: dvf_grid: ") + why);
    if (n_phases < 1 || n_phases > 32 || !grid_ok(ct) || !hu_host || !prm || !dose4d_host || ref_phase < 0 ||
        ref_phase >= n_phases || prm->n_phases != n_phases || (disp_host && !grid_ok(dvf_grid)) ||
        (dose_grid && !grid_ok(dose_grid)) || n_pts < 2 || n_pts > 64 || !hu_pts || !rho_pts)
        return fail(ctx, PBS4D_ERR_ARG, "run_plan_host: bad argument");
    for (int i = 0; i < n_pts; ++i)
        if (!(rho_pts[i] > 0.0f) || (i && !(hu_pts[i] > hu_pts[i - 1])))
            return fail(ctx, PBS4D_ERR_ARG, "run_plan_host: table must ascend in HU with positive densities");
    for (int p = 0; p < n_phases; ++p)
        if (!hu_host[p]) return fail(ctx, PBS4D_ERR_ARG, "run_plan_host: null CT phase");
    if (ctx->shard_world != 1)                              // no exchange happens in here: the dose would be partial
        return fail(ctx, PBS4D_ERR_ORDER, "run_plan_host: history sharding is on (set_shard(0, 1) first); a sharded run "
                                          "needs the caller's sum over ranks between transport and accumulation");
    using clk = std::chrono::steady_clock;
    auto sec = [](clk::time_point a, clk::time_point b) { return std::chrono::duration<double>(b - a).count(); };
    CU(cudaSetDevice(ctx->device));
    const auto t0 = clk::now();

    // a2 + a3 first (host only, ~ms): the sub-plans say which breathing phases receive beam, and only those phases
    // (plus the reference phase) need a density grid, a transport launch and -- as push sources -- a DVF.  With gating
    // most phases of a 4DCT are idle (config 5: 4 of 10 active); their CT and DVF are not uploaded at all.
    int rc = pbs4d_set_plan_spots(ctx, n_fields, fields, n_spots, spots);
    if (rc != PBS4D_OK) return rc;
    rc = pbs4d_simulate_delivery(ctx, prm, total_histories, nullptr);
    if (rc != PBS4D_OK) return rc;
    std::vector<int32_t> active;
    for (int p = 0; p < n_phases; ++p)
        if (ctx->launches[p].n_hist > 0 || p == ref_phase) active.push_back(p);
    const auto t1 = clk::now();

    // H2D: CT of the active phases -> densities (a1)
    uint64_t bytes = 0;
    const pbs4d_grid& g = dose_grid ? *dose_grid : *ct;
    reset_phase_state(ctx, n_phases, g);
    for (int p : active) {                               // launch tables first: see upload_segments
        rc = upload_segments(ctx, p, ctx->stream);
        if (rc != PBS4D_OK) return rc;
    }
    const size_t ct_vox = (size_t)ct->nx * ct->ny * ct->nz;
    DevBuf& hu_dev = ctx->host_hu;
    CU(hu_dev.ensure(active.size() * ct_vox * sizeof(int16_t)));
    CU(ctx->table.ensure(kTableBytes));
    // an early error return must not leave copies from the caller's host buffers in flight: armed before the first copy
    struct CopyGuard {
        cudaStream_t st[3] = { nullptr, nullptr, nullptr }; cudaEvent_t ev = nullptr; bool armed = false;
        ~CopyGuard() { if (armed) for (auto s : st) cudaStreamSynchronize(s); if (ev) cudaEventDestroy(ev); }
    } guard;
    if (!ctx->copy_stream) CU(cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking));
    if (!ctx->prep_stream) CU(cudaStreamCreateWithFlags(&ctx->prep_stream, cudaStreamNonBlocking));
    guard.st[0] = ctx->stream; guard.st[1] = ctx->copy_stream; guard.st[2] = ctx->prep_stream; guard.armed = true;
    // Host -> device traffic is pure DMA on the copy stream, back to back: the CT of every active phase, then the DVFs
    // (each into its own staging area).  The kernels that consume an upload (HU -> density, DVF re-layout) run on a
    // second stream behind per-upload events, so a kernel that has to wait for SM space under a running transport
    // kernel never holds up the next copy.  The transport launch of a phase waits for that phase's density event only
    // (mc_dose_phases): the first phase starts after its own 84 MB, everything else runs underneath the transport.
    if (ctx->rho_ready.size() < (size_t)n_phases) ctx->rho_ready.resize(n_phases, nullptr);
    if (ctx->upload_done.size() < (size_t)2 * n_phases) ctx->upload_done.resize((size_t)2 * n_phases, nullptr);
    auto event_at = [&](std::vector<cudaEvent_t>& v, size_t i) -> cudaError_t {
        return v[i] ? cudaSuccess : cudaEventCreateWithFlags(&v[i], cudaEventDisableTiming);
    };
    CU(cudaMemcpyAsync(ctx->table.p, hu_pts, n_pts * sizeof(float), cudaMemcpyHostToDevice, ctx->copy_stream));
    CU(cudaMemcpyAsync(ctx->table.as<float>() + n_pts, rho_pts, n_pts * sizeof(float), cudaMemcpyHostToDevice,
                       ctx->copy_stream));
    for (size_t a = 0; a < active.size(); ++a) {
        const int p = active[a];
        int16_t* dst = hu_dev.as<int16_t>() + a * ct_vox;
        CU(cudaMemcpyAsync(dst, hu_host[p], ct_vox * sizeof(int16_t), cudaMemcpyHostToDevice, ctx->copy_stream));
        bytes += ct_vox * sizeof(int16_t);
        CU(event_at(ctx->upload_done, 2 * p));
        CU(cudaEventRecord(ctx->upload_done[2 * p], ctx->copy_stream));
        CU(ctx->rho[p]->ensure(ctx->nvox() * sizeof(float)));
        CU(cudaStreamWaitEvent(ctx->prep_stream, ctx->upload_done[2 * p], 0));
        launch_hu_to_density(*ct, dst, dose_grid, n_pts, ctx->table.as<float>(), ctx->table.as<float>() + n_pts,
                             rho_pts[0], reinterpret_cast<double*>(ctx->table.as<char>() + kTableLutOffset),
                             ctx->rho[p]->as<float>(), ctx->prep_stream);
        CU(event_at(ctx->rho_ready, p));
        CU(cudaEventRecord(ctx->rho_ready[p], ctx->prep_stream));
        ctx->rho_valid[p] = true; ctx->rho_pending[p] = true;
    }
    CU(cudaGetLastError());
    ctx->have_density = true;
    // DVFs are not needed before the accumulation (the bulk of the host->device bytes)
    cudaEvent_t& dvf_ready = guard.ev;
    if (disp_host) {
        const size_t dvf_vox = (size_t)dvf_grid->nx * dvf_grid->ny * dvf_grid->nz;
        size_t n_dvf = 0;
        for (int p : active) n_dvf += (p != ref_phase && disp_host[p]) ? 1 : 0;
        DevBuf& tmp = ctx->host_dvf;
        CU(tmp.ensure(std::max<size_t>(n_dvf, 1) * 3 * dvf_vox * sizeof(float)));
        size_t k = 0;
        for (int p : active) {
            if (p == ref_phase || !disp_host[p]) continue;
            auto& d = ctx->dvf[p];
            if (!d.disp) d.disp.reset(new DevBuf);
            CU(d.disp->ensure((4 * dvf_vox + 4) * sizeof(float)));   // + max |u| record
            float* stage = tmp.as<float>() + k * 3 * dvf_vox; ++k;
            CU(cudaMemcpyAsync(stage, disp_host[p], 3 * dvf_vox * sizeof(float), cudaMemcpyHostToDevice, ctx->copy_stream));
            bytes += 3 * dvf_vox * sizeof(float);
            CU(event_at(ctx->upload_done, 2 * p + 1));
            CU(cudaEventRecord(ctx->upload_done[2 * p + 1], ctx->copy_stream));
            CU(cudaStreamWaitEvent(ctx->prep_stream, ctx->upload_done[2 * p + 1], 0));
            launch_dvf_interleave(*dvf_grid, stage, d.disp->as<float>(), ctx->prep_stream);
            d.set = true; d.ref = ref_phase; d.grid = *dvf_grid;
        }
        CU(cudaGetLastError());
        CU(cudaEventCreateWithFlags(&dvf_ready, cudaEventDisableTiming));
        CU(cudaEventRecord(dvf_ready, ctx->prep_stream));
    }
    const auto t2 = clk::now();

    uint64_t run = 0;
    {
        std::vector<pbs4d_mc_stats> st(active.size());
        rc = pbs4d_mc_dose_phases(ctx, (int32_t)active.size(), active.data(), seed, 0.0, st.data(), nullptr);
        if (rc != PBS4D_OK) return rc;
        for (const auto& x : st) run += x.histories;
    }
    const auto t3 = clk::now();

    DevBuf& out = ctx->host_out;
    CU(out.ensure(ctx->nvox() * sizeof(float)));
    if (dvf_ready) CU(cudaStreamWaitEvent(ctx->stream, dvf_ready, 0));
    rc = pbs4d_accumulate_subvoxel(ctx, ref_phase, nsx, nsy, nsz, nullptr, out.as<float>(), nullptr);
    if (rc != PBS4D_OK) return rc;
    CU(cudaMemcpyAsync(dose4d_host, out.p, ctx->nvox() * sizeof(float), cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    const auto t4 = clk::now();
    if (histories_run) *histories_run = run;
    if (h2d_bytes) *h2d_bytes = bytes + (uint64_t)n_spots * sizeof(pbs4d_spot) + (uint64_t)n_fields * sizeof(pbs4d_field);
    if (seconds) { seconds[0] = sec(t0, t1); seconds[1] = sec(t1, t2); seconds[2] = sec(t2, t3); seconds[3] = sec(t3, t4); }
    return PBS4D_OK;
}
catch (...) { return on_exception(ctx); }

// ------------------------------------------------------------------------------------------------------------------
// in-run roofline probes
// ------------------------------------------------------------------------------------------------------------------
extern "C" int pbs4d_roofline_probe(pbs4d_ctx* ctx, int32_t kind, double* value) try
{
    const NvtxRange nvtx_range_("pbs4d_roofline_probe");
    if (!ctx) return PBS4D_ERR_ARG;
    if (!value || kind < PBS4D_PROBE_FP32_ISSUE || kind > PBS4D_PROBE_HBM_COPY)
        return fail(ctx, PBS4D_ERR_ARG, "roofline_probe: bad argument");
    CU(cudaSetDevice(ctx->device));
    *value = 0.0;
    switch (kind) {
        case PBS4D_PROBE_FP32_ISSUE: CU(probe_fp32_issue(ctx->sm_count, ctx->stream, value)); break;
        case PBS4D_PROBE_RED_RANDOM: CU(probe_l2_atomic(ctx->sm_count, 0, ctx->stream, value)); break;
        case PBS4D_PROBE_RED_HOT:    CU(probe_l2_atomic(ctx->sm_count, 1, ctx->stream, value)); break;
        default:                     CU(probe_hbm_copy(ctx->sm_count, ctx->stream, value)); break;
    }
    return PBS4D_OK;
}
catch (...) { return on_exception(ctx); }

// ------------------------------------------------------------------------------------------------------------------
// dose-interpolation accumulation (DIM, Eq. 3): pull every source phase with a T^{R->S} field
// ------------------------------------------------------------------------------------------------------------------
extern "C" int pbs4d_accumulate_dim(pbs4d_ctx* ctx, int32_t ref_phase, int32_t nsx, int32_t nsy, int32_t nsz,
                                    const float* const* phase_dose_dev, float* dose4d_dev, pbs4d_acc_stats* stats) try
{
    const NvtxRange nvtx_range_("pbs4d_accumulate_dim");
    if (!ctx) return PBS4D_ERR_ARG;
    if (!ctx->have_density) return fail(ctx, PBS4D_ERR_ORDER, "accumulate_dim: no grid (set_ct_phases/set_density_phases)");
    if (ref_phase < 0 || ref_phase >= ctx->n_phases || nsx < 1 || nsy < 1 || nsz < 1 || nsx > 64 || nsy > 64 ||
        nsz > 64 || !dose4d_dev)
        return fail(ctx, PBS4D_ERR_ARG, "accumulate_dim: bad argument");
    auto dose_of = [&](int p) -> const float* {
        if (phase_dose_dev) return phase_dose_dev[p];
        return ctx->have_dose[p] ? ctx->dose[p]->as<float>() : nullptr;
    };
    if (!dose_of(ref_phase)) return fail(ctx, PBS4D_ERR_ORDER, "accumulate_dim: no dose for the reference phase");
    std::vector<int> src;
    for (int p = 0; p < ctx->n_phases; ++p)
        if (p != ref_phase && ctx->dvf_pull[p].set && ctx->dvf_pull[p].ref == ref_phase && dose_of(p)) src.push_back(p);
    CU(cudaSetDevice(ctx->device));
    const size_t nvox = ctx->nvox();
    CU(ctx->acc_counters.ensure(sizeof(AccCounters)));
    CU(cudaMemsetAsync(ctx->acc_counters.p, 0, sizeof(AccCounters), ctx->stream));
    CU(ctx->dim_acc.ensure(nvox * sizeof(double)));
    CU(ctx->cover_flags.ensure((size_t)ctx->dose_grid.nx + ctx->dose_grid.ny + ctx->dose_grid.nz));
    EventTrio ev;                                        // destroyed on every return path
    CU(ev.create());
    cudaEvent_t e0 = ev.e[0], e1 = ev.e[1], e2 = ev.e[2];
    launch_dim_init(ctx->dose_grid, dose_of(ref_phase), ctx->dim_acc.as<double>(), ctx->stream);
    CU(cudaEventRecord(e0, ctx->stream));
    std::vector<pbs4d_grid> dg;
    for (int p : src) {                                  // ascending phase order: Eq. 2 is summed in this order
        launch_dim_pull(ctx->dose_grid, nsx, nsy, nsz, ctx->dvf_pull[p].grid, ctx->dvf_pull[p].disp->as<float>(),
                        ctx->dose_grid, dose_of(p), ctx->dim_acc.as<double>(), ctx->acc_counters.as<AccCounters>(),
                        ctx->stream);
        dg.push_back(ctx->dvf_pull[p].grid);
    }
    CU(cudaEventRecord(e1, ctx->stream));
    launch_dim_final(ctx->dose_grid, (int)src.size(), dg.data(), ctx->dim_acc.as<double>(),
                     ctx->cover_flags.as<unsigned char>(), dose4d_dev, ctx->stream);
    CU(cudaEventRecord(e2, ctx->stream));
    CU(cudaGetLastError());
    AccCounters ac{};
    CU(cudaMemcpyAsync(&ac, ctx->acc_counters.p, sizeof(ac), cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    if (stats) {
        stats->subvoxels = (uint64_t)src.size() * nvox * nsx * nsy * nsz;
        stats->dropped_outside_ref = ac.dropped_ref; stats->dropped_outside_dvf = ac.dropped_dvf;
        cudaEventElapsedTime(&stats->push_ms, e0, e1);
        cudaEventElapsedTime(&stats->finalize_ms, e1, e2);
    }
    return PBS4D_OK;
}
catch (...) { return on_exception(ctx); }

// ------------------------------------------------------------------------------------------------------------------
// DVF construction from DICOM minimal grid information
// ------------------------------------------------------------------------------------------------------------------
extern "C" int pbs4d_build_dvf(pbs4d_ctx* ctx, const pbs4d_dicom_dvf* info, const float* delta_dev, float* rf_dev,
                               float* disp_dev, pbs4d_grid* grid_out) try
{
    const NvtxRange nvtx_range_("pbs4d_build_dvf");
    if (!ctx) return PBS4D_ERR_ARG;
    if (!info || !delta_dev || (!rf_dev && !disp_dev) || info->nx < 1 || info->ny < 1 || info->nz < 1 ||
        (double)info->nx * info->ny * info->nz >= 2.0e9 || !(info->delta[0] > 0.0) || !(info->delta[1] > 0.0) ||
        !(info->delta[2] > 0.0))
        return fail(ctx, PBS4D_ERR_ARG, "build_dvf: bad argument");
    if (grid_out) {
        const double* U = info->row_cos; const double* V = info->col_cos;
        if (!(U[0] == 1.0 && U[1] == 0.0 && U[2] == 0.0 && V[0] == 0.0 && V[1] == 1.0 && V[2] == 0.0))
            return fail(ctx, PBS4D_ERR_ARG, "build_dvf: grid_out needs direction cosines along +x, +y");
        grid_out->nx = info->nx; grid_out->ny = info->ny; grid_out->nz = info->nz;
        grid_out->hx = (float)info->delta[0]; grid_out->hy = (float)info->delta[1]; grid_out->hz = (float)info->delta[2];
        grid_out->ox = (float)(info->start[0] - 0.5 * info->delta[0]);      // start = centre of the first voxel
        grid_out->oy = (float)(info->start[1] - 0.5 * info->delta[1]);
        grid_out->oz = (float)(info->start[2] - 0.5 * info->delta[2]);
    }
    CU(cudaSetDevice(ctx->device));
    launch_dvf_build(*info, delta_dev, rf_dev, disp_dev, ctx->stream);
    CU(cudaGetLastError());
    CU(cudaStreamSynchronize(ctx->stream));
    return PBS4D_OK;
}
catch (...) { return on_exception(ctx); }
