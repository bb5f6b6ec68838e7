// C-ABI boundary of libpbs4d (include/pbs4d.h): context, argument checks, device memory, launch sequencing.
// No arithmetic of the method lives here -- it is in delivery.cpp (host, int64), transport.cu, grids.cu and
// accumulate.cu (device).
#include "internal.h"

#include <cuda_runtime.h>

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
    DevBuf table;                                        // hu_pts | rho_pts

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
    std::vector<std::unique_ptr<DevBuf>> seg_phase;      // [phase] launch table (DevSegment[] | seg_begin[])
    std::vector<cudaStream_t> aux;                       // auxiliary streams for concurrent phase launches
    cudaStream_t copy_stream = nullptr;                  // uploads that overlap compute (run_plan_host)

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

#define CU(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return cuda_fail(ctx, e_, #call); } while (0)

bool grid_ok(const pbs4d_grid* g)
{
    return g && g->nx > 0 && g->ny > 0 && g->nz > 0 && g->hx > 0.0f && g->hy > 0.0f && g->hz > 0.0f &&
           std::isfinite(g->ox) && std::isfinite(g->oy) && std::isfinite(g->oz) &&
           (double)g->nx * g->ny * g->nz < 2.0e9;
}

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
    ctx->have_density = false;
}

}  // namespace

extern "C" {

int pbs4d_create(pbs4d_ctx** out, int device, void* cuda_stream)
{
    if (!out) return PBS4D_ERR_ARG;
    *out = nullptr;
    int n_dev = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || device < 0 || device >= n_dev) return PBS4D_ERR_CUDA;
    if (cudaSetDevice(device) != cudaSuccess) return PBS4D_ERR_CUDA;
    pbs4d_ctx* ctx = new (std::nothrow) pbs4d_ctx;
    if (!ctx) return PBS4D_ERR_NOMEM;
    ctx->device = device;
    ctx->stream = static_cast<cudaStream_t>(cuda_stream);
    cudaDeviceProp prop{};
    if (cudaGetDeviceProperties(&prop, device) == cudaSuccess) ctx->sm_count = prop.multiProcessorCount;
    *out = ctx;
    return PBS4D_OK;
}

void pbs4d_destroy(pbs4d_ctx* ctx)
{
    if (!ctx) return;
    cudaSetDevice(ctx->device);
    cudaStreamSynchronize(ctx->stream);
    for (auto st : ctx->aux) if (st) cudaStreamDestroy(st);
    if (ctx->copy_stream) { cudaStreamSynchronize(ctx->copy_stream); cudaStreamDestroy(ctx->copy_stream); }
    delete ctx;
}

const char* pbs4d_last_error(const pbs4d_ctx* ctx) { return ctx ? ctx->err.c_str() : "null context"; }

int pbs4d_set_ct_phases(pbs4d_ctx* ctx, int32_t n_phases, const pbs4d_grid* ct, const int16_t* const* hu_dev,
                        const pbs4d_grid* dose_grid, int32_t n_pts, const float* hu_pts, const float* rho_pts)
{
    if (!ctx) return PBS4D_ERR_ARG;
    if (n_phases < 1 || n_phases > 32 || !grid_ok(ct) || !hu_dev || (dose_grid && !grid_ok(dose_grid)) ||
        n_pts < 2 || n_pts > 64 || !hu_pts || !rho_pts)
        return fail(ctx, PBS4D_ERR_ARG, "set_ct_phases: bad argument");
    for (int i = 0; i < n_pts; ++i) {
        if (!(rho_pts[i] > 0.0f) || (i && !(hu_pts[i] > hu_pts[i - 1])))
            return fail(ctx, PBS4D_ERR_ARG, "set_ct_phases: table must ascend in HU with positive densities");
    }
    for (int p = 0; p < n_phases; ++p) if (!hu_dev[p]) return fail(ctx, PBS4D_ERR_ARG, "set_ct_phases: null phase");
    CU(cudaSetDevice(ctx->device));
    const pbs4d_grid& g = dose_grid ? *dose_grid : *ct;
    reset_phase_state(ctx, n_phases, g);
    CU(ctx->table.ensure(2 * n_pts * sizeof(float)));
    CU(cudaMemcpyAsync(ctx->table.p, hu_pts, n_pts * sizeof(float), cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaMemcpyAsync(ctx->table.as<float>() + n_pts, rho_pts, n_pts * sizeof(float), cudaMemcpyHostToDevice,
                       ctx->stream));
    for (int p = 0; p < n_phases; ++p) {
        CU(ctx->rho[p]->ensure(ctx->nvox() * sizeof(float)));
        launch_hu_to_density(*ct, hu_dev[p], dose_grid, n_pts, ctx->table.as<float>(),
                             ctx->table.as<float>() + n_pts, ctx->rho[p]->as<float>(), ctx->stream);
    }
    CU(cudaGetLastError());
    CU(cudaStreamSynchronize(ctx->stream));
    ctx->have_density = true;
    return PBS4D_OK;
}

int pbs4d_set_density_phases(pbs4d_ctx* ctx, int32_t n_phases, const pbs4d_grid* dose_grid,
                             const float* const* rho_dev)
{
    if (!ctx) return PBS4D_ERR_ARG;
    if (n_phases < 1 || n_phases > 32 || !grid_ok(dose_grid) || !rho_dev)
        return fail(ctx, PBS4D_ERR_ARG, "set_density_phases: bad argument");
    for (int p = 0; p < n_phases; ++p) if (!rho_dev[p]) return fail(ctx, PBS4D_ERR_ARG, "set_density_phases: null phase");
    CU(cudaSetDevice(ctx->device));
    reset_phase_state(ctx, n_phases, *dose_grid);
    for (int p = 0; p < n_phases; ++p) {
        CU(ctx->rho[p]->ensure(ctx->nvox() * sizeof(float)));
        CU(cudaMemcpyAsync(ctx->rho[p]->p, rho_dev[p], ctx->nvox() * sizeof(float), cudaMemcpyDeviceToDevice,
                           ctx->stream));
    }
    CU(cudaStreamSynchronize(ctx->stream));
    ctx->have_density = true;
    return PBS4D_OK;
}

static int store_dvf(pbs4d_ctx* ctx, std::vector<pbs4d_ctx::Dvf>& table, const char* who, int32_t src_phase,
                     int32_t ref_phase, const pbs4d_grid* dvf_grid, const float* disp_dev)
{
    if (!ctx) return PBS4D_ERR_ARG;
    if (!ctx->have_density) return fail(ctx, PBS4D_ERR_ORDER, std::string(who) + ": call set_ct_phases/set_density_phases first");
    if (src_phase < 0 || src_phase >= ctx->n_phases || ref_phase < 0 || ref_phase >= ctx->n_phases ||
        src_phase == ref_phase || !grid_ok(dvf_grid) || !disp_dev)
        return fail(ctx, PBS4D_ERR_ARG, std::string(who) + ": bad argument");
    CU(cudaSetDevice(ctx->device));
    auto& d = table[src_phase];
    if (!d.disp) d.disp.reset(new DevBuf);
    const size_t bytes = (size_t)4 * dvf_grid->nx * dvf_grid->ny * dvf_grid->nz * sizeof(float);
    CU(d.disp->ensure(bytes));
    launch_dvf_interleave(*dvf_grid, disp_dev, d.disp->as<float>(), ctx->stream);
    CU(cudaGetLastError());
    CU(cudaStreamSynchronize(ctx->stream));
    d.set = true; d.ref = ref_phase; d.grid = *dvf_grid;
    return PBS4D_OK;
}

int pbs4d_set_dvf(pbs4d_ctx* ctx, int32_t src_phase, int32_t ref_phase, const pbs4d_grid* dvf_grid,
                  const float* disp_dev)
{
    if (!ctx) return PBS4D_ERR_ARG;
    return store_dvf(ctx, ctx->dvf, "set_dvf", src_phase, ref_phase, dvf_grid, disp_dev);
}

int pbs4d_set_dvf_pull(pbs4d_ctx* ctx, int32_t src_phase, int32_t ref_phase, const pbs4d_grid* dvf_grid,
                       const float* disp_dev)
{
    if (!ctx) return PBS4D_ERR_ARG;
    return store_dvf(ctx, ctx->dvf_pull, "set_dvf_pull", src_phase, ref_phase, dvf_grid, disp_dev);
}

int pbs4d_set_plan_spots(pbs4d_ctx* ctx, int32_t n_fields, const pbs4d_field* fields,
                         int64_t n_spots, const pbs4d_spot* spots)
{
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

int pbs4d_set_mc_flags(pbs4d_ctx* ctx, uint32_t flags)
{
    if (!ctx) return PBS4D_ERR_ARG;
    ctx->mc_flags = flags;
    return PBS4D_OK;
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------------------------
// a3: delivery simulation (host) and per-phase launch tables
// ------------------------------------------------------------------------------------------------------------------
extern "C" int pbs4d_simulate_delivery_ext(pbs4d_ctx* ctx, const pbs4d_delivery_params* prm,
                                           const pbs4d_delivery_ext* ext, uint64_t total_histories,
                                           pbs4d_phase_lists* out, int64_t* n_fills);

extern "C" int pbs4d_simulate_delivery(pbs4d_ctx* ctx, const pbs4d_delivery_params* prm, uint64_t total_histories,
                                       pbs4d_phase_lists* out)
{
    return pbs4d_simulate_delivery_ext(ctx, prm, nullptr, total_histories, out, nullptr);
}

// ext == NULL: the base simulator; else the extended model.  Both end in the same per-phase launch tables.
extern "C" int pbs4d_simulate_delivery_ext(pbs4d_ctx* ctx, const pbs4d_delivery_params* prm,
                                           const pbs4d_delivery_ext* ext, uint64_t total_histories,
                                           pbs4d_phase_lists* out, int64_t* n_fills)
{
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

// ------------------------------------------------------------------------------------------------------------------
// a4-a7: transport + scoring + finalize for one phase
// ------------------------------------------------------------------------------------------------------------------
namespace {
constexpr int kAuxStreams = 4;
}

extern "C" int pbs4d_mc_dose_phases(pbs4d_ctx* ctx, int32_t n, const int32_t* phases, uint64_t seed, double per_protons,
                                    pbs4d_mc_stats* stats, float* elapsed_ms)
{
    if (!ctx) return PBS4D_ERR_ARG;
    if (!ctx->have_density) return fail(ctx, PBS4D_ERR_ORDER, "mc_dose_phases: no densities (set_ct_phases)");
    if (!ctx->have_delivery) return fail(ctx, PBS4D_ERR_ORDER, "mc_dose_phases: call simulate_delivery first");
    if (n < 1 || n > 32 || !phases) return fail(ctx, PBS4D_ERR_ARG, "mc_dose_phases: bad argument");
    for (int a = 0; a < n; ++a) {
        if (phases[a] < 0 || phases[a] >= ctx->n_phases || phases[a] >= ctx->deliv_phases)
            return fail(ctx, PBS4D_ERR_ARG, "mc_dose_phases: phase out of range");
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
    if (ctx->seg_phase.size() < (size_t)ctx->n_phases) {
        ctx->seg_phase.resize(ctx->n_phases);
        for (auto& b : ctx->seg_phase) if (!b) b.reset(new DevBuf);
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
        guard(cudaEventRecord(ev[2 * a], st), "record");
        if (L.n_hist > 0) {
            DevBuf& sb = *ctx->seg_phase[phase];
            const size_t seg_bytes = L.segs.size() * sizeof(DevSegment);
            guard(sb.ensure(seg_bytes + L.segs.size() * sizeof(long long)), "alloc segments");
            if (rc != PBS4D_OK) break;
            guard(cudaMemcpyAsync(sb.p, L.segs.data(), seg_bytes, cudaMemcpyHostToDevice, st), "segments H2D");
            guard(cudaMemcpyAsync(sb.as<char>() + seg_bytes, L.seg_begin.data(), L.segs.size() * sizeof(long long),
                                  cudaMemcpyHostToDevice, st), "segments H2D");
            guard(cudaEventRecord(ev[2 * a], st), "record");
            launch_transport(ctx->dose_grid, ctx->rho[phase]->as<float>(), sb.as<DevSegment>(),
                             reinterpret_cast<const long long*>(sb.as<char>() + seg_bytes), (int32_t)L.segs.size(),
                             L.n_hist, seed, ctx->mc_flags, ctx->q[phase]->as<long long>(),
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
            s.fixed_shift = ctx->fixed_shift; s.pad = 0; s.pad2 = 0; s.scoring_atomics = tc[a].reds;
            s.kernel_ms = 0.0f;
            cudaEventElapsedTime(&s.kernel_ms, ev[2 * a], ev[2 * a + 1]);
        }
        if (elapsed_ms) cudaEventElapsedTime(elapsed_ms, span0, span1);
    }
    destroy_events();
    return rc;
}

extern "C" int pbs4d_mc_dose_phase(pbs4d_ctx* ctx, int32_t phase, uint64_t seed, double per_protons,
                                   float* dose_dev, float* rho_dev, pbs4d_mc_stats* stats)
{
    if (!ctx) return PBS4D_ERR_ARG;
    const int rc = pbs4d_mc_dose_phases(ctx, 1, &phase, seed, per_protons, stats, nullptr);
    if (rc != PBS4D_OK) return rc;
    const size_t nvox = ctx->nvox();
    if (dose_dev) CU(cudaMemcpyAsync(dose_dev, ctx->dose[phase]->p, nvox * sizeof(float), cudaMemcpyDeviceToDevice, ctx->stream));
    if (rho_dev)  CU(cudaMemcpyAsync(rho_dev, ctx->rho[phase]->p, nvox * sizeof(float), cudaMemcpyDeviceToDevice, ctx->stream));
    if (dose_dev || rho_dev) CU(cudaStreamSynchronize(ctx->stream));
    return PBS4D_OK;
}

extern "C" int pbs4d_get_phase_energy(pbs4d_ctx* ctx, int32_t phase, int64_t* q_dev)
{
    if (!ctx) return PBS4D_ERR_ARG;
    if (phase < 0 || phase >= ctx->n_phases || !q_dev) return fail(ctx, PBS4D_ERR_ARG, "get_phase_energy: bad argument");
    if (!ctx->have_dose[phase]) return fail(ctx, PBS4D_ERR_ORDER, "get_phase_energy: mc_dose_phase not run for this phase");
    CU(cudaSetDevice(ctx->device));
    CU(cudaMemcpyAsync(q_dev, ctx->q[phase]->p, ctx->nvox() * sizeof(long long), cudaMemcpyDeviceToDevice, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    return PBS4D_OK;
}

// ------------------------------------------------------------------------------------------------------------------
// a8-a9: subvoxel energy/mass push of every source phase with a DVF to ref_phase, then ratio + sum + mask
// ------------------------------------------------------------------------------------------------------------------
extern "C" int pbs4d_accumulate_subvoxel(pbs4d_ctx* ctx, int32_t ref_phase, int32_t nsx, int32_t nsy, int32_t nsz,
                                         const float* const* phase_dose_dev, float* dose4d_dev,
                                         pbs4d_acc_stats* stats)
{
    if (!ctx) return PBS4D_ERR_ARG;
    if (!ctx->have_density) return fail(ctx, PBS4D_ERR_ORDER, "accumulate_subvoxel: no densities");
    if (ref_phase < 0 || ref_phase >= ctx->n_phases || nsx < 1 || nsy < 1 || nsz < 1 || nsx > 64 || nsy > 64 ||
        nsz > 64 || !dose4d_dev)
        return fail(ctx, PBS4D_ERR_ARG, "accumulate_subvoxel: bad argument");
    auto dose_of = [&](int p) -> const float* {
        if (phase_dose_dev) return phase_dose_dev[p];
        return ctx->have_dose[p] ? ctx->dose[p]->as<float>() : nullptr;
    };
    if (!dose_of(ref_phase)) return fail(ctx, PBS4D_ERR_ORDER, "accumulate_subvoxel: no dose for the reference phase");
    std::vector<int> src;
    for (int p = 0; p < ctx->n_phases; ++p)
        if (p != ref_phase && ctx->dvf[p].set && ctx->dvf[p].ref == ref_phase && dose_of(p)) src.push_back(p);
    if (src.size() > 32) return fail(ctx, PBS4D_ERR_ARG, "accumulate_subvoxel: more than 32 source phases");
    CU(cudaSetDevice(ctx->device));
    const size_t nvox = ctx->nvox();
    CU(ctx->acc_counters.ensure(sizeof(AccCounters)));
    CU(cudaMemsetAsync(ctx->acc_counters.p, 0, sizeof(AccCounters), ctx->stream));
    EventTrio ev;                                        // destroyed on every return path
    CU(ev.create());
    cudaEvent_t e0 = ev.e[0], e1 = ev.e[1], e2 = ev.e[2];
    std::fill(ctx->have_acc.begin(), ctx->have_acc.end(), false);
    for (int p : src) {
        CU(ctx->accE[p]->ensure(nvox * sizeof(long long)));
        CU(ctx->accM[p]->ensure(nvox * sizeof(long long)));
        CU(cudaMemsetAsync(ctx->accE[p]->p, 0, nvox * sizeof(long long), ctx->stream));
        CU(cudaMemsetAsync(ctx->accM[p]->p, 0, nvox * sizeof(long long), ctx->stream));
    }
    CU(cudaEventRecord(e0, ctx->stream));
    std::vector<const long long*> Ep, Mp; std::vector<pbs4d_grid> dg;
    for (int p : src) {
        launch_emtm_push(ctx->dose_grid, dose_of(p), ctx->rho[p]->as<float>(), ctx->dvf[p].grid,
                         ctx->dvf[p].disp->as<float>(), ctx->dose_grid, nsx, nsy, nsz,
                         ctx->accE[p]->as<long long>(), ctx->accM[p]->as<long long>(),
                         ctx->acc_counters.as<AccCounters>(), ctx->stream);
        Ep.push_back(ctx->accE[p]->as<long long>()); Mp.push_back(ctx->accM[p]->as<long long>());
        dg.push_back(ctx->dvf[p].grid);
        ctx->have_acc[p] = true;
    }
    CU(cudaEventRecord(e1, ctx->stream));
    CU(ctx->cover_flags.ensure((size_t)ctx->dose_grid.nx + ctx->dose_grid.ny + ctx->dose_grid.nz));
    launch_emtm_finalize(ctx->dose_grid, dose_of(ref_phase), (int)src.size(), Ep.data(), Mp.data(), dg.data(),
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

extern "C" int pbs4d_get_accumulators(pbs4d_ctx* ctx, int32_t src_phase, int64_t* e_dev, int64_t* m_dev)
{
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

// ------------------------------------------------------------------------------------------------------------------
// whole path with host buffers (end-to-end entry used by bench.py's e2e leg)
// ------------------------------------------------------------------------------------------------------------------
extern "C" int pbs4d_run_plan_host(pbs4d_ctx* ctx, int32_t n_phases, const pbs4d_grid* ct, const int16_t* const* hu_host,
                                   const pbs4d_grid* dose_grid, int32_t n_pts, const float* hu_pts, const float* rho_pts,
                                   const pbs4d_grid* dvf_grid, const float* const* disp_host, int32_t ref_phase,
                                   int32_t n_fields, const pbs4d_field* fields, int64_t n_spots, const pbs4d_spot* spots,
                                   const pbs4d_delivery_params* prm, uint64_t total_histories, uint64_t seed,
                                   int32_t nsx, int32_t nsy, int32_t nsz, float* dose4d_host, uint64_t* histories_run,
                                   double* seconds)
{
    if (!ctx) return PBS4D_ERR_ARG;
    if (n_phases < 1 || n_phases > 32 || !grid_ok(ct) || !hu_host || !prm || !dose4d_host || ref_phase < 0 ||
        ref_phase >= n_phases || prm->n_phases != n_phases || (disp_host && !grid_ok(dvf_grid)))
        return fail(ctx, PBS4D_ERR_ARG, "run_plan_host: bad argument");
    using clk = std::chrono::steady_clock;
    auto sec = [](clk::time_point a, clk::time_point b) { return std::chrono::duration<double>(b - a).count(); };
    CU(cudaSetDevice(ctx->device));
    const auto t0 = clk::now();

    // H2D: CT phases -> densities, DVFs
    const size_t ct_vox = (size_t)ct->nx * ct->ny * ct->nz;
    DevBuf& hu_dev = ctx->host_hu;
    CU(hu_dev.ensure((size_t)n_phases * ct_vox * sizeof(int16_t)));
    std::vector<const int16_t*> hu_ptrs(n_phases);
    for (int p = 0; p < n_phases; ++p) {
        if (!hu_host[p]) return fail(ctx, PBS4D_ERR_ARG, "run_plan_host: null CT phase");
        hu_ptrs[p] = hu_dev.as<int16_t>() + (size_t)p * ct_vox;
        CU(cudaMemcpyAsync((void*)hu_ptrs[p], hu_host[p], ct_vox * sizeof(int16_t), cudaMemcpyHostToDevice, ctx->stream));
    }
    int rc = pbs4d_set_ct_phases(ctx, n_phases, ct, hu_ptrs.data(), dose_grid, n_pts, hu_pts, rho_pts);
    if (rc != PBS4D_OK) return rc;
    // DVFs are not needed before the accumulation: their upload (the bulk of the host->device bytes) and re-layout
    // run on a copy stream underneath the delivery simulation and the transport kernels
    struct CopyGuard {                                   // an early error return must not leave copies from the
        cudaStream_t st = nullptr; cudaEvent_t ev = nullptr;   // caller's host buffers in flight
        ~CopyGuard() { if (ev) { cudaStreamSynchronize(st); cudaEventDestroy(ev); } }
    } guard;
    cudaEvent_t& dvf_ready = guard.ev;
    if (disp_host) {
        if (!ctx->copy_stream) CU(cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking));
        const size_t dvf_vox = (size_t)dvf_grid->nx * dvf_grid->ny * dvf_grid->nz;
        DevBuf& tmp = ctx->host_dvf;
        CU(tmp.ensure(3 * dvf_vox * sizeof(float)));
        for (int p = 0; p < n_phases; ++p) {
            if (p == ref_phase || !disp_host[p]) continue;
            auto& d = ctx->dvf[p];
            if (!d.disp) d.disp.reset(new DevBuf);
            CU(d.disp->ensure(4 * dvf_vox * sizeof(float)));
            CU(cudaMemcpyAsync(tmp.p, disp_host[p], 3 * dvf_vox * sizeof(float), cudaMemcpyHostToDevice, ctx->copy_stream));
            launch_dvf_interleave(*dvf_grid, tmp.as<float>(), d.disp->as<float>(), ctx->copy_stream);
            d.set = true; d.ref = ref_phase; d.grid = *dvf_grid;
        }
        CU(cudaGetLastError());
        guard.st = ctx->copy_stream;
        CU(cudaEventCreateWithFlags(&dvf_ready, cudaEventDisableTiming));
        CU(cudaEventRecord(dvf_ready, ctx->copy_stream));
    }
    const auto t1 = clk::now();

    rc = pbs4d_set_plan_spots(ctx, n_fields, fields, n_spots, spots);
    if (rc != PBS4D_OK) return rc;
    rc = pbs4d_simulate_delivery(ctx, prm, total_histories, nullptr);
    if (rc != PBS4D_OK) return rc;
    const auto t2 = clk::now();

    uint64_t run = 0;
    {
        std::vector<int32_t> todo;
        for (int p = 0; p < n_phases; ++p)
            if (ctx->launches[p].n_hist > 0 || p == ref_phase) todo.push_back(p);
        std::vector<pbs4d_mc_stats> st(todo.size());
        rc = pbs4d_mc_dose_phases(ctx, (int32_t)todo.size(), todo.data(), seed, 0.0, st.data(), nullptr);
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
    if (seconds) { seconds[0] = sec(t0, t1); seconds[1] = sec(t1, t2); seconds[2] = sec(t2, t3); seconds[3] = sec(t3, t4); }
    return PBS4D_OK;
}

// ------------------------------------------------------------------------------------------------------------------
// in-run roofline probes
// ------------------------------------------------------------------------------------------------------------------
extern "C" int pbs4d_roofline_probe(pbs4d_ctx* ctx, int32_t kind, double* value)
{
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

// ------------------------------------------------------------------------------------------------------------------
// dose-interpolation accumulation (DIM, Eq. 3): pull every source phase with a T^{R->S} field
// ------------------------------------------------------------------------------------------------------------------
extern "C" int pbs4d_accumulate_dim(pbs4d_ctx* ctx, int32_t ref_phase, int32_t nsx, int32_t nsy, int32_t nsz,
                                    const float* const* phase_dose_dev, float* dose4d_dev, pbs4d_acc_stats* stats)
{
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

// ------------------------------------------------------------------------------------------------------------------
// DVF construction from DICOM minimal grid information
// ------------------------------------------------------------------------------------------------------------------
extern "C" int pbs4d_build_dvf(pbs4d_ctx* ctx, const pbs4d_dicom_dvf* info, const float* delta_dev, float* rf_dev,
                               float* disp_dev, pbs4d_grid* grid_out)
{
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
