// Host beam-delivery timeline simulator (Sec. 2.B, App. A).
//
// Tracks plan-delivery time against breathing time and splits every spot's protons over the breathing phases they
// are delivered in -> N_g sub-plans per field.  The paper ran this as a GPU kernel over fields
// (PAPER.md:51); here it is a few thousand integer events per field, so it runs on the host (BASELINE.json
// north_star: "a host delivery-timeline simulator").  All arithmetic is int64/int128: the result is unique.
//
// Model (BASELINE.json configs 3, 5): spill at protons_per_s, Euclidean scan move at ns_per_um, constant
// layer-switch time, fixed breathing period, N x layer repainting, gate bitmask.
#include "internal.h"

#include <algorithm>
#include <cmath>

namespace pbs4d {

namespace {

using u128 = unsigned __int128;
constexpr int64_t kNsPerS = 1000000000;

// quotient of two 128-bit values: the operands of this file nearly always fit in 64 bits (times in ns, distances in
// um), where the hardware divide is several times faster than the 128-bit library routine; same result
inline u128 div128(u128 a, u128 b)
{
    if (((a | b) >> 64) == 0) return (u128)((uint64_t)a / (uint64_t)b);
    return a / b;
}

// floor(sqrt(v)) by Newton iteration on integers
int64_t floor_sqrt(u128 v)
{
    if (v == 0) return 0;
    if ((v >> 62) == 0) {                              // the usual case, in 64-bit arithmetic (x + v / x < 2^63)
        const uint64_t w = (uint64_t)v;
        uint64_t x = (uint64_t)std::sqrt((double)w) + 2;
        for (;;) {
            const uint64_t y = (x + w / x) >> 1;
            if (y >= x) break;
            x = y;
        }
        while (x * x > w) --x;
        return (int64_t)x;
    }
    u128 x = (u128)std::sqrt((double)v) + 2;           // start at or above the root
    for (;;) {
        u128 y = (x + v / x) >> 1;
        if (y >= x) break;
        x = y;
    }
    while (x * x > v) --x;
    return (int64_t)x;
}

// Breathing clock of one field: phase bins of length t_ph counted from the start of start_phase.
struct BreathingClock {
    int64_t t_ph; int32_t n_phases, start_phase; uint32_t gate;
    int64_t bin(int64_t t) const { return t / t_ph; }
    int32_t phase(int64_t t) const { return (int32_t)((bin(t) + start_phase) % n_phases); }
    int64_t next_edge(int64_t t) const { return (bin(t) + 1) * t_ph; }
    bool beam_allowed(int64_t t) const { return (gate >> phase(t)) & 1u; }
};

// sub-plans in (field, phase, spot) order, then histories by cumulative rounding
void allocate_histories(const std::vector<int64_t>& delivered, size_t nf, int32_t P, size_t ns, uint64_t total_histories,
                        std::vector<pbs4d_segment>& segments, int64_t& dropped_protons)
{
    segments.clear();
    u128 total = 0;
    for (size_t f = 0; f < nf; ++f)
        for (int32_t p = 0; p < P; ++p)
            for (size_t s = 0; s < ns; ++s) {
                const int64_t c = delivered[(f * P + p) * ns + s];
                if (c <= 0) continue;
                pbs4d_segment sg{};
                sg.field = (int32_t)f; sg.phase = p; sg.spot = (int32_t)s; sg.protons = c;
                segments.push_back(sg);
                total += (u128)c;
            }
    dropped_protons = 0;
    u128 running = 0; int64_t edge_prev = 0;
    for (auto& sg : segments) {
        running += (u128)sg.protons;
        const int64_t edge = total_histories ? (int64_t)div128((u128)total_histories * running, total) : 0;
        sg.first_history = edge_prev;
        sg.n_hist = edge - edge_prev;
        sg.weight = sg.n_hist > 0 ? (double)sg.protons / (double)sg.n_hist : 0.0;
        if (total_histories && sg.n_hist == 0) dropped_protons += sg.protons;
        edge_prev = edge;
    }
}

}  // namespace

int simulate_delivery_host(const std::vector<pbs4d_field>& fields, const std::vector<pbs4d_spot>& spots,
                           const pbs4d_delivery_params& prm, uint64_t total_histories,
                           std::vector<pbs4d_segment>& segments, std::vector<int64_t>& field_time_ns,
                           int64_t& dropped_protons, std::string& err)
{
    const int32_t P = prm.n_phases;
    if (P <= 0 || P > 32) { err = "n_phases must be in [1, 32]"; return PBS4D_ERR_ARG; }
    if (prm.period_ns < P || prm.protons_per_s <= 0 || prm.repaints <= 0 || prm.ns_per_um < 0 ||
        prm.layer_switch_ns < 0 || prm.protons_per_weight < 0) { err = "bad delivery parameter"; return PBS4D_ERR_ARG; }
    const uint32_t all = P == 32 ? 0xFFFFFFFFu : ((1u << P) - 1u);
    if ((prm.gate_mask & all) == 0) { err = "gate_mask allows no phase"; return PBS4D_ERR_ARG; }

    const size_t nf = fields.size(), ns = spots.size();
    std::vector<int64_t> delivered(nf * (size_t)P * std::max<size_t>(ns, 1), 0);   // [field][phase][spot]
    field_time_ns.assign(nf, 0);

    for (size_t f = 0; f < nf; ++f) {
        BreathingClock clk{ prm.period_ns / P, P, fields[f].start_phase % P, prm.gate_mask };
        if (clk.start_phase < 0) clk.start_phase += P;
        int64_t t = 0;
        bool any_layer = false;
        size_t i = 0;
        while (i < ns) {
            if (spots[i].field != (int32_t)f) { ++i; continue; }
            size_t end = i;                                     // layer = run of equal layer ids in array order
            while (end < ns && spots[end].field == (int32_t)f && spots[end].layer == spots[i].layer) ++end;
            if (any_layer) t += prm.layer_switch_ns;
            any_layer = true;

            bool beam_positioned = false; int64_t bx = 0, by = 0;
            for (int32_t paint = 0; paint < prm.repaints; ++paint) {
                for (size_t s = i; s < end; ++s) {
                    const int64_t n_spot  = std::llround((double)spots[s].weight * (double)prm.protons_per_weight);
                    int64_t todo = n_spot / prm.repaints + ((n_spot % prm.repaints) > paint ? 1 : 0);
                    if (todo <= 0) continue;
                    const int64_t x_um = std::llround((double)spots[s].x_mm * 1000.0);
                    const int64_t y_um = std::llround((double)spots[s].y_mm * 1000.0);
                    if (beam_positioned) {
                        const u128 ddx = (u128)(x_um > bx ? x_um - bx : bx - x_um);
                        const u128 ddy = (u128)(y_um > by ? y_um - by : by - y_um);
                        t += floor_sqrt((ddx * ddx + ddy * ddy) * (u128)prm.ns_per_um * (u128)prm.ns_per_um);
                    }
                    beam_positioned = true; bx = x_um; by = y_um;

                    // spill: proton j after the spill clock (re)started at t leaves at t + floor(j * 1e9 / rate)
                    while (todo > 0) {
                        if (!clk.beam_allowed(t)) { t = clk.next_edge(t); continue; }      // gate closed: hold
                        const int64_t window = clk.next_edge(t) - t;                         // ns left in this phase
                        // protons leaving strictly before the edge: j * 1e9 / rate < window
                        const u128 cap = div128((u128)window * (u128)prm.protons_per_s + (kNsPerS - 1), (u128)kNsPerS);
                        const int64_t n = cap < (u128)todo ? (int64_t)cap : todo;
                        delivered[(f * P + clk.phase(t)) * ns + s] += n;
                        todo -= n;
                        t += (int64_t)div128((u128)n * kNsPerS, (u128)prm.protons_per_s);
                    }
                }
            }
            i = end;
        }
        field_time_ns[f] = t;
    }

    allocate_histories(delivered, nf, P, ns, total_histories, segments, dropped_protons);
    return PBS4D_OK;
}

// ------------------------------------------------------------------------------------------------------------------
// Extended model (Sec. 2.B, App. A): irregular breathing cycles,
// the beam discarded whenever extraction (re)starts, synchrotron fills limited by charge capacity and flat-top time
// with an energy-dependent reset, a fixed part of the spot-switch time, iso-layered repainting with a maximum number
// of protons per spot delivery.  Ref. 45's constants are not in the container: every value is an input
// (pbs4d_delivery_ext), including the sampled breathing periods.  With every field zero this is the base model.
// ------------------------------------------------------------------------------------------------------------------
namespace {

// Breathing trace of one field with per-cycle periods: phase edges are generated cycle by cycle as time advances.
class BreathingTrace {
public:
    BreathingTrace(const pbs4d_delivery_params& prm, const pbs4d_delivery_ext& ext, int32_t start_phase)
        : prm_(prm), ext_(ext), P_(prm.n_phases)
    {
        // field time 0 = beginning of start_phase of the first cycle
        cycle_begin_ = -(int64_t)start_phase * phase_len(0);
    }
    void seek(int64_t t)                                   // t never decreases
    {
        while (t >= cycle_begin_ + phase_len(cycle_) * P_) { cycle_begin_ += phase_len(cycle_) * P_; ++cycle_; }
        phase_ = (int32_t)((t - cycle_begin_) / phase_len(cycle_));
    }
    int32_t phase() const { return phase_; }
    int64_t edge() const { return cycle_begin_ + (int64_t)(phase_ + 1) * phase_len(cycle_); }
    bool open() const { return (prm_.gate_mask >> phase_) & 1u; }

private:
    int64_t phase_len(int32_t c) const
    {
        int64_t period = prm_.period_ns;
        if (ext_.cycle_period_ns && ext_.n_cycles > 0) period = ext_.cycle_period_ns[std::min(c, ext_.n_cycles - 1)];
        return period / P_;
    }
    const pbs4d_delivery_params& prm_; const pbs4d_delivery_ext& ext_;
    int32_t P_, cycle_ = 0, phase_ = 0; int64_t cycle_begin_ = 0;
};

// One synchrotron fill: protons left, flat-top deadline, and whether the next extraction must discard beam first.
struct Fill {
    int64_t left = 0, deadline = 0; bool limited_charge = false, limited_time = false, fresh = true;
    void start(int64_t t, const pbs4d_delivery_ext& ext)
    {
        limited_charge = ext.spill_protons_max > 0; limited_time = ext.flat_top_ns > 0;
        left = ext.spill_protons_max; deadline = t + ext.flat_top_ns; fresh = true;
    }
    bool spent(int64_t t) const { return (limited_time && t >= deadline) || (limited_charge && left == 0); }
};

// protons that leave strictly before `until` when the spill clock starts at t: ceil((until - t) rate / 1e9)
int64_t protons_before(int64_t t, int64_t until, int64_t rate, int64_t at_most)
{
    const u128 cap = ((u128)(until - t) * (u128)rate + (kNsPerS - 1)) / kNsPerS;
    return cap < (u128)at_most ? (int64_t)cap : at_most;
}

}  // namespace

int simulate_delivery_ext_host(const std::vector<pbs4d_field>& fields, const std::vector<pbs4d_spot>& spots,
                               const pbs4d_delivery_params& prm, const pbs4d_delivery_ext& ext,
                               uint64_t total_histories, std::vector<pbs4d_segment>& segments,
                               std::vector<int64_t>& field_time_ns, int64_t& dropped_protons, int64_t& n_fills,
                               std::string& err)
{
    const int32_t P = prm.n_phases;
    if (P <= 0 || P > 32) { err = "n_phases must be in [1, 32]"; return PBS4D_ERR_ARG; }
    if (prm.period_ns < P || prm.protons_per_s <= 0 || prm.repaints <= 0 || prm.ns_per_um < 0 ||
        prm.layer_switch_ns < 0 || prm.protons_per_weight < 0) { err = "bad delivery parameter"; return PBS4D_ERR_ARG; }
    const uint32_t all = P == 32 ? 0xFFFFFFFFu : ((1u << P) - 1u);
    if ((prm.gate_mask & all) == 0) { err = "gate_mask allows no phase"; return PBS4D_ERR_ARG; }
    if (ext.discard_ns < 0 || ext.spill_protons_max < 0 || ext.flat_top_ns < 0 || ext.spot_switch_fixed_ns < 0 ||
        ext.max_protons_per_paint < 0 || ext.n_cycles < 0 || ext.n_layer_switch < 0) {
        err = "negative extended delivery parameter"; return PBS4D_ERR_ARG;
    }
    int64_t longest = prm.period_ns, shortest = prm.period_ns;
    if (ext.cycle_period_ns && ext.n_cycles > 0) {
        longest = shortest = ext.cycle_period_ns[0];
        for (int32_t c = 0; c < ext.n_cycles; ++c) {
            if (ext.cycle_period_ns[c] < P) { err = "breathing period shorter than n_phases ns"; return PBS4D_ERR_ARG; }
            longest = std::max(longest, ext.cycle_period_ns[c]); shortest = std::min(shortest, ext.cycle_period_ns[c]);
        }
    }
    if (ext.discard_ns > 0 && ext.discard_ns >= shortest / P) {
        err = "discard_ns must be shorter than one breathing phase"; return PBS4D_ERR_ARG;
    }
    if (ext.flat_top_ns > 0 && ext.flat_top_ns <= ext.discard_ns + longest) {
        err = "flat_top_ns must exceed the longest breathing period plus discard_ns"; return PBS4D_ERR_ARG;
    }
    if (ext.layer_switch_ns) for (int32_t l = 0; l < ext.n_layer_switch; ++l)
        if (ext.layer_switch_ns[l] < 0) { err = "negative layer-switch time"; return PBS4D_ERR_ARG; }

    const size_t nf = fields.size(), ns = spots.size();
    std::vector<int64_t> delivered(nf * (size_t)P * std::max<size_t>(ns, 1), 0);
    field_time_ns.assign(nf, 0);
    n_fills = 0;

    for (size_t f = 0; f < nf; ++f) {
        int32_t sp = fields[f].start_phase % P; if (sp < 0) sp += P;
        BreathingTrace breath(prm, ext, sp);
        Fill fill;
        int64_t t = 0;
        bool any_layer = false;
        size_t i = 0;
        while (i < ns) {
            if (spots[i].field != (int32_t)f) { ++i; continue; }
            size_t end = i;
            while (end < ns && spots[end].field == (int32_t)f && spots[end].layer == spots[i].layer) ++end;
            const int32_t layer = spots[i].layer;
            const int64_t reset_ns = (ext.layer_switch_ns && layer >= 0 && layer < ext.n_layer_switch)
                                         ? ext.layer_switch_ns[layer] : prm.layer_switch_ns;
            if (any_layer) t += reset_ns;
            any_layer = true;
            fill.start(t, ext); ++n_fills;

            // protons still owed to every spot of the layer; a painting hands out one slice of each
            std::vector<int64_t> owed(end - i);
            for (size_t s = i; s < end; ++s)
                owed[s - i] = std::llround((double)spots[s].weight * (double)prm.protons_per_weight);
            bool beam_positioned = false; int64_t bx = 0, by = 0;
            for (int64_t paint = 0; ; ++paint) {
                if (ext.max_protons_per_paint == 0 && paint >= prm.repaints) break;
                bool painted = false;
                for (size_t s = i; s < end; ++s) {
                    int64_t todo;
                    if (ext.max_protons_per_paint > 0) {
                        todo = std::min(owed[s - i], ext.max_protons_per_paint);
                        owed[s - i] -= todo;
                    } else {
                        const int64_t n_spot = owed[s - i];
                        todo = n_spot / prm.repaints + ((n_spot % prm.repaints) > paint ? 1 : 0);
                    }
                    if (todo <= 0) continue;
                    painted = true;
                    const int64_t x_um = std::llround((double)spots[s].x_mm * 1000.0);
                    const int64_t y_um = std::llround((double)spots[s].y_mm * 1000.0);
                    if (beam_positioned) {
                        const u128 ddx = (u128)(x_um > bx ? x_um - bx : bx - x_um);
                        const u128 ddy = (u128)(y_um > by ? y_um - by : by - y_um);
                        t += floor_sqrt((ddx * ddx + ddy * ddy) * (u128)prm.ns_per_um * (u128)prm.ns_per_um)
                             + ext.spot_switch_fixed_ns;
                    }
                    beam_positioned = true; bx = x_um; by = y_um;

                    while (todo > 0) {
                        breath.seek(t);
                        if (!breath.open()) { t = breath.edge(); fill.fresh = true; continue; }   // hold for gate-on
                        if (fill.spent(t)) { t += reset_ns; fill.start(t, ext); ++n_fills; continue; }
                        if (fill.fresh) {                                                       // extraction begins
                            fill.fresh = false;
                            if (ext.discard_ns > 0) { t += ext.discard_ns; continue; }
                        }
                        int64_t until = breath.edge();
                        if (fill.limited_time) until = std::min(until, fill.deadline);
                        int64_t n = protons_before(t, until, prm.protons_per_s, todo);
                        if (fill.limited_charge) n = std::min(n, fill.left);
                        delivered[(f * P + breath.phase()) * ns + s] += n;
                        todo -= n;
                        if (fill.limited_charge) fill.left -= n;
                        t += (int64_t)(((u128)n * kNsPerS) / (u128)prm.protons_per_s);
                    }
                }
                if (ext.max_protons_per_paint > 0 && !painted) break;
            }
            i = end;
        }
        field_time_ns[f] = t;
    }
    allocate_histories(delivered, nf, P, ns, total_histories, segments, dropped_protons);
    return PBS4D_OK;
}

// Fixed-point shift k: the whole plan's energy (x 1.1) must fit 2^62 quanta even in one voxel.
int32_t fixed_shift_for(const std::vector<pbs4d_segment>& segments, const std::vector<pbs4d_spot>& spots)
{
    double tot = 0.0;
    for (const auto& sg : segments) tot += (double)sg.protons * (double)spots[sg.spot].energy_mev;
    tot *= 1.1;
    if (!(tot > 0.0)) return 40;
    int32_t k = (int32_t)std::floor(std::log2(4611686018427387904.0 / tot));
    return std::min(k, 40);
}

}  // namespace pbs4d

extern "C" int pbs4d_simulate_delivery_host(int32_t n_fields, const pbs4d_field* fields, int64_t n_spots,
                                            const pbs4d_spot* spots, const pbs4d_delivery_params* prm,
                                            uint64_t total_histories, pbs4d_segment* segs_out, int64_t max_segs,
                                            int64_t* n_segs_out, int64_t* field_time_ns, int64_t* dropped_protons,
                                            int32_t* fixed_shift) try
{
    if (n_fields < 1 || !fields || n_spots < 1 || !spots || !prm || !n_segs_out) return PBS4D_ERR_ARG;
    std::vector<pbs4d_field> f(fields, fields + n_fields);
    std::vector<pbs4d_spot> s(spots, spots + n_spots);
    for (const auto& sp : s) if (sp.field < 0 || sp.field >= n_fields) return PBS4D_ERR_ARG;
    std::vector<pbs4d_segment> segs; std::vector<int64_t> times; int64_t dropped = 0; std::string err;
    const int rc = pbs4d::simulate_delivery_host(f, s, *prm, total_histories, segs, times, dropped, err);
    if (rc != PBS4D_OK) return rc;
    *n_segs_out = (int64_t)segs.size();
    if (segs_out) {
        if (max_segs < (int64_t)segs.size()) return PBS4D_ERR_ARG;
        std::copy(segs.begin(), segs.end(), segs_out);
    }
    if (field_time_ns) std::copy(times.begin(), times.end(), field_time_ns);
    if (dropped_protons) *dropped_protons = dropped;
    if (fixed_shift) *fixed_shift = pbs4d::fixed_shift_for(segs, s);
    return PBS4D_OK;
}
catch (...) { return PBS4D_ERR_NOMEM; }     // std::bad_alloc: nothing throws across the C boundary

extern "C" int pbs4d_simulate_delivery_ext_host(int32_t n_fields, const pbs4d_field* fields, int64_t n_spots,
                                                const pbs4d_spot* spots, const pbs4d_delivery_params* prm,
                                                const pbs4d_delivery_ext* ext, uint64_t total_histories,
                                                pbs4d_segment* segs_out, int64_t max_segs, int64_t* n_segs_out,
                                                int64_t* field_time_ns, int64_t* dropped_protons, int32_t* fixed_shift,
                                                int64_t* n_fills) try
{
    if (n_fields < 1 || !fields || n_spots < 1 || !spots || !prm || !ext || !n_segs_out) return PBS4D_ERR_ARG;
    std::vector<pbs4d_field> f(fields, fields + n_fields);
    std::vector<pbs4d_spot> s(spots, spots + n_spots);
    for (const auto& sp : s) if (sp.field < 0 || sp.field >= n_fields) return PBS4D_ERR_ARG;
    std::vector<pbs4d_segment> segs; std::vector<int64_t> times; int64_t dropped = 0, fills = 0; std::string err;
    const int rc = pbs4d::simulate_delivery_ext_host(f, s, *prm, *ext, total_histories, segs, times, dropped, fills, err);
    if (rc != PBS4D_OK) return rc;
    *n_segs_out = (int64_t)segs.size();
    if (segs_out) {
        if (max_segs < (int64_t)segs.size()) return PBS4D_ERR_ARG;
        std::copy(segs.begin(), segs.end(), segs_out);
    }
    if (field_time_ns) std::copy(times.begin(), times.end(), field_time_ns);
    if (dropped_protons) *dropped_protons = dropped;
    if (fixed_shift) *fixed_shift = pbs4d::fixed_shift_for(segs, s);
    if (n_fills) *n_fills = fills;
    return PBS4D_OK;
}
catch (...) { return PBS4D_ERR_NOMEM; }     // std::bad_alloc: nothing throws across the C boundary
