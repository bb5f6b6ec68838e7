// Delivery-uncertainty sampling for the paper's uncertainty trials: for each of
// T trials the breathing phase in which delivery commences ~ U{CT_0..CT_90}, the breathing period ~ U{3..7} s, the
// per-cycle phase length t_ph ~ N(mu, sigma)/N and every synchrotron timing parameter ~ N(central, uncertainty) are
// drawn together; the 4D dose is then recomputed per trial (pbs4d_run_trials in api.cu).  Host only, integers out.
//
// The paper drew with cuRAND state; here each draw is one Philox4x32-10 block addressed by
// (block, stream, trial), so any trial can be re-sampled alone and the result does not depend on T or on the order.
// Draw table (U0-U5):
//   stream 0, block 0, word 0        mean breathing period, index into {lo, lo + step, ...}
//   stream 1, block f / 4, word f%4  start phase of field f
//   stream 2, block c                period of breathing cycle c          (Box-Muller, cosine branch of words 0, 1)
//   stream 3, block j                synchrotron parameter j              (same)
#include "internal.h"

#include <algorithm>
#include <cmath>

namespace pbs4d {

namespace {

struct Draws {
    uint32_t k0, k1, trial;
    void words(uint32_t stream, uint32_t blk, uint32_t out[4]) const
    {
        uint32_t c[4] = { blk, stream, trial, 0x55545249u };        // 'UTRI'
        uint32_t ka = k0, kb = k1;
        for (int round = 0; round < 10; ++round) {
            const uint64_t a = (uint64_t)0xD2511F53u * c[0], b = (uint64_t)0xCD9E8D57u * c[2];
            const uint32_t n0 = (uint32_t)(b >> 32) ^ c[1] ^ ka, n2 = (uint32_t)(a >> 32) ^ c[3] ^ kb;
            c[1] = (uint32_t)b; c[3] = (uint32_t)a; c[0] = n0; c[2] = n2;
            ka += 0x9E3779B9u; kb += 0xBB67AE85u;
        }
        for (int i = 0; i < 4; ++i) out[i] = c[i];
    }
    static double unit(uint32_t w) { return ((double)(w >> 9) + 0.5) * (1.0 / 8388608.0); }
    double uniform(uint32_t stream, uint32_t blk, int word) const
    {
        uint32_t w[4]; words(stream, blk, w);
        return unit(w[word]);
    }
    double normal(uint32_t stream, uint32_t blk) const
    {
        uint32_t w[4]; words(stream, blk, w);
        return std::sqrt(-2.0 * std::log(unit(w[0]))) * std::cos(6.283185307179586476925286766559 * unit(w[1]));
    }
    // central + sigma * N(0,1), rounded to the nearest integer, not below `least`; sigma <= 0: the central value
    int64_t around(uint32_t j, int64_t central, int64_t sigma, int64_t least) const
    {
        if (sigma <= 0) return central;
        return std::max<int64_t>(std::llround((double)central + (double)sigma * normal(3u, j)), least);
    }
};

}  // namespace

int sample_trial_host(const pbs4d_trial_spec& spec, int32_t trial, int32_t n_fields, const pbs4d_delivery_params& prm,
                      const pbs4d_delivery_ext& ext, int32_t* start_phase, int64_t* cycle_period_ns,
                      int64_t* layer_switch_ns, pbs4d_delivery_params& prm_out, pbs4d_delivery_ext& ext_out)
{
    const int32_t N = prm.n_phases;
    if (trial < 0 || trial >= spec.n_trials || n_fields < 1 || !start_phase || N < 1 || N > 32 || spec.n_cycles < 0 ||
        (spec.n_cycles > 0 && !cycle_period_ns) || (ext.n_layer_switch > 0 && ext.layer_switch_ns && !layer_switch_ns))
        return PBS4D_ERR_ARG;
    const Draws rng{ (uint32_t)spec.seed, (uint32_t)(spec.seed >> 32), (uint32_t)trial };

    // mean breathing period: discrete uniform, inclusive
    int64_t mean_period = prm.period_ns;
    if (spec.period_lo_ns > 0) {
        mean_period = spec.period_lo_ns;
        if (spec.period_step_ns > 0 && spec.period_hi_ns > spec.period_lo_ns) {
            const int64_t choices = (spec.period_hi_ns - spec.period_lo_ns) / spec.period_step_ns + 1;
            mean_period += spec.period_step_ns * (int64_t)std::floor(rng.uniform(0u, 0u, 0) * (double)choices);
        }
    }
    // phase in which delivery of each field commences
    for (int32_t f = 0; f < n_fields; ++f)
        start_phase[f] = (int32_t)std::floor(rng.uniform(1u, (uint32_t)(f / 4), f % 4) * (double)N);
    // irregular breathing: one period per cycle, t_ph = period / N; never below a quarter of the mean
    int64_t fastest = mean_period, slowest = mean_period;
    for (int32_t c = 0; c < spec.n_cycles; ++c) {
        int64_t period = mean_period;
        if (spec.period_sigma_ns > 0)
            period = std::llround((double)mean_period + (double)spec.period_sigma_ns * rng.normal(2u, (uint32_t)c));
        period = std::max<int64_t>({ period, mean_period / 4, (int64_t)N });
        cycle_period_ns[c] = period;
        fastest = c ? std::min(fastest, period) : period;
        slowest = c ? std::max(slowest, period) : period;
    }
    // synchrotron parameters ~ N(central value, uncertainty); a limit that is off stays off
    prm_out = prm; ext_out = ext;
    prm_out.period_ns = mean_period;
    ext_out.n_cycles = spec.n_cycles;
    ext_out.cycle_period_ns = spec.n_cycles > 0 ? cycle_period_ns : nullptr;
    ext_out.discard_ns = rng.around(0u, ext.discard_ns, spec.discard_sigma_ns, 0);
    ext_out.flat_top_ns = ext.flat_top_ns > 0 ? rng.around(1u, ext.flat_top_ns, spec.flat_top_sigma_ns, 1) : 0;
    ext_out.spot_switch_fixed_ns = rng.around(2u, ext.spot_switch_fixed_ns, spec.spot_switch_sigma_ns, 0);
    ext_out.spill_protons_max = ext.spill_protons_max > 0
        ? rng.around(3u, ext.spill_protons_max, spec.spill_protons_sigma, 1) : 0;
    prm_out.protons_per_s = rng.around(4u, prm.protons_per_s, spec.protons_per_s_sigma, 1);
    prm_out.layer_switch_ns = rng.around(5u, prm.layer_switch_ns, spec.layer_switch_sigma_ns, 0);
    if (ext.n_layer_switch > 0 && ext.layer_switch_ns) {
        for (int32_t l = 0; l < ext.n_layer_switch; ++l)
            layer_switch_ns[l] = rng.around(6u + (uint32_t)l, ext.layer_switch_ns[l], spec.layer_switch_sigma_ns, 0);
        ext_out.layer_switch_ns = layer_switch_ns;
    }
    // keep every trial deliverable: the discard must fit into the shortest phase, a fill must outlast the longest
    // gate hold (simulate_delivery_ext rejects anything else)
    if (ext_out.discard_ns > 0)
        ext_out.discard_ns = std::max<int64_t>(std::min(ext_out.discard_ns, fastest / N - 1), 0);
    if (ext_out.flat_top_ns > 0)
        ext_out.flat_top_ns = std::max(ext_out.flat_top_ns, ext_out.discard_ns + slowest + 1);
    return PBS4D_OK;
}

}  // namespace pbs4d

extern "C" int pbs4d_sample_delivery_trial(const pbs4d_trial_spec* spec, int32_t trial, int32_t n_fields,
                                           const pbs4d_delivery_params* prm, const pbs4d_delivery_ext* ext,
                                           int32_t* start_phase, int64_t* cycle_period_ns, int64_t* layer_switch_ns,
                                           pbs4d_delivery_params* prm_out, pbs4d_delivery_ext* ext_out)
{
    if (!spec || !prm || !ext || !prm_out || !ext_out) return PBS4D_ERR_ARG;
    try {
        return pbs4d::sample_trial_host(*spec, trial, n_fields, *prm, *ext, start_phase, cycle_period_ns, layer_switch_ns,
                                        *prm_out, *ext_out);
    } catch (...) { return PBS4D_ERR_NOMEM; }
}
