/* oracle/orc_trials.c -- CPU ORACLE (test infrastructure only; see orc.h).
 * Sampling of the delivery uncertainties for the paper's uncertainty trials (second half).
 * PAPER.md:53 "the breathing phase during which delivery commences, which the user could either specify or allow to
 * be randomly selected"; "t_ph ~ N(mu, sigma)/N"; "Uncertainty values were sampled from a
 * Gaussian distribution with mean and standard deviation corresponding to the central value and uncertainty for the
 * given parameter"; "running 25 trials of the 4DDC where, for each trial, the initial-breathing phase,
 * breathing period, and synchrotron delivery parameters were simultaneously varied ...: starting phase ~ U(CT_0,
 * CT_90), synchrotron parameters ~ N(mu, sigma), and breathing period ~ U(3,7) s", U = discrete uniform, inclusive.
 * The paper drew with cuRAND; here every draw is a Philox4x32-10 block addressed by (what, which, trial),
 * so a trial can be re-sampled on its own and both sides of the parity test implement the same generator.
 * Steps:
 *  U0  block(stream, b) = Philox4x32-10(counter = (b, stream, trial, 0x55545249), key = (seed_lo, seed_hi));
 *      u_i = ((x_i >> 9) + 0.5) 2^-23 (T2); gauss(stream, b) = sqrt(-2 ln u_0) cos(2 pi u_1), double precision.
 *  U1  mean breathing period mu = lo + step * floor(u_0(stream 0, block 0) * K), K = (hi - lo) / step + 1 values;
 *      lo = 0: not sampled, mu = the plan's period_ns.
 *  U2  start phase of field f = floor(u_{f mod 4}(stream 1, block f / 4) * N)
 *  U3  period of breathing cycle c = max(llround(mu + sigma_T gauss(stream 2, block c)), mu / 4, N)
 *  U4  synchrotron parameter j = max(llround(central_j + sigma_j gauss(stream 3, block j)), floor_j); j = 0 discard,
 *      1 flat-top, 2 fixed spot-switch part, 3 charge per fill, 4 spill rate, 5 layer-switch constant, 6 + l
 *      layer-switch time of layer id l.  A limit that is switched off (central 0) stays off; floors: 0 for times,
 *      1 for the two limits (flat-top, charge) and the spill rate.
 *  U5  feasibility: discard <= shortest phase - 1 ns; flat-top (if on) >= discard + longest period + 1 ns, so that
 *      every sampled trial can be delivered (orc_simulate_delivery_ext rejects the opposite). */
#include "orc.h"
#include <math.h>
#include <string.h>

static const double TWO_PI_ = 6.283185307179586476925286766559;

static void block(const orc_trial_spec* s, int32_t trial, uint32_t stream, uint32_t b, double u[4])
{
    uint32_t ctr[4] = { b, stream, (uint32_t)trial, 0x55545249u };
    uint32_t key[2] = { (uint32_t)s->seed, (uint32_t)(s->seed >> 32) };
    uint32_t o[4];
    orc_philox4x32_10(ctr, key, o);
    for (int i = 0; i < 4; ++i) u[i] = ((double)(o[i] >> 9) + 0.5) * (1.0 / 8388608.0);
}

static double gauss(const orc_trial_spec* s, int32_t trial, uint32_t stream, uint32_t b)
{
    double u[4];
    block(s, trial, stream, b, u);
    return sqrt(-2.0 * log(u[0])) * cos(TWO_PI_ * u[1]);
}

static int64_t jitter(const orc_trial_spec* s, int32_t trial, uint32_t j, int64_t central, int64_t sigma, int64_t floor_v)
{
    if (sigma <= 0) return central;
    int64_t v = llround((double)central + (double)sigma * gauss(s, trial, 3u, j));
    return v < floor_v ? floor_v : v;
}

int orc_sample_trial(const orc_trial_spec* s, int32_t trial, int32_t n_fields,
                     const orc_delivery_params* prm, const orc_delivery_ext* ext,
                     int32_t* start_phase, int64_t* cycle_period_ns, int64_t* layer_switch_ns,
                     orc_delivery_params* prm_out, orc_delivery_ext* ext_out)
{
    if (!s || trial < 0 || trial >= s->n_trials || n_fields < 1 || !prm || !ext || !start_phase || !prm_out || !ext_out)
        return -1;
    const int32_t N = prm->n_phases;
    if (N < 1 || N > 32 || s->n_cycles < 0 || (s->n_cycles > 0 && !cycle_period_ns)) return -1;
    if (ext->n_layer_switch > 0 && ext->layer_switch_ns && !layer_switch_ns) return -1;
    double u[4];

    /* U1 */
    int64_t mu = prm->period_ns;
    if (s->period_lo_ns > 0) {
        mu = s->period_lo_ns;
        if (s->period_step_ns > 0 && s->period_hi_ns > s->period_lo_ns) {
            const int64_t K = (s->period_hi_ns - s->period_lo_ns) / s->period_step_ns + 1;
            block(s, trial, 0u, 0u, u);
            mu += s->period_step_ns * (int64_t)floor(u[0] * (double)K);
        }
    }
    /* U2 */
    for (int32_t f = 0; f < n_fields; ++f) {
        block(s, trial, 1u, (uint32_t)(f / 4), u);
        start_phase[f] = (int32_t)floor(u[f % 4] * (double)N);
    }
    /* U3 */
    int64_t shortest = mu, longest = mu;
    for (int32_t c = 0; c < s->n_cycles; ++c) {
        int64_t p = mu;
        if (s->period_sigma_ns > 0) p = llround((double)mu + (double)s->period_sigma_ns * gauss(s, trial, 2u, (uint32_t)c));
        if (p < mu / 4) p = mu / 4;
        if (p < N) p = N;
        cycle_period_ns[c] = p;
        if (c == 0 || p < shortest) shortest = p;
        if (c == 0 || p > longest) longest = p;
    }
    /* U4 */
    *prm_out = *prm;
    *ext_out = *ext;
    prm_out->period_ns = mu;
    ext_out->n_cycles = s->n_cycles;
    ext_out->cycle_period_ns = s->n_cycles > 0 ? cycle_period_ns : 0;
    ext_out->discard_ns = jitter(s, trial, 0u, ext->discard_ns, s->discard_sigma_ns, 0);
    ext_out->flat_top_ns = ext->flat_top_ns > 0 ? jitter(s, trial, 1u, ext->flat_top_ns, s->flat_top_sigma_ns, 1) : 0;
    ext_out->spot_switch_fixed_ns = jitter(s, trial, 2u, ext->spot_switch_fixed_ns, s->spot_switch_sigma_ns, 0);
    ext_out->spill_protons_max = ext->spill_protons_max > 0
        ? jitter(s, trial, 3u, ext->spill_protons_max, s->spill_protons_sigma, 1) : 0;
    prm_out->protons_per_s = jitter(s, trial, 4u, prm->protons_per_s, s->protons_per_s_sigma, 1);
    prm_out->layer_switch_ns = jitter(s, trial, 5u, prm->layer_switch_ns, s->layer_switch_sigma_ns, 0);
    if (ext->n_layer_switch > 0 && ext->layer_switch_ns) {
        for (int32_t l = 0; l < ext->n_layer_switch; ++l)
            layer_switch_ns[l] = jitter(s, trial, 6u + (uint32_t)l, ext->layer_switch_ns[l], s->layer_switch_sigma_ns, 0);
        ext_out->layer_switch_ns = layer_switch_ns;
    }
    /* U5 */
    if (ext_out->discard_ns > 0 && ext_out->discard_ns > shortest / N - 1) {
        ext_out->discard_ns = shortest / N - 1;
        if (ext_out->discard_ns < 0) ext_out->discard_ns = 0;
    }
    if (ext_out->flat_top_ns > 0 && ext_out->flat_top_ns < ext_out->discard_ns + longest + 1)
        ext_out->flat_top_ns = ext_out->discard_ns + longest + 1;
    return 0;
}
