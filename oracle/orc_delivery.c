/* oracle/orc_delivery.c -- CPU ORACLE (test infrastructure only; see orc.h).
 * Beam-delivery timeline simulation, integer arithmetic only.
 * PAPER.md:49-55 (Sec. 2.B): track breathing time against plan-delivery time -> N_g sub-plans per field "indicating
 * the number and weighting of spots which would be delivered on each breathing phase"; phase gating with a beam-on
 * window; repainting; start phase.  PAPER.md:239-245 (App. A): spot-spill, spot-switch and layer-switch times.
 * Timing model of BASELINE.json configs 3 and 5: spill at protons_per_s, scan speed (ns per um), one layer-switch
 * constant, fixed breathing period, N x layer repainting, gate bitmask. */
#include "orc.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>

typedef __int128 i128;

/* floor integer square root of a non-negative 128-bit value that fits 2^126 */
static int64_t isqrt128(i128 v)
{
    if (v <= 0) return 0;
    i128 x = (i128)sqrtl((long double)v);
    while (x * x > v) --x;
    while ((x + 1) * (x + 1) <= v) ++x;
    return (int64_t)x;
}

/* emission offset of proton i after the spill clock started: floor(i 1e9 / protons_per_s)  (D5) */
static int64_t emit_off(int64_t i, int64_t pps) { return (int64_t)(((i128)i * 1000000000) / pps); }

/* D6 + D7 from the per-(field, phase, spot) proton counts */
static int64_t emit_segments(int32_t n_fields, int32_t P, int64_t n_spots, const int64_t* counts, uint64_t total_histories,
                             orc_segment* segs, int64_t max_segs, int64_t* dropped_protons)
{
    /* D6: segments in (field, phase, spot) order, protons > 0 */
    int64_t nseg = 0; i128 c_total = 0;
    for (size_t i = 0; i < (size_t)n_fields * P * (size_t)n_spots; ++i) if (counts[i] > 0) { ++nseg; c_total += counts[i]; }
    if (!segs) return nseg;
    if (max_segs < nseg) return -1;

    /* D7: history allocation by cumulative rounding, b_k = floor(H C_k / C_total) */
    int64_t j = 0, dropped = 0; i128 C = 0; int64_t b_prev = 0;
    for (int32_t f = 0; f < n_fields; ++f)
    for (int32_t p = 0; p < P; ++p)
    for (int64_t k = 0; k < n_spots; ++k) {
        int64_t c = counts[((size_t)f * P + p) * n_spots + k];
        if (c <= 0) continue;
        C += c;
        int64_t b = total_histories ? (int64_t)(((i128)total_histories * C) / c_total) : 0;
        orc_segment* sg = &segs[j++];
        sg->field = f; sg->phase = p; sg->spot = (int32_t)k; sg->pad = 0;
        sg->protons = c; sg->first_history = b_prev; sg->n_hist = b - b_prev;
        sg->weight = sg->n_hist > 0 ? (double)c / (double)sg->n_hist : 0.0;
        if (sg->n_hist == 0) dropped += c;
        b_prev = b;
    }
    if (dropped_protons) *dropped_protons = total_histories ? dropped : 0;
    return nseg;
}

int64_t orc_simulate_delivery(int32_t n_fields, const orc_field* fields, int64_t n_spots, const orc_spot* spots,
                              const orc_delivery_params* prm, uint64_t total_histories,
                              orc_segment* segs, int64_t max_segs, int64_t* total_time_ns,
                              int64_t* dropped_protons)
{
    if (n_fields <= 0 || !fields || n_spots < 0 || (!spots && n_spots) || !prm) return -1;
    const int32_t P = prm->n_phases;
    if (P <= 0 || P > 32 || prm->period_ns < P || prm->protons_per_s <= 0 || prm->repaints <= 0) return -1;
    uint32_t all = (P == 32) ? 0xFFFFFFFFu : ((1u << P) - 1u);
    if ((prm->gate_mask & all) == 0) return -1;                      /* beam never allowed */
    const int64_t t_ph = prm->period_ns / P;                          /* D2 (reading B4) */

    /* counts[f][p][s]: protons of spot s (global id) delivered by field f in phase p */
    int64_t* counts = (int64_t*)calloc((size_t)n_fields * P * (size_t)(n_spots ? n_spots : 1), sizeof(int64_t));
    if (!counts) return -4;

    for (int32_t f = 0; f < n_fields; ++f) {
        int64_t t = 0;                                                /* D2: each field starts at t = 0 */
        int32_t sp0 = fields[f].start_phase % P; if (sp0 < 0) sp0 += P;   /* phases are counted modulo N (B2), as in _ext */
        int first_layer = 1;
        int64_t s = 0;
        while (s < n_spots) {
            if (spots[s].field != f) { ++s; continue; }
            /* a layer = maximal run (in array order) of this field's spots with the same layer id */
            int64_t e = s;
            while (e < n_spots && spots[e].field == f && spots[e].layer == spots[s].layer) ++e;
            if (!first_layer) t += prm->layer_switch_ns;              /* D3 */
            first_layer = 0;
            int have_prev = 0; int64_t px = 0, py = 0;
            for (int32_t q = 0; q < prm->repaints; ++q) {
                for (int64_t k = s; k < e; ++k) {
                    int64_t N  = llround((double)spots[k].weight * (double)prm->protons_per_weight);   /* D1 */
                    int64_t nq = N / prm->repaints + ((N % prm->repaints) > q ? 1 : 0);               /* D3 */
                    if (nq <= 0) continue;                            /* nothing to paint: spot skipped, no move */
                    int64_t x = llround((double)spots[k].x_mm * 1000.0), y = llround((double)spots[k].y_mm * 1000.0);
                    if (have_prev) {                                  /* D4: Euclidean move, integer sqrt */
                        i128 dx = x - px, dy = y - py;
                        t += isqrt128((dx * dx + dy * dy) * (i128)prm->ns_per_um * prm->ns_per_um);
                    }
                    have_prev = 1; px = x; py = y;
                    /* D5: spill walked by phase intervals */
                    int64_t remaining = nq;
                    while (remaining > 0) {
                        int64_t bin   = t / t_ph;
                        int32_t phase = (int32_t)((bin + sp0) % P);
                        int64_t tb    = (bin + 1) * t_ph;             /* next phase boundary */
                        if (!((prm->gate_mask >> phase) & 1u)) { t = tb; continue; }   /* gate off: wait (B8) */
                        /* protons with emission time t + floor(i c) < tb  <=>  i < (tb - t) pps / 1e9 */
                        i128 num = (i128)(tb - t) * prm->protons_per_s;
                        int64_t fit = (int64_t)((num + 999999999) / 1000000000);
                        int64_t n = remaining < fit ? remaining : fit;
                        counts[((size_t)f * P + phase) * n_spots + k] += n;
                        remaining -= n;
                        t += emit_off(n, prm->protons_per_s);         /* emission time of the next proton */
                    }
                }
            }
            s = e;
        }
        if (total_time_ns) total_time_ns[f] = t;
    }

    int64_t nseg = emit_segments(n_fields, P, n_spots, counts, total_histories, segs, max_segs, dropped_protons);
    free(counts);
    return nseg;
}

/* ---------------------------------------------------------------------------------------------------------------
 * Extended delivery model: the synchrotron features the paper describes beyond the config
 * model -- PAPER.md:53 iso-layered repainting with a maximum MU per spot delivery; PAPER.md:55 irregular breathing
 * (t_ph ~ N(mu, sigma)/N); PAPER.md:59 the 70 ms of beam discarded when extraction begins (after every synchrotron
 * reset, and in a gated delivery after the gate-on signal); PAPER.md:239 extraction ends when the layer is complete,
 * the charge capacity (~2 nC) is depleted or the flat-top limit (~8 s) is exceeded, followed by a reset of
 * energy-dependent duration (the "layer-switch time"); PAPER.md:245 a fixed prepare/verify part of the spot-switch
 * time.  Ref. 45's constants are not available: every value is an input, and so are the sampled breathing periods
 * (random numbers the method draws are passed in).  Steps E1-E5, integers only:
 *  E1 breathing cycle c has period per[min(c, n-1)], phase length tau_c = per_c / N, duration N tau_c; the field's
 *     timeline t = 0 is the beginning of start_phase of cycle 0.
 *  E2 before every layer but the first: t += sw(layer); then a new fill: fill_left = capacity, flat_start = t,
 *     need_discard = 1.  sw(l) = layer_switch_ns[l] if given, else the base constant.
 *  E3 paintings: with max_protons_per_paint = m > 0, painting q delivers min(m, N_s - q m) of every spot that still
 *     has protons, until none has; else the base N x scheme.
 *  E4 before every delivered spot except the first of the layer: t += move + spot_switch_fixed_ns.
 *  E5 while protons of the spot painting remain: (a) gate closed -> t = next phase boundary, need_discard = 1;
 *     (b) flat-top exceeded or fill empty -> t += sw(layer), new fill; (c) need_discard -> t += discard_ns;
 *     (d) deliver n = min(remaining, protons emitted before the next phase boundary, before the flat-top end, fill).
 * --------------------------------------------------------------------------------------------------------------- */
typedef struct { int32_t c; int64_t start; } cycle_cursor;   /* breathing cycle containing the current time */

static int64_t period_of(const orc_delivery_params* prm, const orc_delivery_ext* x, int32_t c)
{
    if (!x || !x->cycle_period_ns || x->n_cycles <= 0) return prm->period_ns;
    return x->cycle_period_ns[c < x->n_cycles ? c : x->n_cycles - 1];
}

/* phase and next phase boundary (in field time) at breathing time b = t + off; the cursor only moves forward */
static void phase_at(const orc_delivery_params* prm, const orc_delivery_ext* x, cycle_cursor* cur, int64_t b,
                     int32_t* phase, int64_t* next_boundary_b)
{
    const int32_t P = prm->n_phases;
    for (;;) {
        int64_t tau = period_of(prm, x, cur->c) / P;
        if (b < cur->start + tau * P) {
            int64_t k = (b - cur->start) / tau;
            *phase = (int32_t)k;
            *next_boundary_b = cur->start + (k + 1) * tau;
            return;
        }
        cur->start += tau * P; cur->c += 1;
    }
}

int64_t orc_simulate_delivery_ext(int32_t n_fields, const orc_field* fields, int64_t n_spots, const orc_spot* spots,
                                  const orc_delivery_params* prm, const orc_delivery_ext* x, uint64_t total_histories,
                                  orc_segment* segs, int64_t max_segs, int64_t* total_time_ns,
                                  int64_t* dropped_protons, int64_t* n_fills)
{
    if (n_fields <= 0 || !fields || n_spots < 0 || (!spots && n_spots) || !prm || !x) return -1;
    const int32_t P = prm->n_phases;
    if (P <= 0 || P > 32 || prm->period_ns < P || prm->protons_per_s <= 0 || prm->repaints <= 0) return -1;
    uint32_t all = (P == 32) ? 0xFFFFFFFFu : ((1u << P) - 1u);
    if ((prm->gate_mask & all) == 0) return -1;
    if (x->discard_ns < 0 || x->spill_protons_max < 0 || x->flat_top_ns < 0 || x->spot_switch_fixed_ns < 0 ||
        x->max_protons_per_paint < 0) return -1;
    int64_t per_max = prm->period_ns, per_min = prm->period_ns;
    if (x->cycle_period_ns && x->n_cycles > 0) {
        per_max = per_min = x->cycle_period_ns[0];
        for (int32_t c = 0; c < x->n_cycles; ++c) {
            if (x->cycle_period_ns[c] < P) return -1;
            if (x->cycle_period_ns[c] > per_max) per_max = x->cycle_period_ns[c];
            if (x->cycle_period_ns[c] < per_min) per_min = x->cycle_period_ns[c];
        }
    }
    /* the discard must fit inside one phase, or a gated extraction could never start */
    if (x->discard_ns > 0 && x->discard_ns >= per_min / P) return -1;
    /* a fill must be able to outlast the longest gate hold plus the discard, or extraction never starts */
    if (x->flat_top_ns > 0 && x->flat_top_ns <= x->discard_ns + per_max) return -1;

    int64_t* counts = (int64_t*)calloc((size_t)n_fields * P * (size_t)(n_spots ? n_spots : 1), sizeof(int64_t));
    if (!counts) return -4;
    int64_t fills = 0;

    for (int32_t f = 0; f < n_fields; ++f) {
        int64_t t = 0;
        cycle_cursor cur = { 0, 0 };
        int32_t sp0 = fields[f].start_phase % P; if (sp0 < 0) sp0 += P;     /* phases are counted modulo N (B2) */
        const int64_t off = (int64_t)sp0 * (period_of(prm, x, 0) / P);                      /* E1 */
        int first_layer = 1;
        int64_t s = 0;
        while (s < n_spots) {
            if (spots[s].field != f) { ++s; continue; }
            int64_t e = s;
            while (e < n_spots && spots[e].field == f && spots[e].layer == spots[s].layer) ++e;
            const int32_t lay = spots[s].layer;
            const int64_t sw = (x->layer_switch_ns && lay >= 0 && lay < x->n_layer_switch) ? x->layer_switch_ns[lay]
                                                                                           : prm->layer_switch_ns;
            if (!first_layer) t += sw;                                                          /* E2 */
            first_layer = 0;
            int64_t fill_left = x->spill_protons_max, flat_start = t; int need_discard = 1; fills += 1;
            int have_prev = 0; int64_t px = 0, py = 0;
            const int64_t m = x->max_protons_per_paint;
            for (int64_t q = 0; ; ++q) {                                                        /* E3 */
                int any = 0;
                if (m == 0 && q >= prm->repaints) break;
                for (int64_t k = s; k < e; ++k) {
                    int64_t N = llround((double)spots[k].weight * (double)prm->protons_per_weight);
                    int64_t nq;
                    if (m > 0) { nq = N - q * m; if (nq > m) nq = m; }
                    else       nq = N / prm->repaints + ((N % prm->repaints) > q ? 1 : 0);
                    if (nq <= 0) continue;
                    any = 1;
                    int64_t X = llround((double)spots[k].x_mm * 1000.0), Y = llround((double)spots[k].y_mm * 1000.0);
                    if (have_prev) {                                                            /* E4 */
                        i128 dx = X - px, dy = Y - py;
                        t += isqrt128((dx * dx + dy * dy) * (i128)prm->ns_per_um * prm->ns_per_um) + x->spot_switch_fixed_ns;
                    }
                    have_prev = 1; px = X; py = Y;
                    int64_t remaining = nq;
                    while (remaining > 0) {                                                     /* E5 */
                        int32_t ph; int64_t nb;
                        phase_at(prm, x, &cur, t + off, &ph, &nb);
                        int32_t phase = ph;
                        int64_t tb = nb - off;
                        if (!((prm->gate_mask >> phase) & 1u)) { t = tb; need_discard = 1; continue; }            /* a */
                        if ((x->flat_top_ns > 0 && t - flat_start >= x->flat_top_ns) ||
                            (x->spill_protons_max > 0 && fill_left == 0)) {                                        /* b */
                            t += sw; fill_left = x->spill_protons_max; flat_start = t; need_discard = 1; fills += 1;
                            continue;
                        }
                        if (need_discard) { t += x->discard_ns; need_discard = 0; if (x->discard_ns > 0) continue; }  /* c */
                        i128 num = (i128)(tb - t) * prm->protons_per_s;                                             /* d */
                        int64_t n = (int64_t)((num + 999999999) / 1000000000);
                        if (x->flat_top_ns > 0) {
                            i128 nf = (i128)(flat_start + x->flat_top_ns - t) * prm->protons_per_s;
                            int64_t fitf = (int64_t)((nf + 999999999) / 1000000000);
                            if (fitf < n) n = fitf;
                        }
                        if (x->spill_protons_max > 0 && fill_left < n) n = fill_left;
                        if (remaining < n) n = remaining;
                        counts[((size_t)f * P + phase) * n_spots + k] += n;
                        remaining -= n;
                        if (x->spill_protons_max > 0) fill_left -= n;
                        t += emit_off(n, prm->protons_per_s);
                    }
                }
                if (m > 0 && !any) break;
            }
            s = e;
        }
        if (total_time_ns) total_time_ns[f] = t;
    }
    if (n_fills) *n_fills = fills;
    int64_t nseg = emit_segments(n_fields, P, n_spots, counts, total_histories, segs, max_segs, dropped_protons);
    free(counts);
    return nseg;
}
