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
        const int32_t sp0 = fields[f].start_phase;
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

    /* D6: segments in (field, phase, spot) order, protons > 0 */
    int64_t nseg = 0; i128 c_total = 0;
    for (size_t i = 0; i < (size_t)n_fields * P * (size_t)n_spots; ++i) if (counts[i] > 0) { ++nseg; c_total += counts[i]; }
    if (!segs) { free(counts); return nseg; }
    if (max_segs < nseg) { free(counts); return -1; }

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
    free(counts);
    return nseg;
}
