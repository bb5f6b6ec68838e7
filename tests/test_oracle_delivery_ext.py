"""Pins for the extended delivery oracle (orc_simulate_delivery_ext, steps E1-E5):
reduction to the base model, a per-PROTON brute force that keeps one clock per proton (no interval counting),
closed forms for the number of synchrotron fills and the total time, and conservation.  CPU only."""
import math

import numpy as np
import pytest

import oracle as orc
from paper_1809_03927_b200 import synth
from test_oracle_delivery import small_plan


def brute_force_ext(fields, spots, prm, cyc=None, discard=0, cap=0, flat=0, fixed=0, lsw=None, mpp=0):
    """Every proton individually: find its phase from the list of phase boundaries, check gate / fill / flat-top /
    discard state before it is emitted."""
    P = int(prm["n_phases"][0]); pps = int(prm["protons_per_s"][0]); gate = int(prm["gate_mask"][0])
    rep = int(prm["repaints"][0]); base_sw = int(prm["layer_switch_ns"][0]); nsu = int(prm["ns_per_um"][0])
    ppw = int(prm["protons_per_weight"][0])
    periods = [int(prm["period_ns"][0])] if cyc is None else [int(c) for c in cyc]
    counts, totals, fills = {}, [], 0
    for f in range(len(fields)):
        # explicit list of (start, end, phase) breathing bins, long enough for the plan
        off = (int(fields["start_phase"][f]) % P) * (periods[0] // P)        # phases count modulo N
        bins, b = [], 0
        for c in range(4000):
            tau = periods[min(c, len(periods) - 1)] // P
            for k in range(P):
                bins.append((b - off, b + tau - off, k)); b += tau
        bi = 0

        def locate(t):
            nonlocal bi
            while not (bins[bi][0] <= t < bins[bi][1]):
                bi += 1
            return bins[bi]

        ids = [i for i in range(len(spots)) if spots["field"][i] == f]
        layers = []
        for i in ids:
            if layers and spots["layer"][layers[-1][-1]] == spots["layer"][i]:
                layers[-1].append(i)
            else:
                layers.append([i])
        t = 0
        for li, layer in enumerate(layers):
            lay = int(spots["layer"][layer[0]])
            sw = int(lsw[lay]) if (lsw is not None and 0 <= lay < len(lsw)) else base_sw
            if li:
                t += sw
            fill_left, flat_start, need_discard = cap, t, True; fills += 1
            prev = None
            N = {i: int(round(float(spots["weight"][i]) * ppw)) for i in layer}
            q = 0
            while True:
                if mpp == 0 and q >= rep:
                    break
                any_ = False
                for i in layer:
                    nq = min(mpp, N[i] - q * mpp) if mpp else N[i] // rep + (1 if N[i] % rep > q else 0)
                    if nq <= 0:
                        continue
                    any_ = True
                    x = int(round(float(spots["x_mm"][i]) * 1000.0)); y = int(round(float(spots["y_mm"][i]) * 1000.0))
                    if prev is not None:
                        t += math.isqrt(((x - prev[0]) ** 2 + (y - prev[1]) ** 2) * nsu ** 2) + fixed
                    prev = (x, y)
                    t0, j = t, 0                                  # spill clock start, protons since it started
                    for _ in range(nq):
                        while True:
                            te = t0 + (j * 10 ** 9) // pps        # emission time of this proton on the current clock
                            lo, hi, ph = locate(t0)
                            if not (gate >> ph) & 1:              # clock started with the gate closed: hold
                                t0, j, need_discard = hi, 0, True
                                continue
                            if te >= hi:                          # would be emitted in a later phase: restart there
                                t0, j = te, 0
                                continue
                            if (flat and te - flat_start >= flat) or (cap and fill_left == 0):
                                t0, j = te + sw, 0                # synchrotron reset, new fill
                                fill_left, flat_start, need_discard = cap, t0, True; fills += 1
                                continue
                            if need_discard:
                                need_discard = False
                                if discard:
                                    t0, j = te + discard, 0
                                    continue
                            break
                        counts[(f, ph, i)] = counts.get((f, ph, i), 0) + 1
                        j += 1
                        if cap:
                            fill_left -= 1
                    t = t0 + (j * 10 ** 9) // pps
                q += 1
                if mpp and not any_:
                    break
        totals.append(t)
    return counts, totals, fills


CASES = {
    "discard_gated": dict(gate_mask=0b01101, ext=dict(discard=350)),
    "capacity": dict(ext=dict(cap=4000)),
    "flat_top": dict(ext=dict(flat=30_000, discard=200)),
    "irregular": dict(gate_mask=0b10110, ext=dict(cyc=[20_000, 26_500, 17_005, 23_330], discard=120)),
    "isolayer": dict(ext=dict(mpp=700, fixed=55)),
    "layer_switch_table": dict(ext=dict(lsw=[0, 5_000, 900], cap=5000, fixed=10)),
    "everything": dict(gate_mask=0b11010, protons_per_s=7 * 10 ** 8,
                       ext=dict(cyc=[21_000, 19_000, 24_000], discard=300, cap=2500, flat=40_000, fixed=33,
                                lsw=[0, 4_000, 2_500], mpp=900)),
}


@pytest.mark.parametrize("case", list(CASES))
def test_brute_force_per_proton(case):
    rng = np.random.default_rng(21)
    fields, spots = small_plan(rng)
    spec = dict(CASES[case]); ext = spec.pop("ext")
    kw = dict(n_phases=5, period_s=2.0e-5, protons_per_weight=3000, protons_per_s=10 ** 9, ns_per_um=1,
              layer_switch_s=3.3e-6, repaints=2)
    kw.update(spec)
    prm = synth.make_delivery(**kw)
    segs, tt, dropped, fills = orc.simulate_delivery_ext(
        fields, spots, prm, 0, cycle_period_ns=ext.get("cyc"), discard_ns=ext.get("discard", 0),
        spill_protons_max=ext.get("cap", 0), flat_top_ns=ext.get("flat", 0), spot_switch_fixed_ns=ext.get("fixed", 0),
        layer_switch_ns=ext.get("lsw"), max_protons_per_paint=ext.get("mpp", 0))
    counts, totals, bf_fills = brute_force_ext(fields, spots, prm, **ext)
    got = {(int(s["field"]), int(s["phase"]), int(s["spot"])): int(s["protons"]) for s in segs}
    assert got == counts
    assert [int(x) for x in tt] == totals and fills == bf_fills
    assert len({k[1] for k in got}) > 1


def test_all_off_is_the_base_model():
    rng = np.random.default_rng(22)
    fields, spots = small_plan(rng, n_fields=2, n_layers=4, per_layer=7, start_phases=(1, 4))
    for kw in [dict(), dict(gate_mask=0b0011111000, repaints=4)]:
        prm = synth.make_delivery(n_phases=10, period_s=0.004, protons_per_weight=10 ** 6, layer_switch_s=0.001, **kw)
        a, ta, da = orc.simulate_delivery(fields, spots, prm, 12345)
        b, tb, db, fills = orc.simulate_delivery_ext(fields, spots, prm, 12345)
        assert a.tobytes() == b.tobytes() and (ta == tb).all() and da == db
        assert fills == 2 * 4                                     # one fill per layer and field
        # a uniform table of cycle periods equal to the base period changes nothing either
        c, tc, _, _ = orc.simulate_delivery_ext(fields, spots, prm, 12345, cycle_period_ns=[4_000_000] * 3)
        assert a.tobytes() == c.tobytes() and (ta == tc).all()


def test_fill_count_and_total_time_closed_forms():
    # ungated, one field, one layer: fills = ceil(total protons / capacity); every extra fill costs one reset, every
    # fill one discard:  T = sum spill + sum moves + (fills - 1) sw + fills discard   (1 ns per proton)
    rng = np.random.default_rng(23)
    fields, spots = small_plan(rng, n_fields=1, n_layers=1, per_layer=9, start_phases=(0,))
    prm = synth.make_delivery(n_phases=10, period_s=4.0, protons_per_weight=10 ** 6, layer_switch_s=0.5, ns_per_um=100)
    N = np.rint(spots["weight"].astype(np.float64) * 10 ** 6).astype(np.int64)
    cap, discard = 1_300_000, 70_000_000
    segs, tt, _, fills = orc.simulate_delivery_ext(fields, spots, prm, 0, spill_protons_max=cap, discard_ns=discard)
    assert fills == -(-int(N.sum()) // cap)
    x = np.rint(spots["x_mm"].astype(np.float64) * 1000).astype(np.int64)
    y = np.rint(spots["y_mm"].astype(np.float64) * 1000).astype(np.int64)
    moves = sum(math.isqrt(int((x[i] - x[i - 1]) ** 2 + (y[i] - y[i - 1]) ** 2) * 100 ** 2) for i in range(1, len(x)))
    assert int(tt[0]) == int(N.sum()) + moves + (fills - 1) * 500_000_000 + fills * discard
    per_spot = np.zeros(len(spots), np.int64)
    np.add.at(per_spot, segs["spot"], segs["protons"])
    assert (per_spot == N).all()                                  # conservation
    # iso-layered repainting: paintings = ceil(max N_s / m); same protons per spot; more moves => longer delivery
    segs2, tt2, _, _ = orc.simulate_delivery_ext(fields, spots, prm, 0, max_protons_per_paint=200_000)
    per_spot2 = np.zeros(len(spots), np.int64)
    np.add.at(per_spot2, segs2["spot"], segs2["protons"])
    assert (per_spot2 == N).all() and tt2[0] > orc.simulate_delivery(fields, spots, prm, 0)[1][0]


def test_bad_parameters_are_rejected():
    rng = np.random.default_rng(24)
    fields, spots = small_plan(rng, n_fields=1, start_phases=(0,))
    prm = synth.make_delivery(n_phases=10, period_s=4.0)
    with pytest.raises(ValueError):
        orc.simulate_delivery_ext(fields, spots, prm, 0, discard_ns=400_000_000)          # discard >= one phase
    with pytest.raises(ValueError):
        orc.simulate_delivery_ext(fields, spots, prm, 0, flat_top_ns=3_000_000_000)       # flat-top <= period + discard
    with pytest.raises(ValueError):
        orc.simulate_delivery_ext(fields, spots, prm, 0, cycle_period_ns=[4_000_000_000, 5])
