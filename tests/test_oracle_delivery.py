"""Pins for the delivery-timeline oracle: invariants and per-proton brute force.  CPU only."""
import math

import numpy as np
import pytest

import oracle as orc
from paper_1809_03927_b200 import synth


def small_plan(rng, n_fields=2, n_layers=3, per_layer=5, start_phases=(0, 3)):
    fields = np.concatenate([synth.make_field((0, 0, 1), (1, 0, 0), (0, 1, 0), (0, 0, 0), start_phases[f])
                             for f in range(n_fields)])
    spots = []
    for f in range(n_fields):
        for l in range(n_layers):
            for _ in range(per_layer):
                spots.append((f, l, rng.uniform(-30, 30), rng.uniform(-30, 30), 100.0 + 10 * l, 4.0,
                              rng.uniform(0.5, 1.5)))
    return fields, np.array(spots, synth.SPOT_DT)


def brute_force(fields, spots, prm):
    """Per-PROTON walk (no closed-form counting): every proton gets its own emission time and phase."""
    P = int(prm["n_phases"][0]); t_ph = int(prm["period_ns"][0]) // P
    pps = int(prm["protons_per_s"][0]); gate = int(prm["gate_mask"][0]); rep = int(prm["repaints"][0])
    counts = {}
    totals = []
    for f in range(len(fields)):
        sp0 = int(fields["start_phase"][f])
        ids = [i for i in range(len(spots)) if spots["field"][i] == f]
        layers = []
        for i in ids:
            if layers and spots["layer"][layers[-1][-1]] == spots["layer"][i]:
                layers[-1].append(i)
            else:
                layers.append([i])
        t = 0
        for li, layer in enumerate(layers):
            if li:
                t += int(prm["layer_switch_ns"][0])
            prev = None
            for q in range(rep):
                for i in layer:
                    N = int(round(float(spots["weight"][i]) * int(prm["protons_per_weight"][0])))
                    nq = N // rep + (1 if N % rep > q else 0)
                    if nq == 0:
                        continue
                    x = int(round(float(spots["x_mm"][i]) * 1000.0)); y = int(round(float(spots["y_mm"][i]) * 1000.0))
                    if prev is not None:
                        t += math.isqrt(((x - prev[0]) ** 2 + (y - prev[1]) ** 2) * int(prm["ns_per_um"][0]) ** 2)
                    prev = (x, y)
                    t0, j, done = t, 0, 0                     # spill clock start, protons since clock start
                    while done < nq:
                        te = t0 + (j * 10 ** 9) // pps        # emission time of the next proton
                        tb0 = (t0 // t_ph + 1) * t_ph
                        if not (gate >> ((t0 // t_ph + sp0) % P)) & 1:
                            t0, j = tb0, 0                    # gate closed when the clock started: wait for boundary
                            continue
                        if te >= tb0:                         # crossed into the next phase: restart the clock there
                            t0, j = te, 0
                            continue
                        ph = (te // t_ph + sp0) % P
                        counts[(f, ph, i)] = counts.get((f, ph, i), 0) + 1
                        j += 1; done += 1
                    t = t0 + (j * 10 ** 9) // pps
        totals.append(t)
    return counts, totals


@pytest.mark.parametrize("case", ["plain", "gated", "repaint", "gated_repaint_slowspill"])
def test_brute_force_per_proton(case):
    rng = np.random.default_rng(7)
    fields, spots = small_plan(rng)
    kw = dict(n_phases=5, period_s=2.0e-5, protons_per_weight=3000, protons_per_s=10 ** 9, ns_per_um=1,
              layer_switch_s=3.3e-6)
    if case == "gated":
        kw["gate_mask"] = 0b01101
    if case == "repaint":
        kw["repaints"] = 4
    if case == "gated_repaint_slowspill":
        kw.update(repaints=3, gate_mask=0b10010, protons_per_s=7 * 10 ** 8)
    prm = synth.make_delivery(**kw)
    segs, tt, dropped = orc.simulate_delivery(fields, spots, prm, 0)
    counts, totals = brute_force(fields, spots, prm)
    got = {(int(s["field"]), int(s["phase"]), int(s["spot"])): int(s["protons"]) for s in segs}
    assert got == counts
    assert [int(x) for x in tt] == totals
    # D6 ordering
    keys = [(int(s["field"]), int(s["phase"]), int(s["spot"])) for s in segs]
    assert keys == sorted(keys)
    assert len({k[1] for k in keys}) > 1                     # the plan really straddles phases


def test_conservation_and_single_phase():
    rng = np.random.default_rng(8)
    fields, spots = small_plan(rng, n_fields=1, start_phases=(0,))
    N = np.rint(spots["weight"].astype(np.float64) * 10 ** 6).astype(np.int64)
    for P, gate in [(10, None), (10, 0b0011111000), (4, 0b0101)]:
        prm = synth.make_delivery(n_phases=P, period_s=0.004, protons_per_weight=10 ** 6, gate_mask=gate,
                                  layer_switch_s=0.001, repaints=2)
        segs, tt, _ = orc.simulate_delivery(fields, spots, prm, 0)
        per_spot = np.zeros(len(spots), np.int64)
        np.add.at(per_spot, segs["spot"], segs["protons"])
        assert (per_spot == N).all()                         # sum_p list[f][p][s] = N_s
        if gate is not None:
            assert all((gate >> int(p)) & 1 for p in segs["phase"])
    # single phase: the whole plan lands on it, spot by spot (second 3D comparison test)
    prm = synth.make_delivery(n_phases=1, protons_per_weight=10 ** 6)
    segs, _, _ = orc.simulate_delivery(fields, spots, prm, 0)
    assert (segs["spot"] == np.arange(len(spots))).all() and (segs["protons"] == N).all()
    assert (segs["phase"] == 0).all()


def test_ungated_total_time_closed_form():
    # total = sum spill + sum moves + (L-1) switch, at 1 ns per proton (SURVEY pins: Delivery)
    rng = np.random.default_rng(9)
    fields, spots = small_plan(rng, n_fields=1, n_layers=4, per_layer=6, start_phases=(2,))
    prm = synth.make_delivery(n_phases=10, period_s=4.0, protons_per_weight=10 ** 7, layer_switch_s=1.0, ns_per_um=100)
    _, tt, _ = orc.simulate_delivery(fields, spots, prm, 0)
    N = np.rint(spots["weight"].astype(np.float64) * 10 ** 7).astype(np.int64)
    x = np.rint(spots["x_mm"].astype(np.float64) * 1000).astype(np.int64)
    y = np.rint(spots["y_mm"].astype(np.float64) * 1000).astype(np.int64)
    moves = 0
    for i in range(1, len(spots)):
        if spots["layer"][i] == spots["layer"][i - 1]:
            moves += math.isqrt(int((x[i] - x[i - 1]) ** 2 + (y[i] - y[i - 1]) ** 2) * 100 * 100)
    assert int(tt[0]) == int(N.sum()) + moves + 3 * 10 ** 9


def test_start_phase_rotates_the_lists():
    rng = np.random.default_rng(10)
    fields, spots = small_plan(rng, n_fields=1, start_phases=(0,))
    prm = synth.make_delivery(n_phases=6, period_s=0.006, protons_per_weight=10 ** 6, layer_switch_s=0.0005)
    a, _, _ = orc.simulate_delivery(fields, spots, prm, 0)
    f2 = fields.copy(); f2["start_phase"] = 4
    b, _, _ = orc.simulate_delivery(f2, spots, prm, 0)
    da = {((int(s["phase"]) + 4) % 6, int(s["spot"])): int(s["protons"]) for s in a}
    db = {(int(s["phase"]), int(s["spot"])): int(s["protons"]) for s in b}
    assert da == db
    # phases are counted modulo N (reading B2): start phases -2 and 10 are start phase 4 of 6, in both oracle entries
    for sp in (-2, 10):
        f3 = fields.copy(); f3["start_phase"] = sp
        c, _, _ = orc.simulate_delivery(f3, spots, prm, 0)
        assert c.tobytes() == b.tobytes()
        cx, _, _, _ = orc.simulate_delivery_ext(f3, spots, prm, 0)
        assert cx.tobytes() == b.tobytes()


def test_history_allocation_d7():
    rng = np.random.default_rng(12)
    fields, spots = small_plan(rng)
    prm = synth.make_delivery(n_phases=5, period_s=0.003, protons_per_weight=10 ** 6, layer_switch_s=0.0004)
    H = 12345
    segs, _, dropped = orc.simulate_delivery(fields, spots, prm, H)
    assert int(segs["n_hist"].sum()) == H
    assert (segs["first_history"] == np.concatenate([[0], np.cumsum(segs["n_hist"])[:-1]])).all()
    C = np.cumsum([int(p) for p in segs["protons"]], dtype=object)
    b = [(H * int(c)) // int(C[-1]) for c in C]
    assert [int(x) for x in (segs["first_history"] + segs["n_hist"])] == b
    live = segs["n_hist"] > 0
    assert np.allclose(segs["weight"][live], segs["protons"][live] / segs["n_hist"][live], rtol=1e-15)
    assert dropped == int(segs["protons"][~live].sum())
    # far fewer histories than segments: some segments are dropped and reported
    segs2, _, dropped2 = orc.simulate_delivery(fields, spots, prm, 7)
    assert int(segs2["n_hist"].sum()) == 7 and dropped2 > 0


def test_bad_arguments():
    rng = np.random.default_rng(13)
    fields, spots = small_plan(rng)
    with pytest.raises(ValueError):
        orc.simulate_delivery(fields, spots, synth.make_delivery(n_phases=4, gate_mask=0), 10)
    with pytest.raises(ValueError):
        orc.simulate_delivery(fields, spots, synth.make_delivery(n_phases=4, repaints=0), 10)
