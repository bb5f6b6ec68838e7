"""Pins for the uncertainty-trial sampler of the oracle (orc_sample_trial, steps U0-U5).  CPU only.

Pinned against things other than itself: the counter layout and the uniform of the first draw through an independent
Python Philox (the Random123 known answers pin that one in test_oracle_tiny_full.py), the distributions the paper
states (discrete uniforms, Gaussians) through their moments and frequencies, determinism and independence of trials,
the degenerate case (all sigmas zero = the plain extended delivery), and proton conservation in every trial."""
import math

import numpy as np
import pytest

import oracle as orc
from paper_1809_03927_b200 import synth
from test_oracle_tiny_full import philox

S = 10 ** 9
SPEC = dict(seed=(7 << 32) | 99, n_trials=4000, n_cycles=6, period_lo_ns=3 * S, period_hi_ns=7 * S, period_step_ns=S,
            period_sigma_ns=300_000_000, discard_sigma_ns=5_000_000, flat_top_sigma_ns=200_000_000,
            spot_switch_sigma_ns=200_000, layer_switch_sigma_ns=100_000_000, spill_protons_sigma=10 ** 9,
            protons_per_s_sigma=5 * 10 ** 7)
EXT = dict(discard_ns=70_000_000, spill_protons_max=12 * 10 ** 9, flat_top_ns=8 * S + 2 * S, spot_switch_fixed_ns=2_000_000,
           layer_switch_ns=np.array([2 * S, 2 * S + 10 ** 8, 2 * S + 2 * 10 ** 8], np.int64), max_protons_per_paint=0)


def u01(x):
    return ((x >> 9) + 0.5) / 8388608.0


def test_first_draws_against_an_independent_philox():
    prm = synth.make_delivery(n_phases=10, period_s=4.0)
    t = orc.sample_trial(SPEC, 17, 5, prm, **EXT)
    key = (SPEC["seed"] & 0xFFFFFFFF, SPEC["seed"] >> 32)
    # U1: counter (block 0, stream 0, trial, tag)
    o = philox((0, 0, 17, 0x55545249), key)
    assert int(t["prm"]["period_ns"][0]) == 3 * S + S * math.floor(u01(o[0]) * 5)
    # U2: field f uses word f mod 4 of block f / 4 of stream 1
    o0, o1 = philox((0, 1, 17, 0x55545249), key), philox((1, 1, 17, 0x55545249), key)
    assert [int(x) for x in t["start_phase"]] == [math.floor(u01(o0[f]) * 10) for f in range(4)] + \
        [math.floor(u01(o1[0]) * 10)]
    # U3: cycle 2 = block 2 of stream 2, Box-Muller cosine branch
    o = philox((2, 2, 17, 0x55545249), key)
    g = math.sqrt(-2.0 * math.log(u01(o[0]))) * math.cos(2.0 * math.pi * u01(o[1]))
    mu = int(t["prm"]["period_ns"][0])
    assert int(t["ext"]["cycle_period_ns"][2]) == max(round(mu + 3e8 * g), mu // 4)
    # U4: parameter 4 (spill rate) = block 4 of stream 3
    o = philox((4, 3, 17, 0x55545249), key)
    g = math.sqrt(-2.0 * math.log(u01(o[0]))) * math.cos(2.0 * math.pi * u01(o[1]))
    assert int(t["prm"]["protons_per_s"][0]) == max(round(1e9 + 5e7 * g), 1)


def test_distributions_match_the_papers_statement():
    prm = synth.make_delivery(n_phases=10, period_s=4.0, layer_switch_s=2.0)
    T = SPEC["n_trials"]
    tr = [orc.sample_trial(SPEC, i, 3, prm, **EXT) for i in range(T)]
    # breathing period ~ discrete U{3,4,5,6,7} s
    mu = np.array([int(t["prm"]["period_ns"][0]) for t in tr])
    assert set(mu) == {3 * S, 4 * S, 5 * S, 6 * S, 7 * S}
    freq = np.array([(mu == k * S).mean() for k in range(3, 8)])
    assert np.abs(freq - 0.2).max() < 4.5 * math.sqrt(0.16 / T)
    # starting phase ~ discrete U{CT_0 .. CT_90}, independent between fields
    sp = np.array([t["start_phase"] for t in tr])
    assert sp.min() == 0 and sp.max() == 9
    for f in range(3):
        assert np.abs(np.bincount(sp[:, f], minlength=10) / T - 0.1).max() < 4.5 * math.sqrt(0.09 / T)
    assert abs(np.corrcoef(sp[:, 0], sp[:, 1])[0, 1]) < 0.06
    # t_ph ~ N(mu, sigma)/N per cycle: standardised cycle periods are N(0, 1)
    z = np.array([(t["ext"]["cycle_period_ns"] - int(t["prm"]["period_ns"][0])) / 3e8 for t in tr]).ravel()
    assert abs(z.mean()) < 4 / math.sqrt(z.size) and abs(z.std() - 1.0) < 0.02
    assert abs((np.abs(z) < 1).mean() - 0.6827) < 0.012
    # synchrotron parameters ~ N(central, sigma)
    for get, central, sigma in [
            (lambda t: t["ext"]["discard_ns"], 70e6, 5e6),
            (lambda t: t["ext"]["spot_switch_fixed_ns"], 2e6, 2e5),
            (lambda t: t["ext"]["spill_protons_max"], 12e9, 1e9),
            (lambda t: int(t["prm"]["protons_per_s"][0]), 1e9, 5e7),
            (lambda t: int(t["prm"]["layer_switch_ns"][0]), 2e9, 1e8),
            (lambda t: int(t["ext"]["layer_switch_ns"][2]), 2.2e9, 1e8)]:
        v = np.array([get(t) for t in tr], np.float64)
        assert abs(v.mean() - central) < 4.5 * sigma / math.sqrt(T)
        assert abs(v.std() / sigma - 1.0) < 0.05
    # different parameters are drawn from different blocks: uncorrelated
    a = np.array([t["ext"]["discard_ns"] for t in tr], np.float64)
    b = np.array([t["ext"]["spot_switch_fixed_ns"] for t in tr], np.float64)
    assert abs(np.corrcoef(a, b)[0, 1]) < 0.06


def test_determinism_trial_independence_and_degenerate_case():
    prm = synth.make_delivery(n_phases=10, period_s=4.5, layer_switch_s=2.0)
    a = orc.sample_trial(SPEC, 5, 2, prm, **EXT)
    b = orc.sample_trial(SPEC, 5, 2, prm, **EXT)
    assert a["prm"].tobytes() == b["prm"].tobytes() and (a["ext"]["cycle_period_ns"] == b["ext"]["cycle_period_ns"]).all()
    c = orc.sample_trial(dict(SPEC, seed=SPEC["seed"] + 1), 5, 2, prm, **EXT)
    assert (a["ext"]["cycle_period_ns"] != c["ext"]["cycle_period_ns"]).any()
    # a trial does not depend on how many trials are requested, nor on how many fields are sampled before it
    d = orc.sample_trial(dict(SPEC, n_trials=6), 5, 7, prm, **EXT)
    assert (d["start_phase"][:2] == a["start_phase"]).all() and d["prm"].tobytes() == a["prm"].tobytes()
    # all sigmas zero, period not sampled: the central values come back unchanged
    zero = dict(seed=3, n_trials=1, n_cycles=0, period_lo_ns=0, period_hi_ns=0, period_step_ns=0, period_sigma_ns=0,
                discard_sigma_ns=0, flat_top_sigma_ns=0, spot_switch_sigma_ns=0, layer_switch_sigma_ns=0,
                spill_protons_sigma=0, protons_per_s_sigma=0)
    e = orc.sample_trial(zero, 0, 2, prm, **EXT)
    assert e["prm"].tobytes() == np.ascontiguousarray(prm, orc.DELIV_DT).tobytes()
    assert e["ext"]["cycle_period_ns"] is None and e["ext"]["discard_ns"] == EXT["discard_ns"]
    assert (e["ext"]["layer_switch_ns"] == EXT["layer_switch_ns"]).all() and e["ext"]["flat_top_ns"] == EXT["flat_top_ns"]
    with pytest.raises(ValueError):
        orc.sample_trial(SPEC, SPEC["n_trials"], 2, prm, **EXT)


def test_feasibility_clamps():
    prm = synth.make_delivery(n_phases=10, period_s=4.0)
    spec = dict(SPEC, period_lo_ns=S // 2, period_hi_ns=S // 2, period_step_ns=0, period_sigma_ns=S, n_cycles=8,
                discard_sigma_ns=60_000_000, flat_top_sigma_ns=3 * S)
    for i in range(200):
        t = orc.sample_trial(spec, i, 1, prm, discard_ns=40_000_000, flat_top_ns=S)
        cyc = t["ext"]["cycle_period_ns"]
        assert cyc.min() >= max((S // 2) // 4, 10)                       # U3 floor
        assert 0 <= t["ext"]["discard_ns"] <= cyc.min() // 10 - 1         # U5
        assert t["ext"]["flat_top_ns"] >= t["ext"]["discard_ns"] + cyc.max() + 1


def test_every_trial_delivers_every_proton():
    rng = np.random.default_rng(3)
    fields = np.concatenate([synth.make_field((0, 0, 1), (1, 0, 0), (0, 1, 0), (0, 0, 0), 0) for _ in range(2)])
    spots = np.array([(f, l, rng.uniform(-20, 20), rng.uniform(-20, 20), 100.0 + 10 * l, 4.0, rng.uniform(0.5, 1.5))
                      for f in range(2) for l in range(3) for _ in range(6)], synth.SPOT_DT)
    prm = synth.make_delivery(n_phases=10, period_s=0.05, protons_per_weight=2 * 10 ** 6, layer_switch_s=0.02,
                              gate_mask=0b0011111000)
    spec = dict(seed=11, n_trials=25, n_cycles=12, period_lo_ns=30_000_000, period_hi_ns=70_000_000,
                period_step_ns=10_000_000, period_sigma_ns=3_000_000, discard_sigma_ns=50_000, flat_top_sigma_ns=2_000_000,
                spot_switch_sigma_ns=2_000, layer_switch_sigma_ns=1_000_000, spill_protons_sigma=10 ** 5,
                protons_per_s_sigma=5 * 10 ** 7)
    ext = dict(discard_ns=700_000, spill_protons_max=3 * 10 ** 6, flat_top_ns=90_000_000, spot_switch_fixed_ns=20_000)
    N_s = np.rint(spots["weight"].astype(np.float64) * 2 * 10 ** 6).astype(np.int64)
    seen = set()
    for i in range(25):
        t = orc.sample_trial(spec, i, 2, prm, **ext)
        f = fields.copy(); f["start_phase"] = t["start_phase"]
        segs, tt, dropped, fills = orc.simulate_delivery_ext(f, spots, t["prm"], 10_000, **t["ext"])
        got = np.zeros(len(spots), np.int64)
        np.add.at(got, segs["spot"], segs["protons"])
        assert (got == N_s).all()                                        # sum over phases = N_s, every trial
        assert set(int(p) for p in segs["phase"]) <= {3, 4, 5, 6, 7}
        assert int(segs["n_hist"].sum()) == 10_000
        seen.add(segs["protons"].tobytes())
    assert len(seen) == 25                                               # the trials really differ
