"""The library's uncertainty-trial sampler and per-trial delivery (pbs4d_sample_delivery_trial + the extended host
simulator) against the oracle's: byte-equal draws and byte-equal sub-plans for the paper's 25 trials on
the full config-5 plan (BASELINE.json:11).  CPU only (device-free entry points)."""
import numpy as np
import pytest

import oracle as orc
from paper_1809_03927_b200 import binding, synth

S = 10 ** 9
SPEC = dict(seed=(3 << 32) | 20181809, n_trials=25, n_cycles=40, period_lo_ns=3 * S, period_hi_ns=7 * S,
            period_step_ns=S, period_sigma_ns=400_000_000, discard_sigma_ns=5_000_000, flat_top_sigma_ns=300_000_000,
            spot_switch_sigma_ns=200_000, layer_switch_sigma_ns=150_000_000, spill_protons_sigma=2 * 10 ** 9,
            protons_per_s_sigma=4 * 10 ** 7)
# central values in the spirit of PAPER.md:59, 239 (70 ms discard, ~2 nC = 1.25e10 protons, ~8 s flat top, ~2 s reset)
EXT = dict(discard_ns=70_000_000, spill_protons_max=12_500_000_000, flat_top_ns=16 * S, spot_switch_fixed_ns=2_000_000,
           layer_switch_ns=np.array([2 * S - 20_000_000 * l for l in range(25)], np.int64))


@pytest.fixture(scope="module")
def plan():
    c = synth.config5(div=8)                                  # the plan does not depend on div; the phantom is unused
    return c


def test_sampler_draws_equal_the_oracles(plan):
    for trial in range(25):
        a = binding.sample_delivery_trial(SPEC, trial, 3, plan["deliv"], **EXT)
        b = orc.sample_trial(SPEC, trial, 3, plan["deliv"], **EXT)
        assert (a["start_phase"] == b["start_phase"]).all()
        assert a["prm"].tobytes() == b["prm"].tobytes()
        for k in b["ext"]:
            if isinstance(b["ext"][k], np.ndarray):
                assert (a["ext"][k] == b["ext"][k]).all(), k
            else:
                assert a["ext"][k] == b["ext"][k], k
    with pytest.raises(RuntimeError):
        binding.sample_delivery_trial(SPEC, 25, 3, plan["deliv"], **EXT)


@pytest.mark.parametrize("mode", ["gated", "free_breathing_isolayered"])
def test_25_trials_on_the_config5_plan_byte_equal(plan, mode):
    prm = plan["deliv"].copy()
    ext = dict(EXT)
    if mode == "free_breathing_isolayered":                   # free breathing with a max MU per spot delivery
        prm["gate_mask"] = (1 << 10) - 1
        prm["repaints"] = 1
        ext["max_protons_per_paint"] = 2_500_000
    H = 10 ** 8
    ends = set()
    for trial in range(25):
        t = binding.sample_delivery_trial(SPEC, trial, 3, prm, **ext)
        f = plan["fields"].copy(); f["start_phase"] = t["start_phase"]
        got = binding.simulate_delivery_ext_host(f, plan["spots"], t["prm"], H, **t["ext"])
        o = orc.sample_trial(SPEC, trial, 3, prm, **ext)
        fo = plan["fields"].copy(); fo["start_phase"] = o["start_phase"]
        segs, tt, dropped, fills = orc.simulate_delivery_ext(fo, plan["spots"], o["prm"], H, **o["ext"])
        assert got["segments"].tobytes() == np.ascontiguousarray(segs).tobytes(), f"trial {trial}"
        assert (got["field_time_ns"] == tt).all() and got["dropped_protons"] == dropped and got["fills"] == fills
        assert int(segs["n_hist"].sum()) == H
        N_s = np.rint(plan["spots"]["weight"].astype(np.float64) * 10 ** 7).astype(np.int64)
        per_spot = np.zeros(len(N_s), np.int64); np.add.at(per_spot, segs["spot"], segs["protons"])
        assert (per_spot == N_s).all()                        # every proton delivered, every trial
        ends.add(int(tt.max()))
    assert len(ends) == 25                                    # 25 different deliveries
