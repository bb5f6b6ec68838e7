"""The uncertainty-trial loop pbs4d_run_trials (25 trials of the 4D dose with sampled start phase,
breathing period and synchrotron parameters) on the GPU: every trial equals the step-by-step calls bit for bit, its
sub-plans equal the oracle's, the context is re-used, and the trials differ from each other."""
import numpy as np
import pytest
import torch

import oracle as orc
from paper_1809_03927_b200 import binding, build, synth

pytestmark = pytest.mark.gpu

MS = 10 ** 6
SPEC = dict(seed=77, n_trials=25, n_cycles=30, period_lo_ns=3000 * MS, period_hi_ns=7000 * MS, period_step_ns=1000 * MS,
            period_sigma_ns=300 * MS, discard_sigma_ns=5 * MS, flat_top_sigma_ns=200 * MS, spot_switch_sigma_ns=200_000,
            layer_switch_sigma_ns=100 * MS, spill_protons_sigma=10 ** 9, protons_per_s_sigma=5 * 10 ** 7)
EXT = dict(discard_ns=70 * MS, spill_protons_max=12_500_000_000, flat_top_ns=16_000 * MS, spot_switch_fixed_ns=2 * MS)


def test_run_trials_equals_stepwise_and_oracle_delivery():
    build.build()
    cfg = synth.config5(div=8, n_hist=60_000)
    P = cfg["hu"].shape[0]
    ctx = binding.Context(0)
    hu = torch.from_numpy(cfg["hu"]).cuda()
    ctx.set_ct_phases(cfg["ct_grid"], [hu[p] for p in range(P)], cfg["dose_grid"])
    for p in range(P):
        if cfg["dvf"][p] is not None:
            ctx.set_dvf(p, cfg["ref_phase"], cfg["dvf_grid"], torch.from_numpy(cfg["dvf"][p]).cuda())
    ctx.set_plan_spots(cfg["fields"], cfg["spots"])
    planned = ctx.simulate_delivery(cfg["deliv"], cfg["histories"])
    outs, res = ctx.run_trials(SPEC, 0, 25, cfg["deliv"], cfg["histories"], 1000, cfg["ref_phase"], cfg["subvox"], **EXT)
    assert len(outs) == 25 and all(r["histories"] == cfg["histories"] for r in res)
    assert all(1 <= r["phases_run"] <= 5 and r["fills"] >= 75 and r["delivery_ns"] > 0 for r in res)
    sums = [float(o.double().sum()) for o in outs]
    assert len(set(sums)) == 25 and min(sums) > 0                       # 25 different 4D doses
    assert len(set(r["delivery_ns"] for r in res)) == 25
    # the trials start the fields in sampled phases; the plan itself must come out of the loop untouched
    again = ctx.simulate_delivery(cfg["deliv"], cfg["histories"])
    assert again["segments"].tobytes() == planned["segments"].tobytes()
    assert (again["field_time_ns"] == planned["field_time_ns"]).all()
    for trial in (0, 7, 24):
        d = ctx.simulate_delivery_trial(SPEC, trial, cfg["deliv"], cfg["histories"], **EXT)
        o = orc.sample_trial(SPEC, trial, 3, cfg["deliv"], **EXT)
        f = cfg["fields"].copy(); f["start_phase"] = o["start_phase"]
        if trial == 7:
            assert (o["start_phase"] != cfg["fields"]["start_phase"]).any()   # a trial that does move the start
            assert ctx.simulate_delivery(cfg["deliv"], cfg["histories"])["segments"].tobytes() == planned["segments"].tobytes()
            d = ctx.simulate_delivery_trial(SPEC, trial, cfg["deliv"], cfg["histories"], **EXT)
        segs, tt, _, fills = orc.simulate_delivery_ext(f, cfg["spots"], o["prm"], cfg["histories"], **o["ext"])
        assert d["segments"].tobytes() == np.ascontiguousarray(segs).tobytes() and d["fills"] == fills
        assert res[trial]["delivery_ns"] == int(tt.max())
        phases = sorted(set(int(x) for x in d["segments"]["phase"]) | {cfg["ref_phase"]})
        ctx.mc_dose_phases(phases, 1000 + trial)
        want, _ = ctx.accumulate_subvoxel(cfg["ref_phase"], cfg["subvox"])
        # run_trials marks the doses of earlier trials stale; the stepwise path here only ran `phases`, like the loop
        assert torch.equal(want.view(torch.int32), outs[trial].view(torch.int32)), f"trial {trial}"
    # a slice of the trial range gives the same doses as the full loop
    outs2, _ = ctx.run_trials(SPEC, 7, 2, cfg["deliv"], cfg["histories"], 1000, cfg["ref_phase"], cfg["subvox"], **EXT)
    assert torch.equal(outs2[0], outs[7]) and torch.equal(outs2[1], outs[8])
    ctx.close()
