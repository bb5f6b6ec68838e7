"""The end-to-end entry pbs4d_run_plan_host (host buffers in, 4D dose out; the call bench.py's e2e leg times) must give
exactly the result of the step-by-step device path: transport scores integers and the accumulation is bit-exact, so
the two 4D doses are compared bit for bit."""
import numpy as np
import pytest
import torch

from paper_1809_03927_b200 import binding, build, synth

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("name,kw", [("config3", dict(div=4, n_hist=150_000)), ("config5", dict(div=8, n_hist=150_000))])
def test_run_plan_host_equals_stepwise_path(name, kw):
    build.build()
    cfg = getattr(synth, name)(**kw)
    P = cfg["hu"].shape[0]
    ctx = binding.Context(0)
    hu = torch.from_numpy(cfg["hu"]).cuda()
    ctx.set_ct_phases(cfg["ct_grid"], [hu[p] for p in range(P)], cfg["dose_grid"])
    for p in range(P):
        if cfg["dvf"][p] is not None:
            ctx.set_dvf(p, cfg["ref_phase"], cfg["dvf_grid"], torch.from_numpy(cfg["dvf"][p]).cuda())
    ctx.set_plan_spots(cfg["fields"], cfg["spots"])
    deliv = ctx.simulate_delivery(cfg["deliv"], cfg["histories"])
    phases = sorted(set(int(x) for x in deliv["segments"]["phase"]) | {cfg["ref_phase"]})
    n = 0
    for p in phases:
        _, _, st = ctx.mc_dose_phase(p, cfg["seed"], want_dose=False)
        n += st["histories"]
    want, _ = ctx.accumulate_subvoxel(cfg["ref_phase"], cfg["subvox"])
    want = want.cpu().numpy()
    ctx.close()

    ctx2 = binding.Context(0)
    g = cfg["ct_grid"] if cfg["dose_grid"] is None else cfg["dose_grid"]
    out = np.full((int(g["nz"][0]), int(g["ny"][0]), int(g["nx"][0])), -1.0, np.float32)
    for rep in range(2):                                     # second call reuses the staging buffers
        run, secs, h2d = ctx2.run_plan_host(cfg["ct_grid"], [cfg["hu"][p] for p in range(P)], cfg["dose_grid"], cfg["dvf_grid"],
                                       cfg["dvf"], cfg["ref_phase"], cfg["fields"], cfg["spots"], cfg["deliv"],
                                       cfg["histories"], cfg["seed"], cfg["subvox"], out)
        assert run == n == cfg["histories"] and len(secs) == 4 and all(s >= 0 for s in secs)
        assert out.view(np.uint32).tobytes() == want.view(np.uint32).tobytes()
        assert want.max() > 0
        # only the phases that receive beam (plus the reference phase) are uploaded, CT and DVF
        expect = sum(cfg["hu"][p].nbytes for p in phases) + cfg["spots"].nbytes + cfg["fields"].nbytes + \
            sum(cfg["dvf"][p].nbytes for p in phases if p != cfg["ref_phase"] and cfg["dvf"][p] is not None)
        assert h2d == expect
    ctx2.close()
