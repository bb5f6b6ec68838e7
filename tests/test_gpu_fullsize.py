"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (same calls, same grids, same
history counts), plus reduced-H reruns of the full-size phantoms that the oracle can follow history by history.

What the oracle cannot recompute at 1e7-1e8 histories is checked through properties that hold at any size:
  * delivery lists of the full plan: bit-equal to the oracle's (int64 event simulation, unique result);
  * per launch: histories run == histories allocated; the int64 dose grid sums to the deposited tally exactly;
    deposited + escaped == incident up to the fp32 rounding of the running energy (north_star: 0.1 %);
  * deposited fraction of the incident energy equals the oracle's on a bounded sample of the same plan within 0.1 %;
  * accumulation at full size: BIT-EXACT against the oracle (the oracle pushes all 3.4e9 subvoxels in ~10-20 s).
"""
import numpy as np
import pytest
import torch

import oracle as orc
from paper_1809_03927_b200 import binding, build, synth
from test_gpu_transport import check_parity, gpu_run, oracle_run

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx():
    build.build()
    c = binding.Context(0)
    yield c
    c.close()


def run_like_bench(ctx, cfg):
    """the device-resident pass of bench.py's step_device(), keeping what the checks need"""
    P = cfg["hu"].shape[0]
    hu = torch.from_numpy(cfg["hu"]).cuda()
    ctx.set_ct_phases(cfg["ct_grid"], [hu[p] for p in range(P)], cfg["dose_grid"])
    for p in range(P):
        if cfg["dvf"][p] is not None:
            ctx.set_dvf(p, cfg["ref_phase"], cfg["dvf_grid"], torch.from_numpy(cfg["dvf"][p]).cuda())
    ctx.set_plan_spots(cfg["fields"], cfg["spots"])
    deliv = ctx.simulate_delivery(cfg["deliv"], cfg["histories"])
    segs = deliv["segments"]
    phases = sorted(set(int(x) for x in segs["phase"]) | {cfg["ref_phase"]})
    res = {}
    for p in phases:
        dose, _, st = ctx.mc_dose_phase(p, cfg["seed"])
        res[p] = (dose, st)
    out, ast = ctx.accumulate_subvoxel(cfg["ref_phase"], cfg["subvox"])
    return deliv, res, out, ast


def check_launch_invariants(ctx, deliv, res):
    segs = deliv["segments"]
    tot = dict(inc=0, dep=0, esc=0)
    for p, (dose, st) in res.items():
        alloc = int(segs["n_hist"][segs["phase"] == p].sum())
        assert st["histories"] == alloc, f"phase {p}: ran {st['histories']} of {alloc} histories"
        Q = ctx.get_phase_energy(p)
        assert int(Q.sum().item()) == st["q_deposited"], f"phase {p}: grid sum != deposited tally"
        assert int((Q < 0).sum().item()) == 0
        bal = st["q_incident"] - st["q_deposited"] - st["q_escaped"]
        assert abs(bal) <= 2e-5 * max(st["q_incident"], 1), f"phase {p}: energy balance {bal}"
        assert torch.isfinite(dose).all()
        tot["inc"] += st["q_incident"]; tot["dep"] += st["q_deposited"]; tot["esc"] += st["q_escaped"]
        del Q
    return tot


def oracle_fraction(cfg, budget):
    """deposited / incident of the oracle on `budget` histories of the same plan (own delivery + allocation)"""
    segs, _, _ = orc.simulate_delivery(cfg["fields"], cfg["spots"], cfg["deliv"], budget)
    k = orc.fixed_shift(segs, cfg["spots"])
    g = cfg["ct_grid"] if cfg["dose_grid"] is None else cfg["dose_grid"]
    inc = dep = 0
    rhos = {}
    for p in sorted(set(int(x) for x in segs["phase"])):
        rhos[p] = orc.hu_to_density(cfg["ct_grid"], cfg["hu"][p], cfg["dose_grid"])
        _, st, _, _ = orc.transport(g, rhos[p], cfg["fields"], cfg["spots"], segs[segs["phase"] == p], cfg["seed"], k)
        inc += int(st["q_incident"]); dep += int(st["q_deposited"])
    return dep / inc, rhos


def test_config5_full_size_bench_configuration(ctx):
    cfg = synth.config5()                                            # 512x512x160 x 10 phases, 1e8 histories
    deliv, res, out, ast = run_like_bench(ctx, cfg)
    # delivery: bit-equal to the oracle on the full plan
    segs_o, tt_o, dropped_o = orc.simulate_delivery(cfg["fields"], cfg["spots"], cfg["deliv"], cfg["histories"])
    assert deliv["segments"].tobytes() == np.ascontiguousarray(segs_o).tobytes()
    assert (deliv["field_time_ns"] == tt_o).all() and deliv["dropped_protons"] == int(dropped_o)
    assert set(int(x) for x in segs_o["phase"]) <= set(cfg["gate_phases"])              # gated: phases 3..7 only
    tot = check_launch_invariants(ctx, deliv, res)
    assert sum(st["histories"] for _, st in res.values()) == cfg["histories"]
    # deposited fraction vs the oracle on a bounded sample of the same plan (north_star: total energy within 0.1 %)
    f_orc, rhos = oracle_fraction(cfg, 100_000)
    assert abs(tot["dep"] / tot["inc"] - f_orc) <= 1e-3, (tot["dep"] / tot["inc"], f_orc)
    # accumulation of the MC doses at (2,2,5): bit-exact against the oracle at full size
    P = cfg["hu"].shape[0]
    g = cfg["ct_grid"]
    doses = [None] * P; rho_l = [None] * P
    for p in range(P):
        if p in res:
            doses[p] = res[p][0].cpu().numpy()
            rho_l[p] = rhos[p] if p in rhos else orc.hu_to_density(cfg["ct_grid"], cfg["hu"][p], None)
    dvf = [cfg["dvf"][p] if p in res else None for p in range(P)]
    want, st_o = orc.accumulate_subvoxel(g, doses, rho_l, dvf, [cfg["dvf_grid"]] * P, cfg["ref_phase"], cfg["subvox"])
    got = out.cpu().numpy()
    assert got.view(np.uint32).tobytes() == want.view(np.uint32).tobytes()
    for k in ("subvoxels", "dropped_outside_ref", "dropped_outside_dvf"):
        assert ast[k] == int(st_o[k]), k


def test_config3_full_size_bench_configuration_and_reduced_h_parity(ctx):
    cfg = synth.config3()                                            # 10 phases, dose grid 128x128x160, 1e7 histories
    deliv, res, out, ast = run_like_bench(ctx, cfg)
    segs_o, tt_o, _ = orc.simulate_delivery(cfg["fields"], cfg["spots"], cfg["deliv"], cfg["histories"])
    assert deliv["segments"].tobytes() == np.ascontiguousarray(segs_o).tobytes()
    tot = check_launch_invariants(ctx, deliv, res)
    assert sum(st["histories"] for _, st in res.values()) == cfg["histories"]
    # accumulation at full size, bit-exact
    P = cfg["hu"].shape[0]
    g = cfg["dose_grid"]
    rhos = [orc.hu_to_density(cfg["ct_grid"], cfg["hu"][p], g) for p in range(P)]
    doses = [res[p][0].cpu().numpy() for p in range(P)]
    want, st_o = orc.accumulate_subvoxel(g, doses, rhos, cfg["dvf"], [cfg["dvf_grid"]] * P, cfg["ref_phase"],
                                         cfg["subvox"])
    assert out.cpu().numpy().view(np.uint32).tobytes() == want.view(np.uint32).tobytes()
    assert ast["subvoxels"] == int(st_o["subvoxels"])
    # same full-size phantom and plan at H = 4e5: the oracle follows every history; per-voxel parity on two phases
    small = dict(cfg, histories=400_000)
    gq, dg = gpu_run(ctx, small, phases=[0, 5])
    oq, do = oracle_run(small, phases=[0, 5])
    assert dg["segments"].tobytes() == np.ascontiguousarray(do["segments"]).tobytes()
    f_g = f_o = 0.0
    for p in (0, 5):
        # 4e5 histories over ~3000 spots and 10 phases leave only tens of histories per voxel, so one decorrelated
        # history moves a voxel by several % of Dmax; the 2 %-of-Dmax bound is therefore applied to the deposited
        # energy binned in 4x4x4-voxel (8 mm) blocks, where every block above 10 % of the maximum holds >1e3 deposits
        (dose_g, Qg, stg, rho_g), (dose_o, Qo, sto, rho_o) = gq[p], oq[p]
        assert (rho_g == rho_o).all() and stg["histories"] == int(sto["histories"])
        assert int(Qg.sum()) == stg["q_deposited"]
        assert abs(stg["q_deposited"] - int(sto["q_deposited"])) <= 1e-3 * int(sto["q_deposited"])
        assert abs(stg["q_incident"] - int(sto["q_incident"])) <= 1e-6 * int(sto["q_incident"])
        nz, ny, nx = Qo.shape
        blk = lambda Q: Q.astype(np.float64).reshape(nz // 4, 4, ny // 4, 4, nx // 4, 4).sum((1, 3, 5))
        Bg, Bo = blk(Qg), blk(Qo)
        sel = Bo > 0.1 * Bo.max()
        err = np.abs(Bg - Bo)[sel].max() / Bo.max()
        assert sel.sum() > 20 and err <= 0.02, f"config3 full grid, H=4e5, phase {p}: block error {err:.4f} of max"
        f_g += stg["q_deposited"]; f_o += int(sto["q_deposited"])
    assert abs(f_g / f_o - 1.0) <= 1e-3
    assert 0.5 < tot["dep"] / tot["inc"] <= 1.0


# ---------------------------------------------------------------------------------------------------------------
# Per-voxel transport parity on the FULL config-5 and config-3 grids (north_star's criteria, unrelaxed).
# The plan is restricted (a few central spots of two layers per field) so that 1e6 histories give every voxel above
# 10 % Dmax thousands of deposits; grid, voxel size, phantom, field geometry, energies and spot sizes are the
# configs' own.  Each field is delivered in a phase of its own (breathing period long enough that a field fits in
# one phase, start_phase = that phase), so the per-phase grids are per-field doses and R80 can be taken along each
# oblique beam axis.
# ---------------------------------------------------------------------------------------------------------------
def restrict_plan(cfg, layers, n_central, field_phases, histories):
    sp = cfg["spots"]
    r2 = sp["x_mm"].astype(np.float64) ** 2 + sp["y_mm"].astype(np.float64) ** 2
    keep = []
    for f in range(len(cfg["fields"])):
        for l in layers:
            idx = np.nonzero((sp["field"] == f) & (sp["layer"] == l))[0]
            keep.extend(sorted(idx[np.argsort(r2[idx], kind="stable")[:n_central]]))
    out = dict(cfg)
    out["spots"] = sp[np.array(keep)].copy()
    out["spots"]["weight"] = 1.0
    out["fields"] = cfg["fields"].copy()
    out["fields"]["start_phase"] = field_phases
    out["deliv"] = synth.make_delivery(n_phases=cfg["hu"].shape[0], period_s=1000.0, protons_per_weight=10 ** 7,
                                       layer_switch_s=1.0)
    out["histories"] = histories
    return out


def depth_r80(Q, grid, field, bin_mm=2.0):
    """distal 80 % point of the deposited energy binned by depth along the field direction (voxel centres)"""
    nz, ny, nx = Q.shape
    x, y, z = synth.centres(grid)
    d = field["dir"].astype(np.float64)
    vz, vy, vx = np.nonzero(Q)
    depth = x[vx] * d[0] + y[vy] * d[1] + z[vz] * d[2]
    lo = depth.min()
    dd = np.bincount(((depth - lo) / bin_mm).astype(np.int64), weights=Q[vz, vy, vx].astype(np.float64))
    k = int(np.nonzero(dd >= 0.8 * dd.max())[0].max())              # last bin above 80 % of the maximum
    return lo + (k + 0.5) * bin_mm + (dd[k] - 0.8 * dd.max()) / (dd[k] - dd[k + 1]) * bin_mm


def full_grid_parity(ctx, cfg, label):
    phases = sorted(int(p) for p in cfg["fields"]["start_phase"])
    g, dg = gpu_run(ctx, cfg, phases=phases)
    o, do = oracle_run(cfg, phases=phases)
    assert dg["segments"].tobytes() == np.ascontiguousarray(do["segments"]).tobytes()
    grid = cfg["ct_grid"] if cfg["dose_grid"] is None else cfg["dose_grid"]
    worst = 0.0
    for f, p in enumerate(cfg["fields"]["start_phase"]):
        p = int(p)
        assert set(int(x) for x in do["segments"]["field"][do["segments"]["phase"] == p]) == {f}
        err = check_parity(g[p], o[p], f"{label} field {f} (phase {p})")       # 2 % Dmax above 10 % Dmax, energy 0.1 %
        worst = max(worst, err)
        rg, ro = depth_r80(g[p][1], grid, cfg["fields"][f]), depth_r80(o[p][1], grid, cfg["fields"][f])
        assert abs(rg - ro) <= 0.3, f"{label} field {f}: R80 along the beam axis {rg:.3f} vs {ro:.3f} mm"
        n_sel = int((o[p][0] > 0.1 * o[p][0].max()).sum())
        assert n_sel > 2000, f"{label} field {f}: only {n_sel} voxels above 10 % Dmax"
        print(f"{label} field {f}: max voxel err {err:.4f} of Dmax over {n_sel} voxels, R80 {rg:.2f} / {ro:.2f} mm")
    return worst


def test_config5_full_grid_per_voxel_parity(ctx):
    cfg = synth.config5()                                            # 512x512x160 at 0.98x0.98x2.5 mm, ribs, 3 fields
    small = restrict_plan(cfg, layers=(9, 17), n_central=5, field_phases=(3, 5, 6), histories=1_200_000)
    assert len(small["spots"]) == 30
    full_grid_parity(ctx, small, "config5 full grid")


def test_config3_full_grid_per_voxel_parity(ctx):
    cfg = synth.config3()                                            # CT 256x256x128 resampled to 128x128x160 at 2 mm
    small = restrict_plan(cfg, layers=(4, 12), n_central=5, field_phases=(2,), histories=600_000)
    assert len(small["spots"]) == 10
    full_grid_parity(ctx, small, "config3 full grid")
