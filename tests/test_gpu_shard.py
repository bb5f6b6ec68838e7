"""History sharding over GPUs, exercised on ONE device: the shards of a
world of 2 and of 3 ranks are run one after the other through the same calls a multi-process run makes, their int64
grids are summed, and the result must be BIT-IDENTICAL to the unsharded run -- energy grids, phase doses and the
accumulated 4D dose.  (The sum over ranks is an integer all-reduce in a real run; bench.py --gpus N issues it through
torch.distributed / NCCL.)"""
import numpy as np
import pytest
import torch

from paper_1809_03927_b200 import binding, build, synth

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx():
    build.build()
    c = binding.Context(0)
    yield c
    c.close()


def setup(ctx, cfg):
    P = cfg["hu"].shape[0]
    hu = torch.from_numpy(cfg["hu"]).cuda()
    ctx.set_ct_phases(cfg["ct_grid"], [hu[p] for p in range(P)], cfg["dose_grid"])
    for p in range(P):
        if cfg["dvf"][p] is not None:
            ctx.set_dvf(p, cfg["ref_phase"], cfg["dvf_grid"], torch.from_numpy(cfg["dvf"][p]).cuda())
    ctx.set_plan_spots(cfg["fields"], cfg["spots"])
    deliv = ctx.simulate_delivery(cfg["deliv"], cfg["histories"])
    return sorted(set(int(x) for x in deliv["segments"]["phase"]) | {cfg["ref_phase"]}), deliv


@pytest.mark.parametrize("world", [2, 3])
def test_sharded_run_is_bit_identical(ctx, world):
    cfg = synth.config3(div=4, n_hist=90_001)                  # odd count: uneven slices
    phases, deliv = setup(ctx, cfg)
    ctx.set_shard(0, 1)
    sts0, _ = ctx.mc_dose_phases(phases, cfg["seed"])
    Q0 = {p: ctx.get_phase_energy(p).clone() for p in phases}
    D0 = {p: ctx.mc_dose_phase(p, cfg["seed"])[0].clone() for p in phases}
    out0, ast0 = ctx.accumulate_subvoxel(cfg["ref_phase"], cfg["subvox"])
    E0 = {p: ctx.get_accumulators(p) for p in phases if p != cfg["ref_phase"]}

    # ---- transport: every rank its slice of every phase; integer sum of the grids ----
    Qsum = {p: torch.zeros_like(Q0[p]) for p in phases}
    tot = {k: 0 for k in ("histories", "steps", "q_incident", "q_deposited", "q_escaped", "scoring_atomics")}
    for r in range(world):
        ctx.set_shard(r, world)
        sts, _ = ctx.mc_dose_phases(phases, cfg["seed"])
        for p, st in zip(phases, sts):
            n_p = int(deliv["segments"]["n_hist"][deliv["segments"]["phase"] == p].sum())
            assert st["histories"] == binding.shard_window(n_p, r, world)[1]
            Qsum[p] += ctx.phase_energy_view(p)
            for k in tot:
                tot[k] += st[k]
    for k in tot:
        assert tot[k] == sum(st[k] for st in sts0), k
    for p in phases:
        assert torch.equal(Qsum[p], Q0[p]), f"phase {p}: summed shard grids differ from the unsharded grid"
        ctx.phase_energy_view(p).copy_(Qsum[p])                # what the all-reduce leaves in every rank's context
        ctx.finalize_phase_dose(p)
    ctx.set_shard(0, 1)

    # ---- accumulation sharded by source phase: rank r pushes every world-th source phase ----
    src = [p for p in phases if p != cfg["ref_phase"]]
    got = {}
    sub = 0
    for r in range(world):
        mask = sum(1 << p for i, p in enumerate(src) if i % world == r)
        st = ctx.accumulate_push(cfg["ref_phase"], cfg["subvox"], mask)
        sub += st["subvoxels"]
        for i, p in enumerate(src):
            E, M = ctx.accumulator_views(p)
            if i % world == r:
                got[p] = (E.clone(), M.clone())
            else:
                assert int(E.abs().sum()) == 0 and int(M.abs().sum()) == 0      # not pushed by this rank: zeros
    assert sub == ast0["subvoxels"]
    for p in src:                                              # the exchange: every rank ends up with every sum
        E, M = ctx.accumulator_views(p)
        E.copy_(got[p][0]); M.copy_(got[p][1])
        assert torch.equal(E, E0[p][0]) and torch.equal(M, E0[p][1])
    out, _ = ctx.accumulate_finalize(cfg["ref_phase"])
    assert torch.equal(out.view(torch.int32), out0.view(torch.int32))
    for p in phases:                                           # phase doses re-derived from the summed grids
        d, _, _ = ctx.mc_dose_phase(p, cfg["seed"])
        assert torch.equal(d.view(torch.int32), D0[p].view(torch.int32))


def test_more_ranks_than_histories_and_bad_arguments(ctx):
    cfg = synth.config1(n_hist=5, n=12)
    hu = torch.from_numpy(cfg["hu"]).cuda()
    ctx.set_ct_phases(cfg["ct_grid"], [hu[0]], None)
    ctx.set_plan_spots(cfg["fields"], cfg["spots"])
    ctx.simulate_delivery(cfg["deliv"], cfg["histories"])
    ctx.set_shard(0, 1)
    _, _, st = ctx.mc_dose_phase(0, 7, want_dose=False)
    Q0 = ctx.get_phase_energy(0).clone()
    Qs = torch.zeros_like(Q0)
    n = 0
    for r in range(8):                                         # 8 ranks, 5 histories: three empty shards
        ctx.set_shard(r, 8)
        _, _, s = ctx.mc_dose_phase(0, 7, want_dose=False)
        n += s["histories"]
        Qs += ctx.phase_energy_view(0)
    assert n == 5 and torch.equal(Qs, Q0)
    with pytest.raises(RuntimeError):
        ctx.set_shard(3, 3)
    with pytest.raises(RuntimeError):
        ctx.set_shard(-1, 2)
    # the whole-path entry points contain no exchange step: with sharding on they would hand back a dose built from a
    # slice of the histories, so they refuse (PBS4D_ERR_ORDER) until the shard is reset
    ctx.set_shard(1, 2)
    out = np.zeros(synth.grid_shape(cfg["ct_grid"]), np.float32)
    with pytest.raises(RuntimeError, match="-2.*sharding"):
        ctx.run_plan_host(cfg["ct_grid"], [cfg["hu"][0]], None, None, None, 0, cfg["fields"], cfg["spots"], cfg["deliv"],
                          cfg["histories"], 7, (1, 1, 1), out)
    spec = dict(seed=1, n_trials=2, n_cycles=0)
    with pytest.raises(RuntimeError, match="-2.*sharding"):
        ctx.run_trials(spec, 0, 1, cfg["deliv"], cfg["histories"], 7, 0, (1, 1, 1))
    ctx.set_shard(0, 1)
    _, _, s = ctx.mc_dose_phase(0, 7, want_dose=False)         # the refused calls left the context as it was
    assert s["histories"] == 5 and torch.equal(ctx.get_phase_energy(0), Q0)


def test_density_validation_rejects_zero_and_nonfinite(ctx):
    g = synth.make_grid((4, 4, 4), (2.0, 2.0, 2.0))
    good = torch.ones((4, 4, 4), dtype=torch.float32, device="cuda")
    ctx.set_density_phases(g, [good])
    for bad_value in (0.0, float("inf"), float("nan"), -1.0):
        bad = good.clone(); bad[1, 2, 3] = bad_value
        with pytest.raises(RuntimeError, match="densities must be finite"):
            ctx.set_density_phases(g, [good, bad])


def test_bench_pass_sharded_equals_single(ctx):
    """bench.py's N > 1 pass (run_pass), driven for world = 2 on one device: the two ranks run one after the other and
    the collectives are replaced by stand-ins that move the same integers (sum of the energy grids, owner's sums to
    everyone).  The 4D dose of the sharded pass must equal the single-GPU pass bit for bit."""
    import bench
    cfg = synth.config5(div=8, n_hist=80_000)
    P = cfg["hu"].shape[0]
    hu_dev = torch.from_numpy(cfg["hu"]).cuda()
    dvf_dev = [None if d is None else torch.from_numpy(d).cuda() for d in cfg["dvf"]]
    n1, out1, st1 = bench.run_pass(ctx, cfg, hu_dev, dvf_dev, 0, 1)
    out1 = out1.clone()
    world = 2
    # pass A: every rank transports its slice; keep its grids
    grids = {}

    def record(r):
        def sum_grids(views, w):
            grids[r] = [v.clone() for v in views]
        return sum_grids

    pushed = {}

    def record_push(r):
        def share(pairs, owners, w):
            for p, (E, M) in pairs.items():
                if owners[p] == r:
                    pushed[p] = (E.clone(), M.clone())
        return share

    hist = 0
    for r in range(world):
        n, _, st = bench.run_pass(ctx, cfg, hu_dev, dvf_dev, r, world, sum_grids=record(r), share=lambda *a: None)
        hist += n
    assert hist == n1 == cfg["histories"]
    total = [sum(grids[r][i] for r in range(world)) for i in range(len(grids[0]))]

    # pass B: the same passes with the exchanges delivering what the collectives would
    def all_reduce_stub(views, w):
        for v, t in zip(views, total):
            v.copy_(t)

    for r in range(world):                                     # first collect every owner's sums (from summed grids)
        bench.run_pass(ctx, cfg, hu_dev, dvf_dev, r, world, sum_grids=all_reduce_stub, share=record_push(r))

    def broadcast_stub(pairs, owners, w):
        for p, (E, M) in pairs.items():
            E.copy_(pushed[p][0]); M.copy_(pushed[p][1])

    for r in range(world):
        n, out, st = bench.run_pass(ctx, cfg, hu_dev, dvf_dev, r, world, sum_grids=all_reduce_stub, share=broadcast_stub)
        assert torch.equal(out.view(torch.int32), out1.view(torch.int32)), f"rank {r}"
        assert st["launches"] > 0 and st["phases"] == st1["phases"]


def test_call_order_and_argument_errors_of_the_split_calls(ctx):
    cfg = synth.config3(div=4, n_hist=20_000)
    phases, deliv = setup(ctx, cfg)
    ref = cfg["ref_phase"]
    with pytest.raises(RuntimeError, match="mc_dose_phase not run"):
        ctx.phase_energy_view(phases[0])                       # no transport yet for this delivery
    with pytest.raises(RuntimeError, match="mc_dose_phase not run"):
        ctx.finalize_phase_dose(phases[0])
    ctx.mc_dose_phases(phases, cfg["seed"])
    with pytest.raises(RuntimeError, match="not pushed|no accumulators"):
        ctx.accumulate_finalize(ref)                           # a9 before any a8
    with pytest.raises(RuntimeError):
        ctx.accumulator_views(ref)                             # the reference phase has no accumulators
    st = ctx.accumulate_push(ref, cfg["subvox"], 0)            # empty mask: nothing pushed, everything zeroed
    assert st["subvoxels"] == 0
    out, _ = ctx.accumulate_finalize(ref)                      # = the reference dose inside the DVF coverage
    d_ref = ctx.mc_dose_phase(ref, cfg["seed"])[0]
    inside = out != 0
    assert int(inside.sum()) > 0 and torch.equal(out[inside], d_ref[inside])
    with pytest.raises(RuntimeError):
        ctx.accumulate_push(ref, (0, 2, 2), 1)
    with pytest.raises(RuntimeError):
        ctx.phase_energy_view(99)
