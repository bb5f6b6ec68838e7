"""GPU parity: EMTM subvoxel accumulation and density kernels vs the oracle -- BIT-EXACT (BASELINE.json north_star:
"accumulation and delivery binning must be bit-exact, which the fixed-point atomics make possible")."""
import numpy as np
import pytest
import torch

import oracle as orc
from paper_1809_03927_b200 import binding, build, synth

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx():
    build.build()
    c = binding.Context(0)
    yield c
    c.close()


def gpu_accumulate(ctx, c, ns, phases=None, dvf_grids=None):
    P = len(c["doses"])
    rho = torch.from_numpy(c["rhos"]).cuda()
    dose = torch.from_numpy(c["doses"]).cuda()
    ctx.set_density_phases(c["grid"], [rho[p] for p in range(P)])
    keep = []
    for p in range(P):
        if c["disps"][p] is None or (phases is not None and p not in phases):
            continue
        d = torch.from_numpy(c["disps"][p]).cuda()
        ctx.set_dvf(p, c["ref_phase"], c["dvf_grid"] if dvf_grids is None else dvf_grids[p], d)
        keep.append(p)
    out, st = ctx.accumulate_subvoxel(c["ref_phase"], ns, [dose[p] for p in range(P)])
    EM = {p: tuple(t.cpu().numpy() for t in ctx.get_accumulators(p)) for p in keep}
    return out.cpu().numpy(), st, EM


def oracle_accumulate(c, ns, phases=None, dvf_grids=None):
    P = len(c["doses"])
    disps = [c["disps"][p] if (phases is None or p in phases) else None for p in range(P)]
    grids = [c["dvf_grid"] if dvf_grids is None else dvf_grids[p] for p in range(P)]
    EM = {}
    for p in range(P):
        if disps[p] is not None:
            E, M, _ = orc.emtm_push(c["grid"], c["doses"][p], c["rhos"][p], grids[p], disps[p], c["grid"], ns)
            EM[p] = (E, M)
    out, st = orc.accumulate_subvoxel(c["grid"], c["doses"], c["rhos"], disps, grids, c["ref_phase"], ns)
    return out, st, EM


def assert_bit_exact(g, o):
    out_g, st_g, EM_g = g
    out_o, st_o, EM_o = o
    assert set(EM_g) == set(EM_o)
    for p in EM_o:
        assert (EM_g[p][0] == EM_o[p][0]).all(), f"E differs, phase {p}"
        assert (EM_g[p][1] == EM_o[p][1]).all(), f"M differs, phase {p}"
    assert out_g.view(np.uint32).tobytes() == out_o.view(np.uint32).tobytes()
    for k in ("subvoxels", "dropped_outside_ref", "dropped_outside_dvf"):
        assert st_g[k] == int(st_o[k]), k


@pytest.mark.parametrize("ns", [(1, 1, 1), (2, 2, 2), (3, 3, 3), (4, 4, 4), (2, 2, 5)])
def test_config4_small_bit_exact(ctx, ns):
    # 44^3: several 32x8 tiles with ragged tails in x and y
    c = synth.config4(n=44, n_phases=4)
    assert_bit_exact(gpu_accumulate(ctx, c, ns), oracle_accumulate(c, ns))


@pytest.mark.parametrize("ns", [(2, 2, 2), (3, 4, 4)])
def test_coarse_and_partial_dvf_grid(ctx, ns):
    # DVF on a coarser grid (paper Table I: deformation grids ~2x coarser than the CT) that does not cover the dose
    # grid: exercises clamp-to-edge, the outside-DVF drop and the coverage mask; nsz = 4 also the shared-memory node
    # box with z-subvoxels outside the DVF extent
    c = synth.config4(n=40, n_phases=3, dvf_div=2)
    dg = c["dvf_grid"].copy()
    dg["ox"], dg["oy"], dg["oz"] = 6.0, 3.0, 9.0
    grids = [dg, dg, dg]
    g = gpu_accumulate(ctx, c, ns, dvf_grids=grids)
    o = oracle_accumulate(c, ns, dvf_grids=grids)
    assert_bit_exact(g, o)
    assert g[1]["dropped_outside_dvf"] > 0 and g[1]["dropped_outside_ref"] > 0
    assert (g[0] == 0).any() and (g[0] != 0).any()


def test_anisotropic_voxels(ctx):
    c = synth.config4(n=36, n_phases=3)
    for name in ("grid", "dvf_grid"):
        c[name] = c[name].copy()
        c[name]["hx"], c[name]["hy"], c[name]["hz"] = 0.98, 0.98, 2.5
        c[name]["ox"], c[name]["oy"], c[name]["oz"] = -17.3, 4.1, 100.0
    for p in range(1, 3):
        c["disps"][p] = (c["disps"][p] * 0.3).astype(np.float32)
    assert_bit_exact(gpu_accumulate(ctx, c, (2, 2, 5)), oracle_accumulate(c, (2, 2, 5)))


def test_huge_displacements_take_the_exact_path(ctx):
    # |u| of thousands of voxels: the index tolerance exceeds 1/4 and every subvoxel is decided by the contract's own
    # operations (the estimate is never trusted); nearly everything lands outside the reference grid
    c = synth.config4(n=24, n_phases=3)
    for p in range(1, 3):
        c["disps"][p] = (c["disps"][p] * np.float32(3.0e5)).astype(np.float32)
        c["disps"][p][:, ::3, ::2, ::2] *= np.float32(1.0e-5)            # some nodes stay small: a few subvoxels land
    g = gpu_accumulate(ctx, c, (2, 2, 2)); o = oracle_accumulate(c, (2, 2, 2))
    assert_bit_exact(g, o)
    assert g[1]["dropped_outside_ref"] > 0.5 * g[1]["subvoxels"]
    assert_bit_exact(gpu_accumulate(ctx, c, (3, 3, 4)), oracle_accumulate(c, (3, 3, 4)))


def test_non_finite_nodes_are_dropped_like_the_oracle_drops_them(ctx):
    # NaN / Inf displacements: the max |u| record is not finite, so the kernel takes the exact path everywhere and the
    # subvoxels that interpolate a bad node fall outside, exactly as floorf() of a NaN does in the oracle
    c = synth.config4(n=28, n_phases=3)
    c["disps"][1][0, 5:8, 9:12, 3:6] = np.nan
    c["disps"][1][2, 15, 15, 15] = np.inf
    c["disps"][2][1, 20:22, 4, 7] = -np.inf
    for ns in [(2, 2, 2), (4, 4, 4)]:
        g = gpu_accumulate(ctx, c, ns); o = oracle_accumulate(c, ns)
        assert_bit_exact(g, o)
        assert g[1]["dropped_outside_ref"] > 0


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_dvf_grid_one_node_wide(ctx, axis):
    # a DVF grid with a single node along one axis (upper node = lower node on that axis; the node box in shared
    # memory is not used when the grid is one node wide in x)
    c = synth.config4(n=32, n_phases=3)
    name = "xyz"[axis]
    dg = c["dvf_grid"].copy()
    n_ax = int(dg["n" + name][0]) if hasattr(dg["n" + name], "__len__") else int(dg["n" + name])
    dg["h" + name] = dg["h" + name] * n_ax
    dg["n" + name] = 1
    for p in range(1, 3):
        sl = [slice(None)] * 4
        sl[3 - axis] = slice(n_ax // 2, n_ax // 2 + 1)                  # disps: [3][z][y][x]
        c["disps"][p] = np.ascontiguousarray(c["disps"][p][tuple(sl)])
    grids = [dg, dg, dg]
    for ns in [(2, 2, 2), (3, 3, 4)]:
        assert_bit_exact(gpu_accumulate(ctx, c, ns, dvf_grids=grids), oracle_accumulate(c, ns, dvf_grids=grids))


def test_identity_dvf_is_the_plain_sum(ctx):
    # identity DVF must reproduce the 3D static sum
    c = synth.config4(n=33, n_phases=3)
    for p in range(1, 3):
        c["disps"][p] = np.zeros_like(c["disps"][p])
    out, st, _ = gpu_accumulate(ctx, c, (2, 2, 2))
    assert np.abs(out - c["doses"].astype(np.float64).sum(0)).max() < 1e-6 * 6
    assert st["dropped_outside_ref"] == 0 and st["dropped_outside_dvf"] == 0


def test_config4_full_size(ctx):
    # BASELINE.json config 4: 10 phases of 128^3 at 2 mm; n = 2 and 4 over all phases; n = 8 on one source phase
    c = synth.config4()
    for ns in [(2, 2, 2), (4, 4, 4)]:
        assert_bit_exact(gpu_accumulate(ctx, c, ns), oracle_accumulate(c, ns))
    assert_bit_exact(gpu_accumulate(ctx, c, (8, 8, 8), phases=[3]), oracle_accumulate(c, (8, 8, 8), phases=[3]))


def test_density_kernels_bit_exact(ctx):
    for cfg in (synth.config2(), synth.config3(div=4, n_hist=10), synth.config5(div=8, n_hist=10)):
        hu = torch.from_numpy(cfg["hu"]).cuda()
        ctx.set_ct_phases(cfg["ct_grid"], [hu[p] for p in range(hu.shape[0])], cfg["dose_grid"])
        ctx.set_plan_spots(cfg["fields"], cfg["spots"])
        ctx.simulate_delivery(cfg["deliv"], 10)
        for p in (0, hu.shape[0] - 1):
            _, rho, _ = ctx.mc_dose_phase(p, 1, want_dose=False, want_rho=True)
            want = orc.hu_to_density(cfg["ct_grid"], cfg["hu"][p], cfg["dose_grid"])
            assert (rho.cpu().numpy() == want).all()


def test_density_and_dose_kernels_on_odd_sizes_and_the_whole_hu_range(ctx):
    # a grid whose voxel count is odd (the vectorised kernels' scalar tails), HU values over the whole int16 range
    # (the 65536-entry table; values beyond the table ends are clamped, A4) and a phase pointer that is not 16-byte aligned
    rng = np.random.default_rng(31)
    cfg = synth.config2(n_hist=10)
    g = synth.make_grid((5, 7, 13), (2.0, 2.0, 2.0))
    hu = rng.integers(-32768, 32768, (5 * 7 * 13 + 3,), dtype=np.int64).astype(np.int16)
    hu[:8] = (-32768, 32767, -1000, -1001, 0, 1000, 1001, -999)
    hu_dev = torch.from_numpy(hu).cuda()
    for off in (0, 3):                                                    # off = 3: a 6-byte offset into the buffer
        phase = hu_dev[off:off + 5 * 7 * 13].view(5, 7, 13)
        ctx.set_ct_phases(g, [phase], None)
        fields = synth.make_field((0, 0, 1), (1, 0, 0), (0, 1, 0), (13.0, 7.0, 0.0))
        spots = cfg["spots"][:1].copy(); spots["x_mm"] = 0.0; spots["y_mm"] = 0.0
        ctx.set_plan_spots(fields, spots)
        ctx.simulate_delivery(cfg["deliv"], 2000)
        dose, rho, stats = ctx.mc_dose_phase(0, 7, want_dose=True, want_rho=True)
        want = orc.hu_to_density(g, hu[off:off + 5 * 7 * 13].reshape(5, 7, 13), None)
        assert (rho.cpu().numpy() == want).all()
        # the dose of a voxel without energy is +0, and the grid holds exactly as many non-zero doses as non-zero energies
        Q = ctx.get_phase_energy(0).cpu().numpy()
        d = dose.cpu().numpy()
        assert ((d != 0) == (Q != 0)).all() and (Q != 0).any() and (Q == 0).any()


def test_call_order_and_argument_errors(ctx):
    c = synth.config4(n=16, n_phases=2)
    fresh = binding.Context(0)
    with pytest.raises(RuntimeError, match="-2"):
        fresh.set_dvf(1, 0, c["dvf_grid"], torch.from_numpy(c["disps"][1]).cuda())
    rho = torch.from_numpy(c["rhos"]).cuda()
    fresh.set_density_phases(c["grid"], [rho[0], rho[1]])
    with pytest.raises(RuntimeError, match="-1"):
        fresh.set_dvf(1, 1, c["dvf_grid"], torch.from_numpy(c["disps"][1]).cuda())
    with pytest.raises(RuntimeError, match="-2"):
        fresh.accumulate_subvoxel(0, (2, 2, 2))                      # no doses yet
    with pytest.raises(RuntimeError, match="-2"):
        fresh.mc_dose_phase(0, 1)                                    # no delivery yet
    # grids longer than the kernels' launch geometry allows are refused by the call that receives them, with a message
    # that says so (not by a failed launch later); the buffers are never touched
    tiny = torch.ones(8, dtype=torch.float32, device="cuda")
    for shape in ((1, 262141, 1), (65536, 1, 1)):
        with pytest.raises(RuntimeError, match="-1.*grid too long"):
            fresh.set_density_phases(synth.make_grid(shape, (2.0, 2.0, 2.0)), [tiny])
        with pytest.raises(RuntimeError, match="-1.*dvf_grid: grid too long"):
            fresh.set_dvf(1, 0, synth.make_grid(shape, (2.0, 2.0, 2.0)), tiny)
    with pytest.raises(RuntimeError, match="-1.*2e9"):
        fresh.set_density_phases(synth.make_grid((2000, 2000, 2000), (2.0, 2.0, 2.0)), [tiny])
    fresh.close()


def test_subdivision_convergence_as_in_the_paper(ctx):
    # PAPER.md:167 (Sec. 3.B, Fig. 3): "EMTM with n = 1 ... differs", n = 2 already agrees with much finer
    # subdivisions; the accumulation time grows as n^3.  Soft, qualitative check on config-4-like data:
    # the n = 2 result is several times closer to the n = 8 result than the n = 1 result is, and n = 1 leaves holes
    # (reference voxels that receive no mass) which n >= 2 fills.
    c = synth.config4(n=64, n_phases=4, max_disp_mm=8.0)
    out = {}
    for n in (1, 2, 8):
        o, st, EM = gpu_accumulate(ctx, c, (n, n, n))
        out[n] = o.astype(np.float64)
        holes = sum(int((EM[p][1] == 0).sum()) for p in EM)
        out[(n, "holes")] = holes
    inner = (slice(8, -8),) * 3                                   # away from the faces, where mass leaves the grid
    d1 = np.abs(out[1] - out[8])[inner].mean(); d2 = np.abs(out[2] - out[8])[inner].mean()
    assert d2 < 0.5 * d1, (d1, d2)
    assert out[(1, "holes")] > 5 * max(out[(2, "holes")], 1) or out[(2, "holes")] < out[(1, "holes")]
    assert out[(8, "holes")] <= out[(2, "holes")] <= out[(1, "holes")]


def test_random_geometries_bit_exact(ctx):
    # seeded sweep over anisotropic spacings, grid offsets, DVF grids that are coarser and / or shifted against the dose
    # grid, displacement scales and per-axis subdivisions: the push and (with subdivisions capped at 4) the pull against
    # the oracle.  A 1000-case run of the same generator was clean when the f32x2 kernels went in.
    import test_gpu_dim as td
    rng = np.random.default_rng(20)
    for _ in range(24):
        n = int(rng.integers(18, 44))
        div = int(rng.choice([1, 1, 2]))
        c = synth.config4(n=n, n_phases=3, dvf_div=div, seed=int(rng.integers(1, 10 ** 6)))
        h = rng.choice([0.98, 2.0, 2.5, 1.27, 1.0, 0.7, 3.1], 3).astype(np.float32)
        o = rng.uniform(-300, 300, 3).astype(np.float32)
        shift = rng.uniform(-1.5, 1.5, 3).astype(np.float32) * h if rng.random() < 0.5 else np.zeros(3, np.float32)
        for name in ("grid", "dvf_grid"):
            c[name] = c[name].copy()
        for k, ax in enumerate("xyz"):
            c["grid"]["h" + ax] = h[k]; c["grid"]["o" + ax] = o[k]
            c["dvf_grid"]["h" + ax] = h[k] * div; c["dvf_grid"]["o" + ax] = o[k] + shift[k]
        scale = np.float32(rng.choice([0.05, 0.3, 1.0, 2.0]) * h.mean() / 2.0)
        for p in range(1, 3):
            c["disps"][p] = (c["disps"][p] * scale).astype(np.float32)
        ns = tuple(int(x) for x in rng.choice([1, 2, 3, 4, 5, 8], 3))
        assert_bit_exact(gpu_accumulate(ctx, c, ns), oracle_accumulate(c, ns))
        ns2 = tuple(min(x, 4) for x in ns)
        td.assert_bit_exact(td.gpu_dim(ctx, c, ns2), td.oracle_dim(c, ns2))
