"""GPU parity: dose-interpolation accumulation (DIM, Eq. 3) vs the oracle -- BIT-EXACT.
Every reference voxel is owned by one thread, the subvoxel sum runs in double in the oracle's (c, b, a) order and the
phases are added in ascending order, so the result is unique.  config4's smooth random fields are used as T^{R->S}."""
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


def gpu_dim(ctx, c, ns, dvf_grids=None):
    P = len(c["doses"])
    rho = torch.from_numpy(c["rhos"]).cuda()
    dose = torch.from_numpy(c["doses"]).cuda()
    ctx.set_density_phases(c["grid"], [rho[p] for p in range(P)])
    for p in range(P):
        if c["disps"][p] is not None:
            ctx.set_dvf_pull(p, c["ref_phase"], c["dvf_grid"] if dvf_grids is None else dvf_grids[p],
                             torch.from_numpy(c["disps"][p]).cuda())
    out, st = ctx.accumulate_dim(c["ref_phase"], ns, [dose[p] for p in range(P)])
    return out.cpu().numpy(), st


def oracle_dim(c, ns, dvf_grids=None):
    P = len(c["doses"])
    grids = [c["dvf_grid"] if dvf_grids is None else dvf_grids[p] for p in range(P)]
    return orc.accumulate_dim(c["grid"], c["doses"], c["disps"], grids, c["ref_phase"], ns)


def assert_bit_exact(g, o):
    (out_g, st_g), (out_o, st_o) = g, o
    assert out_g.view(np.uint32).tobytes() == out_o.view(np.uint32).tobytes()
    for k in ("subvoxels", "dropped_outside_ref", "dropped_outside_dvf"):
        assert st_g[k] == int(st_o[k]), k


@pytest.mark.parametrize("ns", [(1, 1, 1), (2, 2, 2), (3, 3, 3), (4, 4, 4), (2, 2, 5)])
def test_config4_small_bit_exact(ctx, ns):
    c = synth.config4(n=44, n_phases=4)                                    # several 32x4 tiles with ragged tails
    g = gpu_dim(ctx, c, ns)
    assert_bit_exact(g, oracle_dim(c, ns))
    assert g[1]["dropped_outside_ref"] > 0                                 # 20 mm displacements leave the grid


def test_coarse_partial_dvf_grid_and_anisotropic_voxels(ctx):
    c = synth.config4(n=40, n_phases=3, dvf_div=2)
    dg = c["dvf_grid"].copy()
    dg["ox"], dg["oy"], dg["oz"] = 6.0, 3.0, 9.0
    grids = [dg, dg, dg]
    g = gpu_dim(ctx, c, (2, 2, 2), dvf_grids=grids)
    assert_bit_exact(g, oracle_dim(c, (2, 2, 2), dvf_grids=grids))
    assert g[1]["dropped_outside_dvf"] > 0 and (g[0] == 0).any() and (g[0] != 0).any()
    c = synth.config4(n=36, n_phases=3)
    for name in ("grid", "dvf_grid"):
        c[name] = c[name].copy()
        c[name]["hx"], c[name]["hy"], c[name]["hz"] = 0.98, 0.98, 2.5
        c[name]["ox"], c[name]["oy"], c[name]["oz"] = -17.3, 4.1, 100.0
    assert_bit_exact(gpu_dim(ctx, c, (2, 2, 5)), oracle_dim(c, (2, 2, 5)))


def test_spacings_that_exclude_the_known_reciprocal_division(ctx):
    # a spacing whose significand is all ones (0x3FFFFFFF, just below 2 mm) is the exception of Markstein's correction:
    # the launcher must fall back to the IEEE division; a neighbouring spacing takes the fast path.  Also a source grid
    # of a single node along x (the x-neighbour of a dose node is the node itself).
    for hx in (np.nextafter(np.float32(2.0), np.float32(0.0)), np.nextafter(np.float32(2.0), np.float32(3.0))):
        c = synth.config4(n=30, n_phases=3)
        for name in ("grid", "dvf_grid"):
            c[name] = c[name].copy()
            c[name]["hx"] = hx; c[name]["hz"] = 1.27
        assert_bit_exact(gpu_dim(ctx, c, (2, 2, 3)), oracle_dim(c, (2, 2, 3)))
    c = synth.config4(n=24, n_phases=3)
    for name in ("grid", "dvf_grid"):
        c[name] = c[name].copy()
        c[name]["nx"] = 1
    c["doses"] = np.ascontiguousarray(c["doses"][:, :, :, 11:12]); c["rhos"] = np.ascontiguousarray(c["rhos"][:, :, :, 11:12])
    for p in range(1, 3):
        c["disps"][p] = np.ascontiguousarray(c["disps"][p][:, :, :, 11:12])
        c["disps"][p][0] *= 0.02                                           # keep the images inside the single x-voxel
    assert_bit_exact(gpu_dim(ctx, c, (2, 2, 2)), oracle_dim(c, (2, 2, 2)))


def test_identity_field_is_the_plain_sum(ctx):
    # "the same CT image for all phases ... identity" must reproduce the static sum
    c = synth.config4(n=33, n_phases=3)
    for p in range(1, 3):
        c["disps"][p] = np.zeros_like(c["disps"][p])
    out, st = gpu_dim(ctx, c, (1, 1, 1))
    assert np.abs(out - c["doses"].astype(np.float64).sum(0)).max() < 1e-6 * 6
    assert st["dropped_outside_ref"] == 0 and st["dropped_outside_dvf"] == 0


def test_config4_full_size(ctx):
    # BASELINE.json config 4 (10 phases of 128^3, |u| <= 20 mm) at subvoxel edges of 1.0 and 0.5 mm
    c = synth.config4()
    for ns in [(2, 2, 2), (4, 4, 4)]:
        assert_bit_exact(gpu_dim(ctx, c, ns), oracle_dim(c, ns))


def test_argument_and_order_errors(ctx):
    c = synth.config4(n=16, n_phases=2)
    rho = torch.from_numpy(c["rhos"]).cuda()
    ctx.set_density_phases(c["grid"], [rho[0], rho[1]])
    d = torch.from_numpy(c["disps"][1]).cuda()
    with pytest.raises(RuntimeError):
        ctx.set_dvf_pull(1, 1, c["dvf_grid"], d)                           # source == reference
    with pytest.raises(RuntimeError):
        ctx.accumulate_dim(0, (2, 2, 2))                                   # no doses: mc_dose_phase not run, none passed
    with pytest.raises(RuntimeError):
        ctx.accumulate_dim(0, (0, 2, 2), [torch.zeros(16, 16, 16, device="cuda")] * 2)
