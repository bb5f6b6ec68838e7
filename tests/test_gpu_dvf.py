"""GPU parity: DVF construction from DICOM minimal grid information (Eq. 7-8) vs the oracle --
BIT-EXACT (double arithmetic in the same order, no fused multiply-add on either side), on the deformation-grid shapes of
the paper's Table I (~180 x 120 x 160 at ~2.55 mm), then used end to end: the constructed displacement field drives the
EMTM accumulation through set_dvf exactly as a directly supplied one."""
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


def make_info(shape, start, delta, U=(1, 0, 0), V=(0, 1, 0), pre=None, post=None):
    r = np.zeros(1, binding.DICOM_DVF_DT)
    r["nz"], r["ny"], r["nx"] = shape
    r["start"], r["delta"], r["row_cos"], r["col_cos"] = start, delta, U, V
    r["pre"] = (np.eye(4) if pre is None else pre).ravel()
    r["post"] = (np.eye(4) if post is None else post).ravel()
    return r


def rigid(rng):
    q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
    M = np.eye(4); M[:3, :3] = q; M[:3, 3] = rng.uniform(-30, 30, 3)
    return M


def test_table1_sized_grid_bit_exact(ctx):
    rng = np.random.default_rng(41)
    q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
    for U, V, pre, post in [((1, 0, 0), (0, 1, 0), None, None), (q[:, 0], q[:, 1], rigid(rng), rigid(rng))]:
        info = make_info((160, 120, 181), (-229.5, -152.3, -40.0), (2.55, 2.55, 2.5), U, V, pre, post)   # odd nx: ragged tail
        delta = rng.uniform(-7.5, 7.5, size=(3, 160, 120, 181)).astype(np.float32)
        rf, disp = ctx.build_dvf(info, torch.from_numpy(delta).cuda())
        rf_o, disp_o = orc.build_dvf(info, delta)
        assert rf.cpu().numpy().view(np.uint32).tobytes() == rf_o.view(np.uint32).tobytes()
        assert disp.cpu().numpy().view(np.uint32).tobytes() == disp_o.view(np.uint32).tobytes()


def test_constructed_field_drives_the_accumulation(ctx):
    # identity matrices + axis-aligned cosines (the 4DCT case): the constructed displacement equals the
    # stored translation, the returned grid equals the DVF grid, and accumulate_subvoxel gives the same bits
    c = synth.config4(n=40, n_phases=3, dvf_div=2)
    P = 3
    rho = torch.from_numpy(c["rhos"]).cuda(); dose = torch.from_numpy(c["doses"]).cuda()
    dg = c["dvf_grid"]
    info = make_info((int(dg["nz"][0]), int(dg["ny"][0]), int(dg["nx"][0])),
                     tuple(float(dg[o][0]) + 0.5 * float(dg[h][0]) for o, h in (("ox", "hx"), ("oy", "hy"), ("oz", "hz"))),
                     (float(dg["hx"][0]), float(dg["hy"][0]), float(dg["hz"][0])))
    outs = []
    for constructed in (False, True):
        ctx.set_density_phases(c["grid"], [rho[p] for p in range(P)])
        for p in (1, 2):
            d = torch.from_numpy(c["disps"][p]).cuda()
            if constructed:
                _, disp, g = ctx.build_dvf(info, d, want_grid=True)
                assert g.tobytes() == np.ascontiguousarray(dg, binding.GRID_DT).tobytes()
                assert (disp == d).all()
                ctx.set_dvf(p, 0, g, disp)
            else:
                ctx.set_dvf(p, 0, dg, d)
        out, _ = ctx.accumulate_subvoxel(0, (2, 2, 2), [dose[p] for p in range(P)])
        outs.append(out.cpu().numpy())
    assert outs[0].view(np.uint32).tobytes() == outs[1].view(np.uint32).tobytes()
    with pytest.raises(RuntimeError):                                    # an oblique grid has no axis-aligned descriptor
        ctx.build_dvf(make_info((4, 4, 4), (0, 0, 0), (1, 1, 1), U=(0, 1, 0), V=(1, 0, 0)),
                      torch.zeros(3, 4, 4, 4, device="cuda"), want_grid=True)
