"""Pins for the EMTM accumulation oracle (Eq. 2, 4-6).  CPU only."""
import numpy as np
import pytest

import oracle as orc
from paper_1809_03927_b200 import synth

f32 = np.float32


def brute_push(g, dose, rho, dg, disp, ns):
    """Pure-Python per-subvoxel loop with numpy float32 scalars (each operation rounded once, no FMA)."""
    nz, ny, nx = synth.grid_shape(g)
    dz, dy, dx = synth.grid_shape(dg)
    h = [f32(g["hx"][0]), f32(g["hy"][0]), f32(g["hz"][0])]
    o = [f32(g["ox"][0]), f32(g["oy"][0]), f32(g["oz"][0])]
    hd = [f32(dg["hx"][0]), f32(dg["hy"][0]), f32(dg["hz"][0])]
    od = [f32(dg["ox"][0]), f32(dg["oy"][0]), f32(dg["oz"][0])]
    nd = [dx, dy, dz]
    nn = [nx, ny, nz]
    E = np.zeros((nz, ny, nx), np.int64); M = np.zeros((nz, ny, nx), np.int64)
    n_dvf = n_ref = 0
    for k in range(nz):
        for j in range(ny):
            for i in range(nx):
                m_q = int(np.rint(np.float64(rho[k, j, i]) * 2.0 ** 24))
                e_q = int(np.rint(np.float64(rho[k, j, i]) * np.float64(dose[k, j, i]) * 2.0 ** 32))
                for c in range(ns[2]):
                    for b in range(ns[1]):
                        for a in range(ns[0]):
                            idx = (i, j, k); sub = (a, b, c)
                            p, cell, w = [], [], []
                            ok = True
                            for ax in range(3):
                                fa = (f32(sub[ax]) + f32(0.5)) / f32(ns[ax])
                                pa = o[ax] + (f32(idx[ax]) + fa) * h[ax]
                                gq = (pa - od[ax]) / hd[ax] - f32(0.5)
                                if gq < f32(-0.5) or gq >= f32(nd[ax]) - f32(0.5):
                                    ok = False
                                gq = min(max(gq, f32(0)), f32(nd[ax] - 1))
                                i0 = max(min(int(np.floor(gq)), nd[ax] - 2), 0)
                                p.append(pa); cell.append(i0); w.append(f32(gq - f32(i0)))
                            if not ok:
                                n_dvf += 1
                                continue
                            x0, y0, z0 = cell
                            x1, y1, z1 = min(x0 + 1, dx - 1), min(y0 + 1, dy - 1), min(z0 + 1, dz - 1)
                            lerp = lambda A, B, t: f32(A + f32(t * f32(B - A)))
                            dest, inside = [], True
                            for ax in range(3):
                                u = disp[ax]
                                c00 = lerp(u[z0, y0, x0], u[z0, y0, x1], w[0]); c01 = lerp(u[z0, y1, x0], u[z0, y1, x1], w[0])
                                c10 = lerp(u[z1, y0, x0], u[z1, y0, x1], w[0]); c11 = lerp(u[z1, y1, x0], u[z1, y1, x1], w[0])
                                uu = lerp(lerp(c00, c01, w[1]), lerp(c10, c11, w[1]), w[2])
                                q = f32(p[ax] + uu)
                                fl = np.floor(f32(f32(q - o[ax]) / h[ax]))
                                if not (0 <= fl < nn[ax]):
                                    inside = False
                                dest.append(int(fl) if np.isfinite(fl) else -1)
                            if not inside:
                                n_ref += 1
                                continue
                            E[dest[2], dest[1], dest[0]] += e_q
                            M[dest[2], dest[1], dest[0]] += m_q
    return E, M, n_dvf, n_ref


def test_tiny_grid_brute_force():
    rng = np.random.default_rng(21)
    g = synth.make_grid((4, 5, 6), (2.0, 1.5, 2.5), (-3.0, 1.0, 0.5))
    dg = synth.make_grid((3, 4, 4), (2.9, 2.0, 3.1), (-1.9, 0.7, 1.6))       # coarser, slightly smaller than g
    dose = rng.uniform(0, 2, (4, 5, 6)).astype(f32)
    rho = rng.uniform(0.2, 1.6, (4, 5, 6)).astype(f32)
    disp = rng.uniform(-3, 3, (3, 3, 4, 4)).astype(f32)
    for ns in [(2, 2, 2), (3, 1, 2)]:
        E, M, st = orc.emtm_push(g, dose, rho, dg, disp, g, ns)
        Eb, Mb, n_dvf, n_ref = brute_push(g, dose, rho, dg, disp, ns)
        assert (E == Eb).all() and (M == Mb).all()
        assert int(st["dropped_outside_dvf"]) == n_dvf and int(st["dropped_outside_ref"]) == n_ref
        assert n_dvf > 0 and n_ref > 0                       # both drop paths exercised
        assert int(st["subvoxels"]) == 120 * ns[0] * ns[1] * ns[2]


def blobs(n=12, seed=3):
    c = synth.config4(n=n, n_phases=3, seed=seed)
    return c["grid"], c["doses"], c["rhos"]


def test_identity_dvf_reproduces_the_sum_of_phase_doses():
    # PAPER.md:130 (first 3D comparison test): identity DVF, no warping -> accumulated dose = plain sum
    g, doses, rhos = blobs()
    zero = np.zeros((3, 12, 12, 12), f32)
    for ns in [(1, 1, 1), (2, 2, 2), (3, 3, 3)]:
        E, M, st = orc.emtm_push(g, doses[1], rhos[1], g, zero, g, ns)
        assert int(st["dropped_outside_dvf"]) == 0 and int(st["dropped_outside_ref"]) == 0
        D1 = E / M / 256.0
        assert np.abs(D1 - doses[1]).max() < 3e-7 * doses[1].max()
        out, _ = orc.accumulate_subvoxel(g, doses, rhos, [None, zero, zero], [g, g, g], 0, ns)
        assert np.abs(out - doses.astype(np.float64).sum(0)).max() < 6e-7 * doses.max() * 3
    # mass is conserved exactly as integers
    E, M, _ = orc.emtm_push(g, doses[1], rhos[1], g, zero, g, (2, 2, 2))
    assert int(M.sum()) == 8 * int(np.rint(rhos[1].astype(np.float64) * 2 ** 24).sum())


def test_one_voxel_shift():
    g, doses, rhos = blobs()
    shift = np.zeros((3, 12, 12, 12), f32); shift[0] = 2.0                  # +1 voxel in x
    E, M, st = orc.emtm_push(g, doses[1], rhos[1], g, shift, g, (2, 2, 2))
    D = np.where(M > 0, E / np.maximum(M, 1) / 256.0, 0.0)
    assert np.abs(D[:, :, 1:] - doses[1][:, :, :-1]).max() < 3e-7 * doses[1].max()
    assert (M[:, :, 0] == 0).all() and (D[:, :, 0] == 0).all()            # vacated column (reading C4)
    assert int(st["dropped_outside_ref"]) == 12 * 12 * 8                   # last x column pushed out


def test_uniform_dose_is_invariant_under_any_dvf():
    c = synth.config4(n=12, n_phases=2, seed=5, max_disp_mm=5.0)
    g = c["grid"]
    dose = np.full((12, 12, 12), 1.25, f32)
    for ns in [(1, 1, 1), (2, 2, 2)]:
        E, M, st = orc.emtm_push(g, dose, c["rhos"][1], c["dvf_grid"], c["disps"][1], g, ns)
        hit = M > 0
        assert hit.sum() > 1000
        assert np.abs(E[hit] / M[hit] / 256.0 - 1.25).max() < 3e-7 * 1.25
        # integer bookkeeping: everything not dropped landed somewhere
        landed = int(st["subvoxels"]) - int(st["dropped_outside_ref"]) - int(st["dropped_outside_dvf"])
        mq = np.rint(c["rhos"][1].astype(np.float64) * 2 ** 24).astype(np.int64)
        assert int(M.sum()) <= int(mq.sum()) * ns[0] * ns[1] * ns[2]
        assert landed > 0
    # n = 1 leaves holes (EMTM with n = 1 is unstable), n = 2 fills most of them
    E1, M1, _ = orc.emtm_push(g, dose, c["rhos"][1], c["dvf_grid"], c["disps"][1], g, (1, 1, 1))
    E2, M2, _ = orc.emtm_push(g, dose, c["rhos"][1], c["dvf_grid"], c["disps"][1], g, (2, 2, 2))
    assert (M2[2:-2, 2:-2, 2:-2] == 0).sum() <= (M1[2:-2, 2:-2, 2:-2] == 0).sum()


def test_mask_and_reference_phase():
    g, doses, rhos = blobs()
    dg = synth.make_grid((8, 8, 8), (2.0, 2.0, 2.0), (4.0, 4.0, 4.0))       # DVF covers the central 8^3 only
    zero = np.zeros((3, 8, 8, 8), f32)
    out, st = orc.accumulate_subvoxel(g, doses, rhos, [None, zero, None], [g, dg, g], 0, (2, 2, 2))
    inner = np.zeros((12, 12, 12), bool); inner[2:10, 2:10, 2:10] = True
    assert (out[~inner] == 0).all()                                        # PAPER.md:124 mask
    want = doses[0].astype(np.float64) + doses[1]
    assert np.abs(out[inner] - want[inner]).max() < 6e-7 * 4
    assert int(st["dropped_outside_dvf"]) == (12 ** 3 - 8 ** 3) * 8
    # no source phases at all: output is the reference dose (Eq. 2 with an empty sum)
    out0, _ = orc.accumulate_subvoxel(g, doses, rhos, [None, None, None], [g, g, g], 0, (2, 2, 2))
    assert (out0 == doses[0]).all()


def test_per_phase_ratio_then_sum():
    # reading C3: Eq. 5 per phase, then Eq. 2 -- two identical source phases double the mapped dose
    g, doses, rhos = blobs()
    zero = np.zeros((3, 12, 12, 12), f32)
    d = [np.zeros_like(doses[0]), doses[1], doses[1]]
    out, _ = orc.accumulate_subvoxel(g, d, [rhos[0]] * 3, [None, zero, zero], [g, g, g], 0, (2, 2, 2))
    assert np.abs(out - 2.0 * doses[1].astype(np.float64)).max() < 1e-6 * doses[1].max()
