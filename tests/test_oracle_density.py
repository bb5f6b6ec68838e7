"""Pins for `orc_hu_to_density` (readings A4 / A19; "converting Hounsfield Units to
material density") and `orc_fixed_shift` (reading A18).  CPU only.

Expected values are hand arithmetic on BASELINE.json:8's table (-1000 -> 0.001, 0 -> 1.0, 1000 -> 1.6), numpy block
means, exact conservation laws and hand-computed 1-D overlaps -- none of them is produced by the oracle or by the
CUDA path."""
import math

import numpy as np
import pytest

import oracle as orc

HP = (-1000.0, 0.0, 1000.0)
RP = (0.001, 1.0, 1.6)


def _rho_1d(hu_values, **kw):
    hu = np.asarray(hu_values, np.int16).reshape(1, 1, -1)
    g = orc.make_grid(hu.shape, (1.0, 1.0, 1.0))
    return orc.hu_to_density(g, hu, None, **kw)[0, 0]


def test_table_nodes_interior_points_and_clamps():
    # hand arithmetic (BASELINE.json:8): lower branch rho = 0.001 + (HU + 1000) * 0.999e-3, upper 1 + HU * 0.6e-3
    hu = [-1000, -800, -500, 0, 700, 1000, -2000, 3000, -1, 1, -999, 999]
    want = [0.001, 0.2008, 0.5005, 1.0, 1.42, 1.6, 0.001, 1.6, 0.999001, 1.0006, 0.001999, 1.5994]
    got = _rho_1d(hu)
    assert got.dtype == np.float32
    # the oracle interpolates in double on the fp32 table entries; 1e-7 covers the fp32 rounding of 0.001 and 1.6
    assert np.allclose(got, want, rtol=0, atol=1.5e-7)
    # the clamped values are the table ends themselves (reading A4), bit for bit
    assert got[6] == np.float32(0.001) and got[7] == np.float32(1.6)
    assert got[0] == np.float32(0.001) and got[5] == np.float32(1.6) and got[3] == np.float32(1.0)


def test_table_is_monotone_and_continuous_over_all_int16():
    hu = np.arange(-1100, 1101, dtype=np.int16)
    rho = _rho_1d(hu).astype(np.float64)
    assert (np.diff(rho) >= 0).all()
    d = np.diff(rho[100:-100])                                       # -1000 .. 1000
    assert np.allclose(d[:1000], 0.999e-3, atol=2e-7) and np.allclose(d[1000:], 0.6e-3, atol=2e-7)


def test_general_table_interval_search():
    # a 5-point table with unequal intervals: every interior interval, its two end nodes and its midpoint
    hp = (-1000.0, -200.0, 0.0, 100.0, 2000.0)
    rp = (0.0012, 0.8, 1.0, 1.1, 2.5)
    hu = [-1000, -600, -200, -100, 0, 50, 100, 1050, 2000, 2500, -1500]
    want = [0.0012, 0.4006, 0.8, 0.9, 1.0, 1.05, 1.1, 1.8, 2.5, 2.5, 0.0012]
    assert np.allclose(_rho_1d(hu, hu_pts=hp, rho_pts=rp), want, rtol=0, atol=3e-7)


def _random_hu(rng, shape):
    return rng.integers(-1000, 1000, size=shape).astype(np.int16)


@pytest.mark.parametrize("dose", [((7, 5, 3), (1.7, 2.3, 2.5), (-1.0, 0.5, 2.0)),
                                  ((4, 3, 2), (5.0, 5.0, 5.0), (0.0, 0.0, 0.0)),
                                  ((9, 2, 11), (0.4, 9.0, 0.9), (3.3, 1.0, 0.1))])
def test_resample_constant_stays_constant(dose):
    # a constant HU map resamples to the same constant on ANY dose grid that overlaps the CT (weights are normalised)
    ct = orc.make_grid((10, 12, 14), (1.0, 1.5, 2.0))
    hu = np.full((10, 12, 14), -500, np.int16)
    dg = orc.make_grid(*dose)
    rho = orc.hu_to_density(ct, hu, dg)
    assert rho.shape == dose[0]
    assert np.allclose(rho, 0.5005, rtol=0, atol=1e-6)


def test_resample_integer_ratio_is_a_block_mean():
    rng = np.random.default_rng(21)
    ct = orc.make_grid((8, 12, 16), (2.5, 1.0, 1.0))
    hu = _random_hu(rng, (8, 12, 16))
    fine = orc.hu_to_density(ct, hu).astype(np.float64)
    dg = orc.make_grid((4, 6, 8), (5.0, 2.0, 2.0))                    # 2:1 on every axis, aligned
    rho = orc.hu_to_density(ct, hu, dg)
    # the oracle averages the double-precision table values; the fp32 `fine` differs from them by <= 6e-8
    block = fine.reshape(4, 2, 6, 2, 8, 2).mean(axis=(1, 3, 5))
    assert np.allclose(rho, block, rtol=0, atol=2e-7)
    # 1:1 with an identical grid is the plain table map, bit for bit
    assert (orc.hu_to_density(ct, hu, ct) == orc.hu_to_density(ct, hu)).all()


def test_resample_conserves_mass_when_the_dose_grid_tiles_the_ct():
    # non-integer ratio, but the dose grid covers exactly the CT box: sum rho*V is conserved (overlap-volume weights)
    rng = np.random.default_rng(22)
    ct = orc.make_grid((10, 9, 15), (1.0, 1.0, 1.0))
    hu = _random_hu(rng, (10, 9, 15))
    fine = orc.hu_to_density(ct, hu).astype(np.float64)
    dg = orc.make_grid((4, 6, 6), (2.5, 1.5, 2.5))                    # 15/2.5, 9/1.5, 10/2.5
    rho = orc.hu_to_density(ct, hu, dg).astype(np.float64)
    assert rho.sum() * (2.5 * 1.5 * 2.5) == pytest.approx(fine.sum() * 1.0, rel=2e-7)


def test_resample_hand_computed_non_aligned_1d():
    # CT: 10 voxels of 1 mm along z (config 3's z-axis ratio reversed: dose h = 2.5); densities via the table
    hu_z = np.array([0, 1000, -1000, 0, 500, -500, 0, 0, 1000, -200], np.int16)
    r = np.array([1.0, 1.6, 0.001, 1.0, 1.3, 0.5005, 1.0, 1.0, 1.6, 0.8002])      # hand arithmetic
    ct = orc.make_grid((10, 1, 1), (1.0, 1.0, 1.0))
    dg = orc.make_grid((4, 1, 1), (1.0, 1.0, 2.5))
    rho = orc.hu_to_density(ct, hu_z.reshape(10, 1, 1), dg)[:, 0, 0]
    want = [(r[0] + r[1] + 0.5 * r[2]) / 2.5,             # [0, 2.5): voxels 0, 1 and half of 2
            (0.5 * r[2] + r[3] + r[4]) / 2.5,             # [2.5, 5)
            (r[5] + r[6] + 0.5 * r[7]) / 2.5,             # [5, 7.5)
            (0.5 * r[7] + r[8] + r[9]) / 2.5]             # [7.5, 10)
    assert np.allclose(rho, want, rtol=0, atol=2e-7)
    # transposed operands would show here: the same profile along x and along y
    for shape_ct, shape_d, h_d in [((1, 1, 10), (1, 1, 4), (2.5, 1.0, 1.0)), ((1, 10, 1), (1, 4, 1), (1.0, 2.5, 1.0))]:
        got = orc.hu_to_density(orc.make_grid(shape_ct, (1.0, 1.0, 1.0)), hu_z.reshape(shape_ct),
                                orc.make_grid(shape_d, h_d)).ravel()
        assert np.allclose(got, want, rtol=0, atol=2e-7)


def test_resample_offset_origin_and_edge_overhang():
    # CT box [10, 16) mm in x, 6 voxels of 1 mm; dose voxels of 4 mm starting at x = 7:
    #   [7,11): overlaps CT voxel 0 only (1 mm)      -> rho_0 (weights renormalised to the overlapping part)
    #   [11,15): CT voxels 1..4                       -> mean
    #   [15,19): CT voxel 5 only (1 mm)               -> rho_5
    #   [19,23): no overlap                           -> first table density (vacuum-like air)
    hu = np.array([0, 1000, 1000, -1000, 0, 500], np.int16).reshape(1, 1, 6)
    ct = orc.make_grid((1, 1, 6), (1.0, 1.0, 1.0), (10.0, 0.0, 0.0))
    dg = orc.make_grid((1, 1, 4), (4.0, 1.0, 1.0), (7.0, 0.0, 0.0))
    rho = orc.hu_to_density(ct, hu, dg)[0, 0]
    want = [1.0, (1.6 + 1.6 + 0.001 + 1.0) / 4.0, 1.3, 0.001]
    assert np.allclose(rho, want, rtol=0, atol=2e-7)
    assert rho[3] == np.float32(0.001)
    # partial overlap in two axes at once: dose voxel [-1,1)x[-1,1) over CT voxel (0,0) of a 2x2 map
    hu2 = np.array([[700, 0], [0, 0]], np.int16).reshape(1, 2, 2)
    rho2 = orc.hu_to_density(orc.make_grid((1, 2, 2), (1.0, 1.0, 1.0)), hu2,
                             orc.make_grid((1, 1, 1), (2.0, 2.0, 1.0), (-1.0, -1.0, 0.0)))
    assert rho2[0, 0, 0] == pytest.approx(1.42, abs=2e-7)


# ---------------------------------------------------------------------------------------------------------------
# orc_fixed_shift (T11 / A18): k = min(40, floor(log2(2^62 / (1.1 * sum protons * E_spot))))
# ---------------------------------------------------------------------------------------------------------------
def _segs(protons, spot_ids):
    s = np.zeros(len(protons), orc.SEG_DT)
    s["protons"] = protons
    s["spot"] = spot_ids
    return s


def _spots(energies):
    s = np.zeros(len(energies), orc.SPOT_DT)
    s["energy_mev"] = energies
    return s


def test_fixed_shift_hand_computed():
    # plan A: 1e10 protons at 150 MeV + 3e10 at 100 MeV: 1.1 * 4.5e12 = 4.95e12 = 2^42.17 -> k = floor(19.83) = 19
    assert orc.fixed_shift(_segs([10 ** 10, 3 * 10 ** 10], [0, 1]), _spots([150.0, 100.0])) == 19
    # plan B: 2^20 protons at 128 MeV: 1.1 * 2^27 -> 62 - 27 - log2(1.1) = 34.86 -> k = 34
    assert orc.fixed_shift(_segs([2 ** 20], [0]), _spots([128.0])) == 34
    # just across a power of two: 2^62 / (1.1 * tot) slightly above / below 2^30
    tot_hi = 2.0 ** 32 / 1.1 * (1 - 1e-6)
    tot_lo = 2.0 ** 32 / 1.1 * (1 + 1e-6)
    assert orc.fixed_shift(_segs([int(tot_hi)], [0]), _spots([1.0])) == 30
    assert orc.fixed_shift(_segs([int(tot_lo)], [0]), _spots([1.0])) == 29
    # the spot index of a segment is honoured (energy of spot 2, not of spot 0)
    assert orc.fixed_shift(_segs([2 ** 20], [2]), _spots([1.0, 1.0, 128.0])) == 34
    # cap: a tiny plan would give k = 62 - log2(1.1 * 1000 * 100) = 45.2 -> capped at 40 (LSB never below 2^-40 MeV)
    assert orc.fixed_shift(_segs([1000], [0]), _spots([100.0])) == 40
    assert orc.fixed_shift(_segs([], []), _spots([100.0])) == 40
    # no overflow even if all the energy lands in one voxel
    k = orc.fixed_shift(_segs([10 ** 10, 3 * 10 ** 10], [0, 1]), _spots([150.0, 100.0]))
    assert math.ldexp(4.5e12 * 1.1, k) < 2 ** 62 <= math.ldexp(4.5e12 * 1.1, k + 1)
