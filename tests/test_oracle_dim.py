"""Pins of the DIM oracle (oracle/orc_dim.c; Eq. 3) against things other than itself:
a library routine (scipy.ndimage.map_coordinates, order 1, float64) for both interpolations, closed forms (identity,
whole-voxel shift, linear ramp, constant dose) and the counting invariants.  CPU only."""
import numpy as np
import pytest
from scipy import ndimage

import oracle as orc


def grid(shape, h, o=(0.0, 0.0, 0.0)):
    return orc.make_grid(shape, h, o)


def centres(g, ns):
    """subvoxel-centre coordinates (float64) per axis: arrays [n*ns]"""
    out = []
    for ax, (n, h, o) in enumerate([(g["nx"][0], g["hx"][0], g["ox"][0]), (g["ny"][0], g["hy"][0], g["oy"][0]),
                                    (g["nz"][0], g["hz"][0], g["oz"][0])]):
        i = np.repeat(np.arange(int(n)), ns[ax])
        a = np.tile(np.arange(ns[ax]), int(n))
        out.append(float(o) + (i + (a + 0.5) / ns[ax]) * float(h))
    return out


def library_dim(R, ns, Dg, disp, S, dose):
    """Eq. 3 with scipy: displacement and dose by map_coordinates(order=1) in float64, mean over the n^3 centres."""
    x, y, z = centres(R, ns)
    Z, Y, X = np.meshgrid(z, y, x, indexing="ij")
    def idx(P, g):   # mm -> continuous index between voxel centres (z, y, x order)
        return [(P[0] - float(g["oz"][0])) / float(g["hz"][0]) - 0.5, (P[1] - float(g["oy"][0])) / float(g["hy"][0]) - 0.5,
                (P[2] - float(g["ox"][0])) / float(g["hx"][0]) - 0.5]
    ci = idx((Z, Y, X), Dg)
    u = [ndimage.map_coordinates(disp[c].astype(np.float64), ci, order=1, mode="nearest") for c in range(3)]
    Q = (Z + u[2], Y + u[1], X + u[0])
    val = ndimage.map_coordinates(dose.astype(np.float64), idx(Q, S), order=1, mode="nearest")
    nz, ny, nx = int(R["nz"][0]), int(R["ny"][0]), int(R["nx"][0])
    return val.reshape(nz, ns[2], ny, ns[1], nx, ns[0]).mean((1, 3, 5))


def smooth_field(rng, shape, amp):
    u = rng.normal(size=(3,) + shape)
    for _ in range(3):
        u = ndimage.uniform_filter(u, size=(1, 3, 3, 3), mode="nearest")
    return (amp * u / np.abs(u).max()).astype(np.float32)


@pytest.mark.parametrize("ns", [(1, 1, 1), (2, 2, 2), (3, 2, 1)])
def test_matches_scipy_map_coordinates(ns):
    rng = np.random.default_rng(11)
    R = grid((10, 12, 14), (2.0, 1.5, 2.5), (-3.0, 1.0, 0.5))
    S = grid((11, 13, 15), (2.0, 1.5, 2.5), (-4.0, 0.0, -1.0))            # source dose grid differs from R
    Dg = grid((6, 7, 8), (4.0, 3.0, 5.0), (-4.0, -0.5, -1.0))              # coarser DVF grid covering R
    disp = smooth_field(rng, (6, 7, 8), 3.0)
    dose = rng.uniform(0.0, 2.0, size=(11, 13, 15)).astype(np.float32)
    got, st = orc.dim_pull(R, ns, Dg, disp, S, dose)
    assert st["subvoxels"] == 10 * 12 * 14 * ns[0] * ns[1] * ns[2]
    # keep the comparison to voxels whose subvoxels all stay inside both extents (the library clamps, the oracle zeroes)
    assert st["dropped_outside_dvf"] == 0
    want = library_dim(R, ns, Dg, disp, S, dose)
    if st["dropped_outside_ref"] == 0:
        assert np.abs(got - want).max() < 5e-6
    else:
        inner = (slice(2, -2),) * 3
        assert np.abs(got - want)[inner].max() < 5e-6


def test_identity_is_exact_for_n1_and_linear_ramp_for_any_n():
    g = grid((8, 9, 10), (2.0, 2.0, 2.0))
    zero = np.zeros((3, 8, 9, 10), np.float32)
    rng = np.random.default_rng(3)
    dose = rng.uniform(0, 3, size=(8, 9, 10)).astype(np.float32)
    got, _ = orc.dim_pull(g, (1, 1, 1), g, zero, g, dose)
    assert (got[:-1, :-1, :-1] == dose[:-1, :-1, :-1].astype(np.float64)).all()     # weights are exactly 0 ...
    assert np.abs(got - dose).max() < 1e-6                               # ... or exactly 1 in the last cell: A + (B - A)
    z, y, x = np.meshgrid(np.arange(8), np.arange(9), np.arange(10), indexing="ij")
    ramp = (0.5 + 0.25 * x + 0.125 * y + 0.0625 * z).astype(np.float32)   # trilinear interpolation is exact on it
    for ns in [(2, 2, 2), (4, 4, 4), (3, 5, 2)]:
        got, _ = orc.dim_pull(g, ns, g, zero, g, ramp)
        assert np.abs(got - ramp)[1:-1, 1:-1, 1:-1].max() < 1e-6          # symmetric subvoxel lattice -> centre value


def test_whole_voxel_shift_and_constant_dose():
    g = grid((6, 6, 8), (2.0, 2.0, 2.0))
    rng = np.random.default_rng(5)
    dose = rng.uniform(0, 3, size=(6, 6, 8)).astype(np.float32)
    disp = np.zeros((3, 6, 6, 8), np.float32)
    disp[0] = 2.0                                                          # T^{R->S}: +1 voxel in x
    got, st = orc.dim_pull(g, (1, 1, 1), g, disp, g, dose)
    assert (got[:-1, :-1, :-2] == dose[:-1, :-1, 1:-1].astype(np.float64)).all()      # weight exactly 0 in every cell
    assert np.abs(got[:, :, :-1] - dose[:, :, 1:]).max() < 1e-6              # last cells: weight exactly 1, A + (B - A)
    assert (got[:, :, -1] == 0.0).all() and st["dropped_outside_ref"] == 36  # x = 17 mm: outside the 16 mm extent
    disp[0] = 3.0                                                          # 1.5 voxels: the last two columns map outside
    got, st = orc.dim_pull(g, (1, 1, 1), g, disp, g, dose)
    assert (got[:, :, -2:] == 0.0).all() and st["dropped_outside_ref"] == 72
    assert np.abs(got[:, :, :-2] - 0.5 * (dose[:, :, 1:-1].astype(np.float64) + dose[:, :, 2:])).max() < 1e-6
    const = np.full((6, 6, 8), 1.25, np.float32)
    wild = smooth_field(rng, (6, 6, 8), 0.45)                             # < half a subvoxel: nothing leaves the grid
    got, st = orc.dim_pull(g, (2, 2, 2), g, wild, g, const)
    assert st["dropped_outside_ref"] == 0 and np.abs(got - 1.25).max() < 1e-6


def test_subvoxels_outside_the_dvf_grid_contribute_nothing_and_finalize_masks():
    R = grid((4, 4, 6), (2.0, 2.0, 2.0))
    Dg = grid((4, 4, 2), (2.0, 2.0, 2.0), (4.0, 0.0, 0.0))                 # DVF covers x in [4, 8) mm only
    disp = np.zeros((3, 4, 4, 2), np.float32)
    dose = np.full((4, 4, 6), 2.0, np.float32)
    got, st = orc.dim_pull(R, (2, 2, 2), Dg, disp, R, dose)
    assert (got[:, :, 2:4] == 2.0).all() and (got[:, :, :2] == 0.0).all() and (got[:, :, 4:] == 0.0).all()
    assert st["dropped_outside_dvf"] == 4 * 4 * 4 * 8
    out, _ = orc.accumulate_dim(R, [dose, dose], [None, disp], [None, Dg], 0, (2, 2, 2))
    assert (out[:, :, 2:4] == 4.0).all() and (out[:, :, :2] == 0.0).all() and (out[:, :, 4:] == 0.0).all()


def test_eq2_sums_phases_in_double():
    g = grid((5, 5, 5), (2.0, 2.0, 2.0))
    rng = np.random.default_rng(9)
    doses = [rng.uniform(0, 2, size=(5, 5, 5)).astype(np.float32) for _ in range(4)]
    zero = np.zeros((3, 5, 5, 5), np.float32)
    out, st = orc.accumulate_dim(g, doses, [None, zero, zero, zero], [None, g, g, g], 0, (1, 1, 1))
    want = (doses[0].astype(np.float64) + doses[1] + doses[2] + doses[3]).astype(np.float32)
    assert (out[:-1, :-1, :-1] == want[:-1, :-1, :-1]).all() and np.abs(out - want).max() < 1e-6
    assert st["subvoxels"] == 3 * 125


@pytest.mark.parametrize("ns", [(2, 2, 2), (4, 2, 4)])
@pytest.mark.parametrize("decades", [0, 30])
def test_subvoxel_sum_order_is_a_free_choice(ns, decades):
    # Reading D4: Eq. 3 is a plain mean and fixes no summation order; the oracle adds the subvoxels
    # of a voxel in (b, a, c) order (z innermost; round 1 used (c, b, a)).  The choice must not matter beyond the
    # rounding of a double sum.  The per-subvoxel values come from the oracle itself at n = 1 on the refined grid: with
    # power-of-two spacings and subdivisions every subvoxel centre of R is, exactly, a voxel centre of the refined grid.
    # decades = 0: doses of one magnitude -- a few fp32 values add up EXACTLY in double, so every order gives the same
    # bits; decades = 30: doses spread over 30 decades, where the additions do round and the orders may part by ulps.
    rng = np.random.default_rng(5)
    shape = (6, 7, 8)
    R = grid(shape, (2.0, 4.0, 2.0), (-1.0, 0.5, 2.0))
    fine = grid((shape[0] * ns[2], shape[1] * ns[1], shape[2] * ns[0]), (2.0 / ns[0], 4.0 / ns[1], 2.0 / ns[2]),
                (-1.0, 0.5, 2.0))
    Dg = grid((5, 6, 7), (4.0, 8.0, 4.0), (-3.0, -4.0, -2.0))
    S = grid((7, 8, 9), (2.0, 4.0, 2.0), (-2.0, -1.5, 1.0))
    disp = smooth_field(rng, (5, 6, 7), 2.5)
    dose = rng.uniform(0.5, 2.0, size=(7, 8, 9)) * 10.0 ** rng.uniform(-decades, 0, size=(7, 8, 9))
    dose = dose.astype(np.float32)
    got, st = orc.dim_pull(R, ns, Dg, disp, S, dose)
    val, st1 = orc.dim_pull(fine, (1, 1, 1), Dg, disp, S, dose)            # one value per subvoxel (0 where dropped)
    assert st1["subvoxels"] == st["subvoxels"] and st1["dropped_outside_ref"] == st["dropped_outside_ref"]
    assert st1["dropped_outside_dvf"] == st["dropped_outside_dvf"] == 0
    v = val.reshape(shape[0], ns[2], shape[1], ns[1], shape[2], ns[0])     # [k, c, j, b, i, a]
    n3 = float(ns[0] * ns[1] * ns[2])

    def summed(order):
        s = np.zeros(shape, np.float64)
        for idx in order:
            s = s + v[:, idx["c"], :, idx["b"], :, idx["a"]]              # one double addition per subvoxel, in order
        return s / n3

    bac = [dict(b=b, a=a, c=c) for b in range(ns[1]) for a in range(ns[0]) for c in range(ns[2])]
    cba = [dict(b=b, a=a, c=c) for c in range(ns[2]) for b in range(ns[1]) for a in range(ns[0])]
    assert (summed(bac) == got).all()                                      # the order the oracle states, bit for bit
    alt = summed(cba)                                                      # the order of round 1
    if decades == 0:
        assert (alt == got).all()
    else:
        assert np.abs(alt - got).max() > 0                                 # here the order does show ...
    assert (np.abs(alt - got) <= 4 * np.spacing(np.abs(got))).all()        # ... by a few ulp of the double sum, no more
    # far below what the fp32 output of Eq. 2 resolves
    assert (alt.astype(np.float32) == got.astype(np.float32)).mean() > 0.999
