"""Pins for the transport oracle: closed forms, invariants, brute force on tiny grids.  CPU only.

None of the expected values below comes from the CUDA path: they are the survey's closed-form pins
(tests/golden/transport_pins.txt), integrals evaluated here with scipy QUADPACK, or exact invariants."""
import math

import numpy as np
import pytest
from scipy import integrate, optimize

import oracle as orc
from conftest import golden
from paper_1809_03927_b200 import synth

PINS = {}
for key, e0, arg, val, tol in golden("transport_pins.txt"):
    PINS[(key, int(e0), int(arg))] = (float(val), float(tol))

ALL_OFF = orc.NO_MCS | orc.NO_STRAGGLE | orc.NO_ESPREAD | orc.NO_SPOTSIZE


def pencil(E, n_hist, shape_zyx=(110, 5, 5), h=2.0, flags=0, seed=11, sigma=0.0, rho=None, probe=None,
           direction=(0, 0, 1), eu=(1, 0, 0), ev=(0, 1, 0), ref=None):
    g = orc.make_grid(shape_zyx, (h, h, h))
    nz, ny, nx = shape_zyx
    if rho is None:
        rho = np.ones(shape_zyx, np.float32)
    if ref is None:
        ref = (0.5 * nx * h, 0.5 * ny * h, 0.0)
    fields = synth.make_field(direction, eu, ev, ref)
    spots = np.zeros(1, synth.SPOT_DT)
    spots[0] = (0, 0, 0.0, 0.0, E, sigma, 1.0)
    deliv = synth.make_delivery(n_phases=1, protons_per_weight=n_hist)
    segs, _, _ = orc.simulate_delivery(fields, spots, deliv, n_hist)
    k = orc.fixed_shift(segs, spots)
    Q, st, pxy, stop = orc.transport(g, rho, fields, spots, segs, seed, k, flags, probe_faces=probe, trace=(0, n_hist))
    return dict(Q=Q, st=st, pxy=pxy, stop=stop, k=k, scale=2.0 ** -k, grid=g, rho=rho)


def test_csda_range_and_step_count():
    r = pencil(150.0, 8, flags=ALL_OFF)
    val, tol = PINS[("range_nomcs_nostraggle", 150, 0)]
    assert np.allclose(r["stop"][:, 2], val, atol=tol)
    assert r["st"]["steps"] / r["st"]["histories"] == PINS[("steps_nomcs_nostraggle", 150, 0)][0]
    # = R(E0) - R_c from the range table: midpoint rule (reading A5) is good to ~2 um
    assert r["stop"][0, 2] == pytest.approx(10 * (orc.range_water(150.0) - orc.range_water(0.5)), abs=0.01)
    assert np.allclose(r["stop"][:, 0], 5.0) and np.allclose(r["stop"][:, 1], 5.0)


@pytest.mark.parametrize("flags", [0, ALL_OFF, orc.NO_MCS])
def test_energy_conservation_fixed_point(flags):
    # deposited + escaped = incident, exact to 1/2 LSB per rounding (SURVEY pins: "Energy conservation")
    r = pencil(100.0, 2000, shape_zyx=(30, 9, 9), flags=flags, sigma=3.0)
    st = r["st"]
    assert int(r["Q"].sum()) == int(st["q_deposited"])
    bal = int(st["q_incident"]) - int(st["q_deposited"]) - int(st["q_escaped"])
    assert abs(bal) <= 0.5 * (int(st["steps"]) + 2 * int(st["histories"]))
    assert abs(bal) / int(st["q_incident"]) < 1e-9
    assert int(st["q_escaped"]) > 0 and int(st["q_deposited"]) > 0


def _sigma_range_closed_form(E0):
    # sigma_R^2 = int (d sigma_E^2/dx) / S^3 dE  (range straggling in the CSDA/Gaussian approximation)
    val, _ = integrate.quad(lambda e: orc.bohr_var_per_t(e) / orc.bethe_S(e) ** 3, 0.5, E0, epsrel=1e-9)
    return 10.0 * math.sqrt(val)


@pytest.mark.parametrize("E0", [100, 150])
def test_range_straggling_mono(E0):
    val, tol = PINS[("sigma_range_mono", E0, 0)]
    assert _sigma_range_closed_form(E0) == pytest.approx(val, abs=0.004)
    r = pencil(float(E0), 20000, flags=orc.NO_MCS | orc.NO_ESPREAD | orc.NO_SPOTSIZE)
    z = r["stop"][:, 2]
    assert np.isfinite(z).all()
    assert z.std() == pytest.approx(val, abs=tol)
    # mean stop = CSDA range to the cutoff (straggling is symmetric to first order)
    assert z.mean() == pytest.approx(10 * (orc.range_water(E0) - orc.range_water(0.5)), abs=0.08)


@pytest.mark.parametrize("E0", [100, 150])
def test_range_sigma_with_energy_spread(E0):
    val, tol = PINS[("sigma_range_espread", E0, 0)]
    mono = _sigma_range_closed_form(E0)
    spread = 10.0 * 0.01 * E0 / orc.bethe_S(E0)          # dR/dE * sigma_E
    assert math.hypot(mono, spread) == pytest.approx(val, abs=0.01)
    r = pencil(float(E0), 20000, flags=orc.NO_MCS | orc.NO_SPOTSIZE)
    assert r["stop"][:, 2].std() == pytest.approx(val, abs=tol)


def _fermi_eyges_recursion(E0, z_probe, h=2.0):
    """Deterministic second-moment recursion over the straight-line CSDA step sequence (T6-T7), deflection at the
    END of each step (reading A9): drift A2 += 2 s A1 + s^2 A0, A1 += s A0, then A0 += theta0^2."""
    E, z, A0, A1, A2 = E0, 0.0, 0.0, 0.0, 0.0
    out = {}
    while E > 0.5:
        zb = (math.floor(z / h + 1e-12) + 1) * h
        s_lim = min(1.0, 0.02 * 10 * orc.range_water(E))
        s = zb - z if zb - z <= s_lim * (1 + 1 / 1024) else s_lim
        t = s / 10.0
        Em = max(E - 0.5 * orc.bethe_S(E) * t, 1e-3)
        dE = orc.bethe_S(Em) * t
        A2 += 2 * s * A1 + s * s * A0
        A1 += s * A0
        A0 += orc.theta0_sq_per_t(Em) * t
        z = zb if zb - z <= s_lim * (1 + 1 / 1024) else z + s
        E -= dE
        for zp in z_probe:
            if zp not in out and abs(z - zp) < 1e-9:
                out[zp] = math.sqrt(A2)
    return out


def test_lateral_sigma_matches_fermi_eyges():
    probes = [25, 50, 75]                                   # faces at z = 50, 100, 150 mm
    r = pencil(150.0, 20000, shape_zyx=(110, 41, 41), flags=orc.NO_STRAGGLE | orc.NO_ESPREAD | orc.NO_SPOTSIZE,
               probe=probes)
    fe = _fermi_eyges_recursion(150.0, [50.0, 100.0, 150.0])
    for p, zmm in enumerate([50, 100, 150]):
        val, tol = PINS[("sigma_x", 150, zmm)]
        assert fe[float(zmm)] == pytest.approx(val, rel=2e-3)
        x = r["pxy"][p, :, 0] - 41.0
        y = r["pxy"][p, :, 1] - 41.0
        assert np.isfinite(x).all()
        assert x.std() == pytest.approx(val, abs=tol)
        assert y.std() == pytest.approx(val, abs=tol)
        assert abs(x.mean()) < 4 * val / math.sqrt(x.size) and abs(y.mean()) < 4 * val / math.sqrt(y.size)
        assert abs(np.corrcoef(x, y)[0, 1]) < 0.03
        # continuous Fermi-Eyges integral sits ~1 % above the end-of-step convention
        cont, _ = integrate.quad(lambda zz: (zmm - zz) ** 2 * orc.theta0_sq_per_t(_E_at_depth(150.0, zz)) / 10.0, 0, zmm)
        assert 1.0 <= math.sqrt(cont) / val < 1.025


def _E_at_depth(E0, z_mm):
    """energy after z_mm of water along a straight line, by inverting the range table"""
    R = orc.range_water(E0) - z_mm / 10.0
    if R <= orc.range_water(0.5):
        return 0.5
    return optimize.brentq(lambda e: orc.range_water(e) - R, 0.5, E0, xtol=1e-12)


def test_config1_literal_csda_closed_form():
    c = synth.config1(n_hist=64)
    rho = orc.hu_to_density(c["ct_grid"], c["hu"][0])
    assert (rho == 1.0).all()
    segs, _, _ = orc.simulate_delivery(c["fields"], c["spots"], c["deliv"], 64)
    k = orc.fixed_shift(segs, c["spots"])
    Q, st, _, _ = orc.transport(c["ct_grid"], rho, c["fields"], c["spots"], segs, 1, k, ALL_OFF)
    per = 2.0 ** -k / 64
    val, tol = PINS[("config1_deposit", 150, 0)]
    assert int(st["q_deposited"]) * per == pytest.approx(val, abs=tol)
    val, tol = PINS[("config1_exit", 150, 0)]
    assert int(st["q_escaped"]) * per == pytest.approx(val, abs=tol)
    assert st["steps"] / st["histories"] == 100
    slab = Q.sum((1, 2)) * per
    for (key, e0, arg), (val, tol) in PINS.items():
        if key == "config1_slab":
            assert slab[arg] == pytest.approx(val, abs=tol)
    # every slab = E(z_in) - E(z_out) from the inverted range table
    for kz in (0, 10, 30, 49):
        assert slab[kz] == pytest.approx(_E_at_depth(150.0, 2.0 * kz) - _E_at_depth(150.0, 2.0 * kz + 2.0), abs=2e-4)


def test_config1_full_physics_totals():
    c = synth.config1(n_hist=20000)
    rho = orc.hu_to_density(c["ct_grid"], c["hu"][0])
    segs, _, _ = orc.simulate_delivery(c["fields"], c["spots"], c["deliv"], 20000)
    k = orc.fixed_shift(segs, c["spots"])
    Q, st, _, _ = orc.transport(c["ct_grid"], rho, c["fields"], c["spots"], segs, 1, k)
    per = 2.0 ** -k / 20000
    assert int(st["q_deposited"]) * per == pytest.approx(65.04, abs=0.12)     # SURVEY pin: 65.04 with 1 % spread
    # lateral profile at the entrance slab is the spot Gaussian, sigma 5 mm (+ voxel width^2/12)
    prof = Q[0].sum(0).astype(np.float64)
    x = (np.arange(50) + 0.5) * 2.0
    mean = (prof * x).sum() / prof.sum()
    sig = math.sqrt((prof * (x - mean) ** 2).sum() / prof.sum())
    assert mean == pytest.approx(50.0, abs=0.15)
    assert sig == pytest.approx(math.sqrt(25.0 + 4.0 / 12.0), abs=0.1)
    # dose in Gy per proton (T12): voxel mass 8e-6 kg; central-axis entrance voxel
    D = orc.finalize_dose(c["ct_grid"], rho, Q, k, per_protons=20000)
    e_mev = Q[0, 25, 25] * 2.0 ** -k / 20000
    assert D[0, 25, 25] == pytest.approx(e_mev * 1.602176634e-13 / 8e-6, rel=1e-6)


def test_tiny_grid_brute_force_slabs():
    # 4^3 grid, heterogeneous z-slabs, MCS + straggling off: per-voxel deposit = E(z_in) - E(z_out) along the
    # water-equivalent path (SURVEY pins: "Tiny grid")
    dens = np.array([1.0, 0.3, 1.6, 1.0], np.float32)
    rho = np.broadcast_to(dens[:, None, None], (4, 4, 4)).copy()
    E0 = 30.0
    r = pencil(E0, 4, shape_zyx=(4, 4, 4), flags=ALL_OFF, rho=rho, ref=(3.0, 5.0, 0.0))
    per = r["scale"] / 4
    wed = np.concatenate([[0.0], np.cumsum(dens.astype(np.float64) * 2.0)])
    col = r["Q"][:, 2, 1] * per
    assert int(r["Q"].sum()) == int(r["Q"][:, 2, 1].sum())          # nothing outside the beam's column
    for kz in range(4):
        expect = _E_at_depth(E0, wed[kz]) - _E_at_depth(E0, wed[kz + 1])
        assert col[kz] == pytest.approx(expect, abs=1.5e-3)      # midpoint-rule error at 30 MeV, 1 mm steps
    assert int(r["st"]["q_escaped"]) * per == pytest.approx(_E_at_depth(E0, wed[4]), abs=3e-3)


def test_beam_axis_symmetry_and_miss():
    # straight-line transport along +x, -x, +y gives the transposed/flipped +z result bit for bit
    base = pencil(60.0, 16, shape_zyx=(12, 12, 12), flags=ALL_OFF, ref=(13.0, 9.0, 0.0))
    qz = base["Q"]
    rx = pencil(60.0, 16, shape_zyx=(12, 12, 12), flags=ALL_OFF, direction=(1, 0, 0), eu=(0, 0, 1), ev=(0, 1, 0),
                ref=(0.0, 9.0, 13.0))
    assert (rx["Q"] == qz.transpose(2, 1, 0)).all()
    rmx = pencil(60.0, 16, shape_zyx=(12, 12, 12), flags=ALL_OFF, direction=(-1, 0, 0), eu=(0, 0, 1), ev=(0, 1, 0),
                 ref=(100.0, 9.0, 13.0))
    assert (rmx["Q"] == qz.transpose(2, 1, 0)[:, :, ::-1]).all()
    # a beam that misses the grid deposits nothing and escapes entirely
    miss = pencil(60.0, 16, shape_zyx=(12, 12, 12), flags=ALL_OFF, ref=(100.0, 9.0, 0.0))
    assert int(miss["Q"].sum()) == 0 and int(miss["st"]["q_escaped"]) == int(miss["st"]["q_incident"])
    assert int(miss["st"]["steps"]) == 0


def test_r80_close_to_mean_projected_range():
    r = pencil(100.0, 20000, shape_zyx=(50, 31, 31), sigma=2.0)
    dd = r["Q"].sum((1, 2)).astype(np.float64)
    kmax = int(dd.argmax())
    k = kmax
    while dd[k] > 0.8 * dd[kmax]:
        k += 1
    zc = (np.arange(50) + 0.5) * 2.0
    r80 = zc[k - 1] + (0.8 * dd[kmax] - dd[k - 1]) / (dd[k] - dd[k - 1]) * 2.0
    assert r80 == pytest.approx(10 * orc.range_water(100.0), abs=0.5)      # BASELINE.json: range within 0.5 mm
    stop = r["stop"][:, 2]
    assert r80 == pytest.approx(np.nanmean(stop), abs=0.35)


def test_history_streams_are_independent_of_batching():
    # counter-based RNG: running histories [0,300) at once or as [0,100) + [100,300) gives the same integers
    c = synth.config1(n_hist=300, n=20)
    rho = orc.hu_to_density(c["ct_grid"], c["hu"][0])
    segs, _, _ = orc.simulate_delivery(c["fields"], c["spots"], c["deliv"], 300)
    k = 30
    Qall, _, _, _ = orc.transport(c["ct_grid"], rho, c["fields"], c["spots"], segs, 9, k)
    a = segs.copy(); a["n_hist"] = 100
    b = segs.copy(); b["first_history"] = 100; b["n_hist"] = 200
    Qa, _, _, _ = orc.transport(c["ct_grid"], rho, c["fields"], c["spots"], a, 9, k)
    Qb, _, _, _ = orc.transport(c["ct_grid"], rho, c["fields"], c["spots"], b, 9, k)
    assert (Qall == Qa + Qb).all()
    Qs, _, _, _ = orc.transport(c["ct_grid"], rho, c["fields"], c["spots"], segs, 10, k)
    assert (Qs != Qall).any()
