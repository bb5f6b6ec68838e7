"""Pins for the oracle's Philox generator and physics closed forms.  CPU only."""
import math

import numpy as np
import pytest
from scipy import integrate

import oracle as orc
from conftest import golden


def test_philox_known_answers():
    for row in golden("philox4x32_10_kat.txt"):
        v = [int(x, 16) for x in row]
        out = orc.philox4x32_10(v[0:4], v[4:6])
        assert [int(x) for x in out] == v[6:10]


def test_philox_counter_and_key_sensitivity():
    # every counter word and key word must matter (a dropped word in the round function would pass the zero vector)
    base = orc.philox4x32_10([1, 2, 3, 4], [5, 6])
    for i in range(4):
        c = [1, 2, 3, 4]
        c[i] ^= 1
        assert (orc.philox4x32_10(c, [5, 6]) != base).all()
    for i in range(2):
        k = [5, 6]
        k[i] ^= 1
        assert (orc.philox4x32_10([1, 2, 3, 4], k) != base).all()


def test_philox_uniformity():
    # T2 mapping u = ((x>>9)+0.5) 2^-23: mean 1/2, variance 1/12 over 4e4 draws
    xs = np.concatenate([orc.philox4x32_10([m, 0, 7, 0], [1, 0]) for m in range(10000)])
    u = ((xs >> 9).astype(np.float64) + 0.5) / 8388608.0
    assert 0.0 < u.min() and u.max() < 1.0
    assert abs(u.mean() - 0.5) < 4 * math.sqrt(1 / 12 / u.size)
    assert abs(u.var() - 1 / 12) < 0.002


def test_bethe_and_range_against_survey_pins():
    for E, S, R in golden("water_bethe_pins.txt"):
        E = float(E)
        if S != "-":
            assert orc.bethe_S(E) == pytest.approx(float(S), rel=2e-5)
        if R != "-":
            assert 10.0 * orc.range_water(E) == pytest.approx(float(R), abs=1.5e-3)


def test_bethe_and_range_against_pstar():
    for E, S, R in golden("pstar_water.txt"):
        E = float(E)
        assert orc.bethe_S(E) == pytest.approx(float(S), rel=2e-3)
        assert orc.range_water(E) == pytest.approx(float(R), rel=3e-3)


def test_range_table_is_the_csda_integral():
    # R(E2) - R(E1) = int dE/S with an independent adaptive quadrature (scipy QUADPACK) of the oracle's own S(E):
    # pins the table construction (node placement, Gauss rule, log-log interpolation), not S itself
    for E1, E2 in [(0.5, 3.0), (3.0, 70.0), (70.0, 150.0), (150.0, 250.0), (0.77, 123.4)]:
        val, _ = integrate.quad(lambda e: 1.0 / orc.bethe_S(e), E1, E2, epsabs=1e-12, epsrel=1e-11)
        assert orc.range_water(E2) - orc.range_water(E1) == pytest.approx(val, rel=1e-8, abs=1e-10)
    # closure at the cutoff (reading A6): R(0.5 MeV) = Ec / S(Ec) = 11.68 um of water
    assert 1e4 * orc.range_water(0.5) == pytest.approx(11.68, abs=0.005)
    assert orc.range_water(0.5) == pytest.approx(0.5 / orc.bethe_S(0.5), rel=1e-12)


def test_bethe_limits():
    # non-relativistic limit: S beta^2 / (K Z/A) -> 1/2 ln(4 me^2 c^4 beta^4 gamma^4 / I^2) - beta^2, monotone decrease
    Es = np.geomspace(0.5, 400.0, 200)
    S = np.array([orc.bethe_S(e) for e in Es])
    assert (np.diff(S) < 0).all()
    # Bragg-Kleeman: R ~ E^p with p ~ 1.77 around 100-200 MeV
    p = math.log(orc.range_water(200.0) / orc.range_water(100.0)) / math.log(2.0)
    assert 1.72 < p < 1.80


def test_bohr_variance_value_and_limit():
    # 200 MeV, 1 mm of water: mean loss 0.449 MeV, sigma 0.104 MeV
    t = 0.1
    assert orc.bethe_S(200.0) * t == pytest.approx(0.449, abs=0.001)
    assert math.sqrt(orc.bohr_var_per_t(200.0) * t) == pytest.approx(0.104, abs=0.001)
    # non-relativistic limit: sigma^2/t -> 4 pi NA re^2 (me c^2)^2 Z/A = K (Z/A) me c^2 = 0.08710 MeV^2 cm^2/g
    # (up to the finite-proton-mass factor 1/(1 + 2 me/Mp) = 1 - 1.09e-3 in T_max)
    assert orc.bohr_var_per_t(0.01) == pytest.approx(0.307075 * (10 / 18.01528) * 0.51099895 / (1 + 2 * 0.51099895 / 938.27208816), rel=5e-5)


def test_highland_theta0():
    # theta0 = 13.6 MeV / (p v) sqrt(t/X0), no log term; 150 MeV: pv = 279.3 MeV (p = 551.3 MeV/c, beta = 0.5066)
    E = 150.0
    p = math.sqrt(E * E + 2 * E * 938.27208816)
    beta = p / (E + 938.27208816)
    pv = p * beta
    assert pv == pytest.approx(279.33, abs=0.05)
    th0 = math.sqrt(orc.theta0_sq_per_t(E) * 1.0)        # 1 g/cm2 = 1 cm of water
    assert th0 == pytest.approx(13.6 / pv * math.sqrt(1.0 / 36.08), rel=1e-12)
    assert th0 == pytest.approx(8.106e-3, rel=1e-3)
