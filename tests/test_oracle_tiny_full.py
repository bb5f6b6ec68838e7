"""SURVEY 8(c) pin "Tiny grid, everything on": the C oracle `orc_transport` against an INDEPENDENT pure-Python
per-history loop on a 4^3 heterogeneous grid, integer grids compared exactly.  CPU only.

The loop below is written from the step list T1-T10 of SURVEY.md 8(c) (model statement BASELINE.json:5,7; PAPER.md:69
names the engine but gives no physics) in Python float64 with its own Philox4x32-10 (checked here against the Random123
known-answer vectors), its own Bethe / Bohr / Highland closed forms and its own geometry, scattering rotation, face
snapping and tie rule.  The only thing it takes from the oracle is the scalar CSDA range table `orc_range_water`, which
is pinned on its own against QUADPACK and PSTAR in test_oracle_physics.py (a second quadrature would differ from the
table by ~1e-9, enough to flip the last bit of some deposits).  Rounding-order differences between this loop and the C
code are ulp-sized; with the fixed-point shift set to 20 an ulp is ~1e-10 of a quantum, so equal integers are expected
unless a step-type decision flips, and a wrong sign, index, transposed basis vector, dropped term or a different tie /
snapping / residual convention changes thousands of quanta."""
import math

import numpy as np
import pytest

import oracle as orc
from paper_1809_03927_b200 import synth

M32 = 0xFFFFFFFF


def philox(ctr, key):
    """T1: Philox4x32-10"""
    c0, c1, c2, c3 = ctr
    k0, k1 = key
    for _ in range(10):
        p0 = 0xD2511F53 * c0
        p1 = 0xCD9E8D57 * c2
        c0, c1, c2, c3 = (p1 >> 32) ^ c1 ^ k0, p1 & M32, (p0 >> 32) ^ c3 ^ k1, p0 & M32
        k0 = (k0 + 0x9E3779B9) & M32
        k1 = (k1 + 0xBB67AE85) & M32
    return c0, c1, c2, c3


def test_python_philox_known_answers():
    # Random123 kat_vectors (SURVEY 8(c) Pins)
    assert philox((0, 0, 0, 0), (0, 0)) == (0x6627e8d5, 0xe169c58d, 0xbc57ac4c, 0x9b00dbd8)
    assert philox((M32,) * 4, (M32, M32)) == (0x408f276d, 0x41c83b0e, 0xa20bc7c6, 0x6d5451fd)
    assert philox((0x243f6a88, 0x85a308d3, 0x13198a2e, 0x03707344), (0xa4093822, 0x299f31d0)) == \
        (0xd16cfe09, 0x94fdcceb, 0x5001e420, 0x24126ea1)


def uniforms(seed, g, block):
    o = philox((block, 0, g & M32, g >> 32), (seed & M32, seed >> 32))
    return [((x >> 9) + 0.5) / 8388608.0 for x in o]                  # T2


# constants of SURVEY section 8's header
K, ME, MP, ZA, I, X0, ES = 0.307075, 0.51099895, 938.27208816, 10.0 / 18.01528, 75.0e-6, 36.08, 13.6


def kinematics(E):
    gam = 1.0 + E / MP
    b2 = 1.0 - 1.0 / (gam * gam)
    tmax = 2.0 * ME * b2 * gam * gam / (1.0 + 2.0 * gam * ME / MP + (ME / MP) ** 2)
    return b2, gam, tmax


def S(E):                                                             # T5
    b2, gam, tmax = kinematics(E)
    return K * ZA / b2 * (0.5 * math.log(2.0 * ME * b2 * gam * gam * tmax / (I * I)) - b2)


def history(grid, rho, field, spot, w, seed, g, scale, Q, tally, mcs=True, spotsize=True):
    """one history, T3-T10; Q is a dict voxel -> int.  mcs / spotsize = False mirror the oracle's pin switches."""
    n = (int(grid["nx"][0]), int(grid["ny"][0]), int(grid["nz"][0]))
    h = (float(grid["hx"][0]), float(grid["hy"][0]), float(grid["hz"][0]))
    o = (float(grid["ox"][0]), float(grid["oy"][0]), float(grid["oz"][0]))
    # T3 source
    u = uniforms(seed, g, 0)
    rad = math.sqrt(-2.0 * math.log(u[0]))
    gx, gy = rad * math.cos(2 * math.pi * u[1]), rad * math.sin(2 * math.pi * u[1])
    gE = math.sqrt(-2.0 * math.log(u[2])) * math.cos(2 * math.pi * u[3])
    if not spotsize:
        gx = gy = 0.0
    E = float(spot["energy_mev"]) * (1.0 + 0.01 * gE)
    a = float(spot["x_mm"]) + float(spot["sigma_mm"]) * gx
    b = float(spot["y_mm"]) + float(spot["sigma_mm"]) * gy
    r = [float(field["ref"][k]) + a * float(field["eu"][k]) + b * float(field["ev"][k]) for k in range(3)]
    d = [float(field["dir"][k]) for k in range(3)]
    tally["inc"] += round_half_even(E * w * scale)
    # ray / box
    t_in, t_out, ax_in = -math.inf, math.inf, None
    for k in range(3):
        lo, hi = o[k], o[k] + n[k] * h[k]
        if d[k] == 0.0:
            if not (lo <= r[k] < hi):
                tally["esc"] += round_half_even(E * w * scale)
                return
            continue
        t1, t2 = sorted(((lo - r[k]) / d[k], (hi - r[k]) / d[k]))
        if t1 > t_in:
            t_in, ax_in = t1, k
        t_out = min(t_out, t2)
    if ax_in is None or not t_in < t_out:
        tally["esc"] += round_half_even(E * w * scale)
        return
    r = [r[k] + t_in * d[k] for k in range(3)]
    idx = [min(max(int(math.floor((r[k] - o[k]) / h[k])), 0), n[k] - 1) for k in range(3)]
    if d[ax_in] > 0:
        idx[ax_in], r[ax_in] = 0, o[ax_in]
    else:
        idx[ax_in], r[ax_in] = n[ax_in] - 1, o[ax_in] + n[ax_in] * h[ax_in]
    m = 0
    while True:
        m += 1
        vox = (idx[2], idx[1], idx[0])
        dens = float(rho[vox])
        R = 10.0 * orc.range_water(E) / dens                           # T5
        dist = []                                                      # T6
        for k in range(3):
            if d[k] > 0:
                dist.append(max(((idx[k] + 1) * h[k] + o[k] - r[k]) / d[k], 0.0))
            elif d[k] < 0:
                dist.append(max((idx[k] * h[k] + o[k] - r[k]) / d[k], 0.0))
            else:
                dist.append(math.inf)
        s_b = min(dist)
        s_lim = min(1.0, 0.02 * R)
        crossing = s_b <= s_lim * (1.0 + 1.0 / 1024.0)                 # reading A22
        s = s_b if crossing else s_lim
        t = dens * s / 10.0                                            # T7
        Em = max(E - 0.5 * (S(E) * t), 1.0e-3)
        dEm = S(Em) * t
        u = uniforms(seed, g, m)                                       # T8
        b2, gam, tmax = kinematics(Em)
        sig = math.sqrt(0.5 * K * ZA / b2 * tmax * (1.0 - 0.5 * b2) * t)
        dE = dEm + sig * (math.sqrt(-2.0 * math.log(u[2])) * math.cos(2 * math.pi * u[3]))
        dE = min(max(dE, 0.0), E)
        ended = E - dE <= 0.5
        if ended:
            dE = E                                                     # A12
        q = round_half_even(dE * w * scale)                            # T9 / T11
        Q[vox] = Q.get(vox, 0) + q
        tally["dep"] += q
        tally["steps"] += 1
        if ended:
            return
        r = [r[k] + s * d[k] for k in range(3)]
        if crossing:                                                   # T10
            for k in range(3):
                if dist[k] == s_b:
                    if d[k] > 0:
                        idx[k] += 1
                        r[k] = idx[k] * h[k] + o[k]
                    else:
                        r[k] = idx[k] * h[k] + o[k]
                        idx[k] -= 1
        if not mcs:
            E -= dE
            if crossing and not all(0 <= idx[k] < n[k] for k in range(3)):
                tally["esc"] += round_half_even(E * w * scale)
                return
            continue
        # T9 deflection at the end of the step
        pv = (Em * Em + 2.0 * Em * MP) / (Em + MP)
        th = math.sqrt((ES / pv) ** 2 / X0 * t) * math.sqrt(-2.0 * math.log(u[0]))
        ph = 2 * math.pi * u[1]
        sw = math.copysign(1.0, d[2])
        aa = -1.0 / (sw + d[2])
        bb = d[0] * d[1] * aa
        e1 = (1.0 + sw * d[0] * d[0] * aa, sw * bb, -sw * d[0])
        e2 = (bb, sw + d[1] * d[1] * aa, -d[1])
        nd = [math.cos(th) * d[k] + math.sin(th) * (math.cos(ph) * e1[k] + math.sin(ph) * e2[k]) for k in range(3)]
        nn = math.sqrt(nd[0] * nd[0] + nd[1] * nd[1] + nd[2] * nd[2])
        d = [c / nn for c in nd]
        E -= dE
        if crossing and not all(0 <= idx[k] < n[k] for k in range(3)):
            tally["esc"] += round_half_even(E * w * scale)
            return


def round_half_even(x):
    return int(round(x))          # Python's round() is half-to-even, as llrint in the default rounding mode


CASES = {
    # name: (direction, eu, ev, ref, energy, sigma)
    "plus_z": ((0, 0, 1), (1, 0, 0), (0, 1, 0), (4.0, 4.0, 0.0), 24.0, 1.5),
    "oblique": ((0.6, 0.0, 0.8), (0.8, 0.0, -0.6), (0, 1, 0), (1.0, 4.0, 0.0), 26.0, 1.0),
    "minus_y_oblique": ((0.36, -0.8, 0.48), (0.8, 0.6, 0.0), (-0.288, 0.384, 0.8), (2.0, 8.0, 3.0), 30.0, 1.2),
}


@pytest.mark.parametrize("case", list(CASES))
def test_tiny_grid_everything_on(case):
    direction, eu, ev, ref, energy, sigma = CASES[case]
    rng = np.random.default_rng(44)
    grid = orc.make_grid((4, 4, 4), (2.0, 2.0, 2.0))
    rho = rng.uniform(0.25, 1.8, size=(4, 4, 4)).astype(np.float32)     # heterogeneous in all three axes
    H = 240
    fields = synth.make_field(direction, eu, ev, ref)
    spots = np.zeros(1, synth.SPOT_DT)
    spots[0] = (0, 0, 0.3, -0.2, energy, sigma, 1.0)
    segs = np.zeros(1, orc.SEG_DT)
    segs[0] = (0, 0, 0, 0, 3 * H, 7, H, 3.0)                            # histories 7 .. 7+H-1, weight 3
    shift, seed = 20, (5 << 32) | 12345                                 # both key words non-zero
    Qo, st, _, _ = orc.transport(grid, rho, fields, spots, segs, seed, shift)

    Q, tally = {}, dict(inc=0, dep=0, esc=0, steps=0)
    for g in range(7, 7 + H):
        history(grid, rho, fields[0], spots[0], 3.0, seed, g, 2.0 ** shift, Q, tally)
    Qp = np.zeros((4, 4, 4), np.int64)
    for vox, q in Q.items():
        Qp[vox] = q

    assert int(st["steps"]) == tally["steps"]                          # same step sequence in every history
    assert (Qo == Qp).all(), f"max |dQ| = {np.abs(Qo - Qp).max()} quanta"
    assert int(st["q_incident"]) == tally["inc"]
    assert int(st["q_deposited"]) == tally["dep"]
    assert int(st["q_escaped"]) == tally["esc"]
    # the case really exercises what it is meant to pin
    assert tally["steps"] > 50 * H                                      # range-limited steps near the end of range
    assert (Qp > 0).sum() >= 20                                         # scattering + spot size spread over the grid
    assert tally["esc"] > 0 and tally["dep"] > 10 * tally["esc"]        # most histories stop inside, some leave


def test_tiny_grid_exact_two_axis_tie():
    # T10 "for each axis attaining the minimum": a 45-degree beam in the x-z plane entering exactly at the grid corner
    # edge crosses an x-face and a z-face at the same distance on every boundary step (MCS and spot size off, so the
    # tie is exact; straggling and energy spread stay on).  Dose must stay on the ix == iz diagonal of the row iy = 1.
    grid = orc.make_grid((4, 4, 4), (2.0, 2.0, 2.0))
    rho = np.random.default_rng(45).uniform(0.4, 1.6, size=(4, 4, 4)).astype(np.float32)
    c = np.float32(math.sqrt(0.5))
    fields = synth.make_field((c, 0, c), (c, 0, -c), (0, 1, 0), (0.0, 3.0, 0.0))
    spots = np.zeros(1, synth.SPOT_DT)
    spots[0] = (0, 0, 0.0, 0.0, 28.0, 0.0, 1.0)
    H = 40
    segs = np.zeros(1, orc.SEG_DT)
    segs[0] = (0, 0, 0, 0, H, 0, H, 1.0)
    Qo, st, _, _ = orc.transport(grid, rho, fields, spots, segs, 77, 20, orc.NO_MCS | orc.NO_SPOTSIZE)
    Q, tally = {}, dict(inc=0, dep=0, esc=0, steps=0)
    for g in range(H):
        history(grid, rho, fields[0], spots[0], 1.0, 77, g, 2.0 ** 20, Q, tally, mcs=False, spotsize=False)
    Qp = np.zeros((4, 4, 4), np.int64)
    for vox, q in Q.items():
        Qp[vox] = q
    assert (Qo == Qp).all() and int(st["steps"]) == tally["steps"]
    assert int(st["q_escaped"]) == tally["esc"] and int(st["q_deposited"]) == tally["dep"]
    on_diag = np.zeros((4, 4, 4), bool)
    for i in range(4):
        on_diag[i, 1, i] = True
    assert (Qo[~on_diag] == 0).all() and (Qo[on_diag] > 0).sum() >= 3
