"""The pull kernel (csrc/accumulate.cu, dim_pull_kernel) needs the IEEE quotient RN(e / h) of a coordinate by a grid
spacing as a VALUE (the interpolation weight comes from it, reading D2).  With the reciprocal of the spacing at hand it
is formed without the division sequence -- y = RN(1 / h), q0 = RN(e y), r = e - h q0 (one fma, exact), q1 = RN(q0 + r y)
-- which equals RN(e / h) for every e unless the significand of h is all ones (Markstein's correction; the launcher tests
that proviso and falls back to the division).  This CPU test restates the sequence in numpy float32 (fma emulated in long
double) and checks it EXHAUSTIVELY over all 2^23 significands of e (both signs; the identity is invariant under scaling
e by powers of two, so one binade covers every normal e) for the spacings of the configs and for seeded random ones, and
checks that the excluded divisor really is an exception.  It validates the arithmetic argument; the GPU parity tests
check the kernel bit for bit against the oracle."""
import numpy as np
import pytest

f32 = np.float32
ld = np.longdouble


def fma32(a, b, c):
    return (a.astype(ld) * b.astype(ld) + c.astype(ld)).astype(f32)


def mismatches(h, binade=0):
    h = f32(h)
    inv = f32(1.0) / h
    m = np.arange(2 ** 23, 2 ** 24, dtype=np.int64).astype(np.float64) * 2.0 ** (binade - 23)
    bad = 0
    for sign in (1.0, -1.0):
        e = (m * sign).astype(f32)
        q0 = (e * inv).astype(f32)
        r = fma32(np.full_like(e, -h), q0, e)
        q1 = fma32(r, np.full_like(e, inv), q0)
        bad += int((q1 != (e / h).astype(f32)).sum())
    return bad


SPACINGS = [2.0, 0.98, 2.5, 1.0, 1.27, 0.9765625, 3.0000002]


@pytest.mark.parametrize("h", SPACINGS)
def test_known_reciprocal_division_is_the_ieee_quotient(h):
    assert mismatches(h) == 0


def test_random_spacings_and_another_binade():
    rng = np.random.default_rng(11)
    for h in rng.uniform(0.05, 8.0, 3):
        if (np.float32(h).view(np.uint32) & 0x7FFFFF) != 0x7FFFFF:
            assert mismatches(h, binade=int(rng.integers(-6, 9))) == 0


def test_all_ones_significand_is_the_exception_the_launcher_excludes():
    h = np.nextafter(f32(2.0), f32(0.0))                  # 0x3FFFFFFF
    assert (h.view(np.uint32) & 0x7FFFFF) == 0x7FFFFF
    assert mismatches(h) > 0
