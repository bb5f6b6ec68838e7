"""The push kernel (csrc/accumulate.cu, emtm_push_kernel) does not form the contract's destination index on its main
path.  It evaluates an ESTIMATE y of Q - 0.5 (Q = RN(RN(q - o) / h), q = RN(p + RN(c0 + RN(w RN(c1 - c0))))) with the
z-lerp, q = p + u and the division folded into one fma per axis, rounds it to the nearest integer r, and accepts
floor(Q) = r only if y is farther than tol = 2^-23 (8 (n + 2) + 16 U / h + 2 |o| / h) from r +- 0.5 (x, y: |y - r| <=
0.5 - tol; z: y - tol and y + tol round to the same integer).  Everything else goes through the contract's own
operations.  This CPU test restates the RULE in numpy float32 (fma emulated in long double) and checks, on adversarial
inputs whose quotient lies within a few ulp of an integer as well as on random ones, that an accepted estimate always
equals the contract's floor, and that the stated error bound |y - (Q - 0.5)| <= tol / 2.5 holds.  It validates the
arithmetic argument, not the CUDA code (the GPU parity tests do that, bit for bit against the oracle at full size)."""
import numpy as np
import pytest

f32 = np.float32
ld = np.longdouble
MAGIC = f32(12582912.0)                                   # 1.5 * 2^23


def fma32(a, b, c):
    """RN_f32(a b + c): the product of two floats is exact in long double (64-bit significand)"""
    return (a.astype(ld) * b.astype(ld) + c.astype(ld)).astype(f32)


def contract_Q(p, c0, c1, w, o, h):
    dd = (c1 - c0).astype(f32)
    u = (c0 + (w * dd).astype(f32)).astype(f32)
    q = (p + u).astype(f32)
    return ((q - f32(o)).astype(f32) / f32(h)).astype(f32)


def estimate(p, c0, c1, w, o, h):
    ih = f32(1.0) / f32(h)
    P = ((p.astype(np.float64) - np.float64(f32(o))) * (1.0 / np.float64(f32(h))) - 0.5).astype(f32)
    B = ((c1 - c0).astype(f32) * ih).astype(f32)
    A = fma32(c0, np.full_like(c0, ih), P)
    return fma32(w, B, A), A, B, P


def tol_of(n, o, h, U):
    return 2.0 ** -23 * (8.0 * (n + 2) + 16.0 * U / h + 2.0 * abs(o) / h)


def cases(rng, n, o, h, U, m):
    """subvoxels whose image lies within a few float32 ulps of a voxel face (half of them), and random ones"""
    c0 = rng.uniform(-U, U, m).astype(f32)
    c1 = (c0 + rng.uniform(-0.3 * U, 0.3 * U, m).astype(f32)).clip(-U, U).astype(f32)
    w = rng.uniform(0.0, 1.0, m).astype(f32)
    k = rng.integers(0, n + 1, m)
    u = (c0.astype(np.float64) + w.astype(np.float64) * (c1.astype(np.float64) - c0.astype(np.float64)))
    p = (np.float64(o) + k * np.float64(h) - u).astype(f32)       # Q ~ k
    for _ in range(3):                                            # a few floats on either side
        step = rng.integers(-2, 3, m)
        up = np.nextafter(p, f32(np.inf)); dn = np.nextafter(p, f32(-np.inf))
        p = np.where(step > 0, up, np.where(step < 0, dn, p)).astype(f32)
    rnd = rng.uniform(o - 2 * h, o + (n + 2) * h, m).astype(f32)
    return np.where(np.arange(m) % 2 == 0, p, rnd).astype(f32), c0, c1, w


@pytest.mark.parametrize("n,o,h,U", [(128, 0.0, 2.0, 15.3), (128, -128.0, 2.0, 20.0), (512, -250.88, 0.98, 16.0),
                                     (160, 100.0, 2.5, 15.0), (44, -17.3, 0.98, 6.0), (4000, -3000.0, 0.37, 40.0)])
def test_accepted_estimates_equal_the_contract_floor(n, o, h, U):
    rng = np.random.default_rng(int(n * 7 + abs(o)))
    p, c0, c1, w = cases(rng, n, o, h, U, 400_000)
    Q = contract_Q(p, c0, c1, w, o, h)
    want = np.floor(Q)
    y, A, B, P = estimate(p, c0, c1, w, o, h)
    tol = f32(tol_of(n, o, h, U))
    assert tol < 0.25
    relevant = (Q >= -1.0) & (Q <= n + 1.0)

    # the derived bound, with its safety factor
    err = np.abs(y.astype(np.float64) - (Q.astype(np.float64) - 0.5))
    assert err[relevant].max() <= float(tol) / 2.5

    # x / y rule: r = nearest integer of y (ties to even, as the magic-number addition gives)
    t = (y + MAGIC).astype(f32)
    r = (t - MAGIC).astype(f32)
    fr = (y - r).astype(f32)
    accept_xy = np.abs(fr) <= f32(0.5) - tol
    assert (r[accept_xy & relevant] == want[accept_xy & relevant]).all()
    # outside points stay outside: an accepted index is inside [0, n) iff the contract's is
    inside_c = (want >= 0) & (want < n)
    inside_e = (r >= 0) & (r < n)
    assert (inside_c[accept_xy] == inside_e[accept_xy]).all()
    assert accept_xy[::2].mean() < 0.9 and accept_xy[1::2].mean() > 0.95     # the adversarial half really is adversarial

    # z rule: both ends of the tolerance interval round to the same integer
    ih = f32(1.0) / f32(h)
    Az = (c0 * ih).astype(f32)                                               # fma(c0, ih, -+tol) below
    lo = fma32(c0, np.full_like(c0, ih), np.full_like(c0, -tol))
    hi = fma32(c0, np.full_like(c0, ih), np.full_like(c0, tol))
    t1 = (fma32(w, B, (lo + P).astype(f32)) + MAGIC).astype(f32)
    t2 = (fma32(w, B, (hi + P).astype(f32)) + MAGIC).astype(f32)
    accept_z = t1 == t2
    rz = (t1 - MAGIC).astype(f32)
    assert (rz[accept_z & relevant] == want[accept_z & relevant]).all()
    assert (((rz >= 0) & (rz < n))[accept_z] == inside_c[accept_z]).all()
    assert accept_z[1::2].mean() > 0.95
    del Az


def test_exact_integer_quotients_are_never_accepted():
    # Q exactly an integer: the estimate sits on r +- 0.5 and must be sent to the exact path (the n = 8 case that
    # exposed a fused multiply-add in the lerps had Q = 84.0 exactly with y = 83.49999)
    n, o, h, U = 128, 0.0, 2.0, 15.3
    k = np.arange(1, n, dtype=np.float64)
    p = (k * h).astype(f32); z = np.zeros_like(p)
    y, *_ = estimate(p, z, z, z, o, h)
    t = (y + MAGIC).astype(f32); fr = (y - (t - MAGIC)).astype(f32)
    assert (np.abs(fr) > f32(0.5) - f32(tol_of(n, o, h, U))).all()
