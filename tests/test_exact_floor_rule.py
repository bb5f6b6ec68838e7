"""The call-free exact floor used by the accumulation kernels (csrc/accumulate.cu `exact_floor`) decides
floor(RN(e / h)) near an integer k without dividing: RN(e / h) >= k  <=>  (double)e >= m (double)h, with m the midpoint
between k and the float below it.  This CPU test restates that RULE in numpy (float32 / float64 scalars and arrays) and
checks it against the IEEE float32 division on adversarial inputs -- quotients within a few ulp of integers, powers
of two, voxel sizes with long significands.  It validates the arithmetic argument, not the CUDA code (the GPU parity
tests do that, bit for bit against the oracle at full size).  CPU only."""
import numpy as np
import pytest


def rule(e, h):
    """vectorised restatement of exact_floor's last branch for quotients near an integer k >= 1"""
    e = e.astype(np.float32); h = np.float32(h)
    inv_h = np.float32(1.0) / h
    yq = e * inv_h
    k = np.rint(yq).astype(np.float32)
    kb = k.view(np.int32)
    ex = (kb >> 23) - 127
    half_gap_exp = ex - 24 - ((kb & 0x7FFFFF) == 0)
    m = k.astype(np.float64) - np.ldexp(1.0, half_gap_exp)
    ge = e.astype(np.float64) >= m * np.float64(h)                   # the product is exact in double
    return np.where(ge, k, k - 1).astype(np.int64), k


@pytest.mark.parametrize("h", [2.0, 0.98, 2.5, 1.0, 1.27, 0.3, 3.0000002, 0.1, 7.3e-3])
def test_rule_equals_ieee_division_near_integers(h):
    rng = np.random.default_rng(int(h * 1000) + 5)
    hf = np.float32(h)
    ks = np.concatenate([np.arange(1, 600), 2 ** np.arange(1, 22), 2 ** np.arange(2, 22) - 1, 2 ** np.arange(1, 21) + 1,
                         rng.integers(600, 4_000_000, 3000)]).astype(np.float64)
    base = (ks * np.float64(hf)).astype(np.float32)                   # e with e / h ~ k
    cases = []
    for off in range(-6, 7):                                          # a few floats on either side
        e = base.copy()
        for _ in range(abs(off)):
            e = np.nextafter(e, np.float32(np.inf if off > 0 else -np.inf))
        cases.append(e)
    e = np.concatenate(cases)
    want = np.floor(e / hf).astype(np.int64)                          # numpy float32 division is IEEE RN
    got, k = rule(e, hf)
    near = np.abs(e * (np.float32(1.0) / hf) - k) <= np.abs(e * (np.float32(1.0) / hf)) * 3.0e-7
    assert near.sum() > 0.5 * near.size                               # the cases really are the near-integer ones
    assert (got[near] == want[near]).all()
    # both outcomes occur (the rule is not trivially "always k")
    assert (got[near] == k[near]).any() and (got[near] == k[near] - 1).any()


def test_product_multiplication_estimate_is_within_the_stated_bound():
    # |RN(e inv_h) - RN(e / h)| <= (2^-23 + 2^-24) |y|: the bound the kernel's tolerance rests on
    rng = np.random.default_rng(9)
    for h in (0.98, 2.0, 2.5, 1.27, 0.37):
        hf = np.float32(h)
        e = rng.uniform(-50.0, 1200.0, 400_000).astype(np.float32)
        y = e * (np.float32(1.0) / hf)
        q = e / hf
        assert (np.abs(y.astype(np.float64) - q.astype(np.float64)) <= 1.8e-7 * np.abs(q.astype(np.float64)) + 1e-45).all()
