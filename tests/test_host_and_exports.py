"""CPU-side tests of the product: the C-ABI library loads and exports every symbol include/pbs4d.h declares, fails
loudly without a device, and its host delivery simulator is bit-identical to the oracle (BASELINE.json north_star:
"delivery binning must be bit-exact").  No CUDA compute here."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import oracle as orc
from paper_1809_03927_b200 import binding, build, synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.load()


def test_every_declared_symbol_is_exported(lib):
    hdr = open(os.path.join(ROOT, "include", "pbs4d.h")).read()
    declared = set(re.findall(r"\b(pbs4d_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(binding.EXPORTS)
    for name in declared:
        assert getattr(lib, name) is not None


def test_struct_layouts_match_the_header():
    assert binding.GRID_DT.itemsize == 36 and binding.FIELD_DT.itemsize == 52 and binding.SPOT_DT.itemsize == 28
    assert binding.DELIV_DT.itemsize == 56 and binding.SEG_DT.itemsize == 48
    assert C.sizeof(binding.McStats) == 64 and C.sizeof(binding.AccStats) == 32
    for a, b in [(binding.GRID_DT, synth.GRID_DT), (binding.FIELD_DT, synth.FIELD_DT), (binding.SPOT_DT, synth.SPOT_DT),
                 (binding.DELIV_DT, synth.DELIV_DT)]:
        assert a == b


def test_no_cpu_fallback(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    h = C.c_void_p()
    assert lib.pbs4d_create(C.byref(h), C.c_int(0), None) == -3          # PBS4D_ERR_CUDA
    assert not h.value
    with pytest.raises(RuntimeError):
        binding.Context(0)


def test_product_does_not_touch_the_oracle():
    pkg = os.path.join(ROOT, "paper_1809_03927_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cpp", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "orc.h" not in src and \
                    "liborc" not in src, f


CASES = {
    "config3_small": lambda: synth.config3(div=4, n_hist=200_000),
    "config5_small": lambda: synth.config5(div=8, n_hist=300_000),
    "config2": lambda: synth.config2(),
    "config1": lambda: synth.config1(),
}


@pytest.mark.parametrize("name", list(CASES))
def test_delivery_bit_exact_vs_oracle(lib, name):
    c = CASES[name]()
    got = binding.simulate_delivery_host(c["fields"], c["spots"], c["deliv"], c["histories"])
    segs, tt, dropped = orc.simulate_delivery(c["fields"], c["spots"], c["deliv"], c["histories"])
    assert got["segments"].tobytes() == np.ascontiguousarray(segs).tobytes()
    assert (got["field_time_ns"] == tt).all() and got["dropped_protons"] == dropped
    assert got["fixed_shift"] == orc.fixed_shift(segs, c["spots"])


def test_delivery_full_size_plans_bit_exact(lib):
    # plans of configs 3 and 5 at their full spot counts and history totals (phantoms are not needed for delivery)
    rng = np.random.default_rng(3)
    spots3 = synth._plan([0], 70.0, 180.0, 20, 35.0, 6.0, 3.0, rng)
    f3 = synth.make_field((0, 1, 0), (1, 0, 0), (0, 0, 1), (0, 0, 0))
    d3 = synth.make_delivery(n_phases=10, period_s=4.0)
    rng = np.random.default_rng(5)
    f5 = np.concatenate([synth.make_field((0, 1, 0), (1, 0, 0), (0, 0, 1), (0, 0, 0), sp) for sp in (0, 4, 9)])
    spots5 = synth._plan([0, 1, 2], 90.0, 200.0, 25, 30.0, 6.0, 3.0, rng)
    d5 = synth.make_delivery(n_phases=10, period_s=4.5, repaints=4, gate_mask=0b0011111000)
    for f, s, d, H in [(f3, spots3, d3, 10 ** 7), (f5, spots5, d5, 10 ** 8)]:
        got = binding.simulate_delivery_host(f, s, d, H)
        segs, tt, dropped = orc.simulate_delivery(f, s, d, H)
        assert len(segs) > len(s)
        assert got["segments"].tobytes() == np.ascontiguousarray(segs).tobytes()
        assert (got["field_time_ns"] == tt).all() and got["dropped_protons"] == dropped
        assert int(got["segments"]["n_hist"].sum()) == H


def test_delivery_randomised_parameters_bit_exact(lib):
    rng = np.random.default_rng(77)
    for trial in range(40):
        nf = int(rng.integers(1, 4))
        fields = np.concatenate([synth.make_field((0, 0, 1), (1, 0, 0), (0, 1, 0), (0, 0, 0), int(rng.integers(0, 8)))
                                 for _ in range(nf)])
        spots = []
        for f in range(nf):
            for l in range(int(rng.integers(1, 4))):
                for _ in range(int(rng.integers(1, 7))):
                    spots.append((f, l, rng.uniform(-40, 40), rng.uniform(-40, 40), rng.uniform(70, 200), 4.0,
                                  rng.choice([0.0, 1e-7, rng.uniform(0.1, 2.0)])))
        spots = np.array(spots, synth.SPOT_DT)
        P = int(rng.integers(1, 9))
        gate = int(rng.integers(1, 1 << P))
        prm = synth.make_delivery(n_phases=P, period_s=float(rng.uniform(1e-5, 1e-3)),
                                  protons_per_weight=int(rng.integers(1, 20000)),
                                  protons_per_s=int(rng.choice([10 ** 9, 3 * 10 ** 8, 123456789, 4 * 10 ** 9])),
                                  ns_per_um=int(rng.integers(0, 3)), layer_switch_s=float(rng.uniform(0, 1e-4)),
                                  repaints=int(rng.integers(1, 6)), gate_mask=gate)
        H = int(rng.integers(0, 5000))
        segs, tt, dropped = orc.simulate_delivery(fields, spots, prm, H)
        if len(segs) == 0:
            continue
        got = binding.simulate_delivery_host(fields, spots, prm, H)
        assert got["segments"].tobytes() == np.ascontiguousarray(segs).tobytes(), trial
        assert (got["field_time_ns"] == tt).all() and got["dropped_protons"] == dropped


def test_delivery_bad_arguments(lib):
    c = synth.config1()
    bad = c["deliv"].copy(); bad["gate_mask"] = 0
    with pytest.raises(RuntimeError):
        binding.simulate_delivery_host(c["fields"], c["spots"], bad, 10)
    bad = c["deliv"].copy(); bad["n_phases"] = 40
    with pytest.raises(RuntimeError):
        binding.simulate_delivery_host(c["fields"], c["spots"], bad, 10)
