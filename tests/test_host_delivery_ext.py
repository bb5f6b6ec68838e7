"""Host logic: the library's extended delivery simulator (pbs4d_simulate_delivery_ext_host)
against the oracle's (orc_simulate_delivery_ext) -- BIT-EXACT: int64 event simulation, exactly one correct result.
CPU only (the entry needs no device)."""
import numpy as np
import pytest

import oracle as orc
from paper_1809_03927_b200 import binding, synth


def both(fields, spots, prm, H, **ext):
    got = binding.simulate_delivery_ext_host(fields, spots, prm, H, **ext)
    segs, tt, dropped, fills = orc.simulate_delivery_ext(fields, spots, prm, H, **ext)
    assert got["segments"].tobytes() == np.ascontiguousarray(segs).tobytes()
    assert (got["field_time_ns"] == tt).all() and got["dropped_protons"] == dropped and got["fills"] == fills
    assert got["fixed_shift"] == orc.fixed_shift(segs, spots)
    return got


def test_full_size_plans_with_clinical_style_parameters():
    # config-5 plan (3 fields, ~8500 spots, gate on phases 3..7) with App. A style values: 70 ms discard, 2 nC
    # (1.25e10 protons) capacity, 8 s flat-top, energy-dependent reset 1.8-2.2 s, 2 ms fixed spot switch, and breathing
    # periods drawn from N(4.5 s, 0.4 s) by the caller
    rng = np.random.default_rng(5)
    f5 = np.concatenate([synth.make_field((0, 1, 0), (1, 0, 0), (0, 0, 1), (0, 0, 0), sp) for sp in (0, 4, 9)])
    spots5 = synth._plan([0, 1, 2], 90.0, 200.0, 25, 30.0, 6.0, 3.0, rng)
    d5 = synth.make_delivery(n_phases=10, period_s=4.5, repaints=1, gate_mask=0b0011111000, layer_switch_s=2.0)
    periods = np.rint(rng.normal(4.5, 0.4, size=64) * 1e9).astype(np.int64)
    lsw = np.rint(np.linspace(2.2e9, 1.8e9, 25)).astype(np.int64)
    ext = dict(cycle_period_ns=periods, discard_ns=70_000_000, spill_protons_max=12_500_000_000,
               flat_top_ns=8_000_000_000, spot_switch_fixed_ns=2_000_000, layer_switch_ns=lsw)
    a = both(f5, spots5, d5, 10 ** 8, **ext)
    assert int(a["segments"]["n_hist"].sum()) == 10 ** 8 and a["fills"] >= 75
    assert set(int(p) for p in a["segments"]["phase"]) <= {3, 4, 5, 6, 7}
    # iso-layered repainting (max MU per spot delivery) instead of gating
    d5b = synth.make_delivery(n_phases=10, period_s=4.5, layer_switch_s=2.0)
    b = both(f5, spots5, d5b, 10 ** 7, max_protons_per_paint=2_000_000, discard_ns=70_000_000,
             spot_switch_fixed_ns=2_000_000)
    per_spot = np.zeros(len(spots5), np.int64)
    np.add.at(per_spot, b["segments"]["spot"], b["segments"]["protons"])
    assert (per_spot == np.rint(spots5["weight"].astype(np.float64) * 10 ** 7).astype(np.int64)).all()
    assert b["field_time_ns"].min() > binding.simulate_delivery_host(f5, spots5, d5b, 0)["field_time_ns"].max()


def test_all_off_equals_base_entry():
    c = synth.config3(div=4, n_hist=200_000)
    a = binding.simulate_delivery_host(c["fields"], c["spots"], c["deliv"], c["histories"])
    b = binding.simulate_delivery_ext_host(c["fields"], c["spots"], c["deliv"], c["histories"])
    assert a["segments"].tobytes() == b["segments"].tobytes() and (a["field_time_ns"] == b["field_time_ns"]).all()


def test_randomised_parameters_bit_exact():
    rng = np.random.default_rng(78)
    done = 0
    for trial in range(60):
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
        period = int(rng.integers(20_000, 400_000))
        prm = synth.make_delivery(n_phases=P, period_s=period * 1e-9, protons_per_weight=int(rng.integers(1, 20000)),
                                  protons_per_s=int(rng.choice([10 ** 9, 3 * 10 ** 8, 123456789, 4 * 10 ** 9])),
                                  ns_per_um=int(rng.integers(0, 3)), layer_switch_s=float(rng.uniform(0, 1e-4)),
                                  repaints=int(rng.integers(1, 6)), gate_mask=int(rng.integers(1, 1 << P)))
        cyc = None
        if rng.random() < 0.6:
            cyc = rng.integers(int(0.7 * period), int(1.4 * period), size=int(rng.integers(1, 6)))
        per_min = int(period if cyc is None else cyc.min()); per_max = int(period if cyc is None else cyc.max())
        discard = int(rng.integers(0, per_min // P)) if rng.random() < 0.7 else 0
        ext = dict(cycle_period_ns=cyc, discard_ns=discard,
                   spill_protons_max=int(rng.integers(1, 30000)) if rng.random() < 0.6 else 0,
                   flat_top_ns=discard + per_max + int(rng.integers(1, 4 * per_max)) if rng.random() < 0.6 else 0,
                   spot_switch_fixed_ns=int(rng.integers(0, 500)),
                   layer_switch_ns=rng.integers(0, 90_000, size=int(rng.integers(1, 4))) if rng.random() < 0.5 else None,
                   max_protons_per_paint=int(rng.integers(1, 9000)) if rng.random() < 0.5 else 0)
        H = int(rng.integers(0, 5000))
        segs = orc.simulate_delivery_ext(fields, spots, prm, H, **ext)[0]
        if len(segs) == 0:
            continue
        both(fields, spots, prm, H, **ext)
        done += 1
    assert done > 40


def test_bad_arguments():
    c = synth.config3(div=4, n_hist=1000)
    with pytest.raises(RuntimeError):
        binding.simulate_delivery_ext_host(c["fields"], c["spots"], c["deliv"], 10, discard_ns=500_000_000)
    with pytest.raises(RuntimeError):
        binding.simulate_delivery_ext_host(c["fields"], c["spots"], c["deliv"], 10, flat_top_ns=4_000_000_000)
    with pytest.raises(RuntimeError):
        binding.simulate_delivery_ext_host(c["fields"], c["spots"], c["deliv"], 10, spill_protons_max=-1)
