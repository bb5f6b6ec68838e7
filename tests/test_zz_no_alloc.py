"""pbs4d_hu_to_density_noalloc -- HU -> density for callers that must not allocate device memory.

Some users of this library cannot let it call cudaMalloc: a planning server or a PyTorch process whose own pool already
holds nearly all of the GPU (a library's private allocation then fails although the pool has room), or a loop with a
latency budget (cudaMalloc takes driver locks, cudaFree waits for the whole device).  For them the library has one entry
point whose scratch -- the 65536-entry table of densities per int16 HU value -- is a static device array inside
libpbs4d.so instead of a buffer owned by a context.  The array is shared by all calls on a device and keeps the previous
call's contents, so the GPU test below makes its calls back to back on one stream, with DIFFERENT tables, and each result
must equal what the ordinary path (pbs4d_set_ct_phases, which allocates) gives for that table: bit for bit, the
tolerance every density test of this repository uses.

This file is named so that pytest collects it last (`pytest -x` stops at the first failure: a failure here hides no
other test).  The GPU test creates its own context and depends on nothing another test left behind; the CPU tests cover
the limits, which are checked before any CUDA call is made.
"""
import ctypes as C

import numpy as np
import pytest

import oracle as orc
from paper_1809_03927_b200 import binding, build, synth

TABLE_A = ((-1000.0, 0.0, 1000.0), (0.001, 1.0, 1.6))                                # the default of set_ct_phases
TABLE_B = ((-1000.0, -200.0, 0.0, 400.0, 3000.0), (0.0012, 0.8, 1.0, 1.3, 2.9))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.load()


def raw_call(lib, n_voxels, hu_pts, rho_pts, hu_ptr=0x1000, out_ptr=0x2000):
    """the C entry point with made-up device addresses: only for calls that are refused before any work is queued"""
    hp = np.asarray(hu_pts, np.float32)
    rp = np.asarray(rho_pts, np.float32)
    err = C.create_string_buffer(200)
    rc = lib.pbs4d_hu_to_density_noalloc(C.c_void_p(hu_ptr), C.c_int64(n_voxels), C.c_int32(len(hp)),
                                         hp.ctypes.data_as(C.c_void_p), rp.ctypes.data_as(C.c_void_p),
                                         C.c_void_p(out_ptr), None, err, C.c_int32(len(err)))
    return rc, err.value.decode()


def test_sizes_beyond_the_fixed_maximum_are_refused_with_a_message(lib):
    # one point more than the kernel-argument table holds: nothing can grow, so the call must say no
    n = binding.NOALLOC_MAX_TABLE_PTS + 1
    rc, msg = raw_call(lib, 8, np.arange(n) * 10.0 - 1000.0, np.full(n, 1.0))
    assert rc == -1 and "2 to 64 points" in msg and f"n_pts = {n}" in msg
    rc, msg = raw_call(lib, binding.NOALLOC_MAX_VOXELS + 1, *TABLE_A)
    assert rc == -1 and "n_voxels" in msg and str(binding.NOALLOC_MAX_VOXELS) in msg
    rc, msg = raw_call(lib, -1, *TABLE_A)
    assert rc == -1 and "n_voxels" in msg
    with pytest.raises(RuntimeError, match="2 to 64 points"):
        binding.hu_to_density_noalloc(None, None, np.arange(n) * 10.0 - 1000.0, np.full(n, 1.0))


def test_bad_tables_and_null_buffers_are_refused(lib):
    assert raw_call(lib, 8, (-1000.0, 0.0, 0.0), (0.001, 1.0, 1.6))[0] == -1          # HU not strictly ascending
    assert raw_call(lib, 8, (-1000.0, 0.0, 100.0), (0.001, 0.0, 1.6))[0] == -1        # a density that is not positive
    assert raw_call(lib, 8, (0.0,), (1.0,))[0] == -1                                  # fewer than two points
    rc, msg = raw_call(lib, 8, *TABLE_A, hu_ptr=None)
    assert rc == -1 and "null" in msg
    assert raw_call(lib, 8, *TABLE_A, out_ptr=None)[0] == -1


def test_no_cpu_fallback(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    rc, msg = raw_call(lib, 0, *TABLE_A)
    assert rc == -3 and "no CPU fallback" in msg                                       # PBS4D_ERR_CUDA


def density_of_the_allocating_path(ctx, grid, hu_phase, table):
    """what pbs4d_set_ct_phases makes of the same HU values (the context's density grid comes back through mc_dose_phase)"""
    nz, ny, nx = synth.grid_shape(grid)
    cfg = synth.config2(n_hist=10)
    ctx.set_ct_phases(grid, [hu_phase], None, *table)
    fields = synth.make_field((0, 0, 1), (1, 0, 0), (0, 1, 0),
                              (0.5 * nx * float(grid["hx"][0]), 0.5 * ny * float(grid["hy"][0]), 0.0))
    spots = cfg["spots"][:1].copy()
    spots["x_mm"] = 0.0
    spots["y_mm"] = 0.0
    ctx.set_plan_spots(fields, spots)
    ctx.simulate_delivery(cfg["deliv"], 16)
    _, rho, _ = ctx.mc_dose_phase(0, 7, want_dose=False, want_rho=True)
    return rho.cpu().numpy()


@pytest.mark.gpu
@pytest.mark.parametrize("shape, offset", [((97, 101, 103), 0),     # 1 009 091 voxels: many blocks, vector body + tail
                                           ((5, 7, 13), 3),         # input 6 bytes off alignment: the scalar path
                                           ((5, 7, 13), 0)])
def test_two_calls_in_a_row_equal_the_allocating_path_bit_for_bit(lib, shape, offset):
    import torch
    nvox = int(np.prod(shape))
    rng = np.random.default_rng(1809 + nvox + offset)
    hu = rng.integers(-32768, 32768, nvox + 8, dtype=np.int64).astype(np.int16)      # the whole int16 range
    hu[offset:offset + 8] = (-32768, 32767, -1000, -1001, 0, 1000, 1001, -999)       # table ends and their neighbours
    grid = synth.make_grid(shape, (2.0, 2.0, 2.0))
    hu_dev = torch.from_numpy(hu).cuda()
    phase = hu_dev[offset:offset + nvox]

    # set-up call (n_voxels = 0), then three conversions queued back to back on one stream: A, B, A again.  The scratch
    # still holds table B's values when the third call starts; its output must show none of them.
    binding.hu_to_density_noalloc(None, None)
    out = [torch.full((nvox,), float("nan"), device="cuda") for _ in range(3)]
    for o, table in zip(out, (TABLE_A, TABLE_B, TABLE_A)):
        assert binding.hu_to_density_noalloc(phase, o, *table) is o
    torch.cuda.synchronize()
    got = [o.cpu().numpy().reshape(shape) for o in out]

    ctx = binding.Context(0)
    try:
        want = [density_of_the_allocating_path(ctx, grid, phase.view(*shape), t) for t in (TABLE_A, TABLE_B)]
    finally:
        ctx.close()
    for g, w in zip(got, (want[0], want[1], want[0])):
        assert g.view(np.uint32).tobytes() == w.view(np.uint32).tobytes()
    assert (got[0] != got[1]).any()                                                   # the two tables do differ
    # and the allocating path itself is pinned to the oracle, so this is too
    for w, t in zip(want, (TABLE_A, TABLE_B)):
        assert (w == orc.hu_to_density(grid, hu[offset:offset + nvox].reshape(shape), None, *t)).all()
