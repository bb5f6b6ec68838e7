"""Thin Python binding of libpbs4d.so (include/pbs4d.h): argument marshalling only.

Every step of the path runs inside the library's CUDA kernels / host simulator; PyTorch supplies device memory
(tensors) and the CUDA stream.  Method names equal the C entry points without the `pbs4d_` prefix.
There is no CPU fallback: a missing library or a missing CUDA device raises RuntimeError.
"""
import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libpbs4d.so")

GRID_DT = np.dtype([("nx", "i4"), ("ny", "i4"), ("nz", "i4"), ("hx", "f4"), ("hy", "f4"), ("hz", "f4"),
                    ("ox", "f4"), ("oy", "f4"), ("oz", "f4")])
FIELD_DT = np.dtype([("dir", "f4", 3), ("eu", "f4", 3), ("ev", "f4", 3), ("ref", "f4", 3), ("start_phase", "i4")])
SPOT_DT = np.dtype([("field", "i4"), ("layer", "i4"), ("x_mm", "f4"), ("y_mm", "f4"), ("energy_mev", "f4"),
                    ("sigma_mm", "f4"), ("weight", "f4")])
DELIV_DT = np.dtype([("n_phases", "i4"), ("period_ns", "i8"), ("protons_per_weight", "i8"), ("protons_per_s", "i8"),
                     ("ns_per_um", "i4"), ("layer_switch_ns", "i8"), ("repaints", "i4"), ("gate_mask", "u4")],
                    align=True)
SEG_DT = np.dtype([("field", "i4"), ("phase", "i4"), ("spot", "i4"), ("pad", "i4"), ("protons", "i8"),
                   ("first_history", "i8"), ("n_hist", "i8"), ("weight", "f8")])

DICOM_DVF_DT = np.dtype([("nx", "i4"), ("ny", "i4"), ("nz", "i4"), ("pad", "i4"), ("start", "f8", 3), ("delta", "f8", 3),
                         ("row_cos", "f8", 3), ("col_cos", "f8", 3), ("pre", "f8", 16), ("post", "f8", 16)])

NO_MCS, NO_STRAGGLE, NO_ESPREAD, NO_SPOTSIZE, TEST_STEP_CAP_64 = 1, 2, 4, 8, 16

EXPORTS = ["pbs4d_create", "pbs4d_destroy", "pbs4d_last_error", "pbs4d_set_ct_phases", "pbs4d_set_density_phases",
           "pbs4d_set_dvf", "pbs4d_set_plan_spots", "pbs4d_set_mc_flags", "pbs4d_simulate_delivery",
           "pbs4d_mc_dose_phase", "pbs4d_mc_dose_phases", "pbs4d_get_phase_energy", "pbs4d_accumulate_subvoxel", "pbs4d_get_accumulators",
           "pbs4d_run_plan_host", "pbs4d_simulate_delivery_host", "pbs4d_roofline_probe",
           "pbs4d_set_dvf_pull", "pbs4d_accumulate_dim", "pbs4d_simulate_delivery_ext", "pbs4d_simulate_delivery_ext_host",
           "pbs4d_build_dvf", "pbs4d_shard_window", "pbs4d_set_shard", "pbs4d_phase_energy_ptr",
           "pbs4d_finalize_phase_dose", "pbs4d_accumulate_push", "pbs4d_accumulator_ptrs", "pbs4d_accumulate_finalize",
           "pbs4d_sample_delivery_trial", "pbs4d_simulate_delivery_trial", "pbs4d_run_trials",
           "pbs4d_hu_to_density_noalloc"]


class PhaseLists(C.Structure):
    _fields_ = [("n_segments", C.c_int64), ("segments", C.c_void_p), ("n_fields", C.c_int32),
                ("field_time_ns", C.POINTER(C.c_int64)), ("dropped_protons", C.c_int64), ("fixed_shift", C.c_int32)]


class DeliveryExt(C.Structure):
    """pbs4d_delivery_ext: extended delivery model (all zero / None = base model)"""
    _fields_ = [("n_cycles", C.c_int32), ("cycle_period_ns", C.c_void_p), ("discard_ns", C.c_int64),
                ("spill_protons_max", C.c_int64), ("flat_top_ns", C.c_int64), ("spot_switch_fixed_ns", C.c_int64),
                ("n_layer_switch", C.c_int32), ("layer_switch_ns", C.c_void_p), ("max_protons_per_paint", C.c_int64)]


def make_delivery_ext(cycle_period_ns=None, discard_ns=0, spill_protons_max=0, flat_top_ns=0, spot_switch_fixed_ns=0,
                      layer_switch_ns=None, max_protons_per_paint=0):
    """-> (DeliveryExt, keepalive arrays); marshalling only"""
    cyc = None if cycle_period_ns is None else np.ascontiguousarray(cycle_period_ns, np.int64)
    lsw = None if layer_switch_ns is None else np.ascontiguousarray(layer_switch_ns, np.int64)
    x = DeliveryExt(0 if cyc is None else len(cyc), None if cyc is None else cyc.ctypes.data, int(discard_ns),
                    int(spill_protons_max), int(flat_top_ns), int(spot_switch_fixed_ns),
                    0 if lsw is None else len(lsw), None if lsw is None else lsw.ctypes.data, int(max_protons_per_paint))
    return x, (cyc, lsw)


class TrialSpec(C.Structure):
    """pbs4d_trial_spec: distributions of the uncertainty trials"""
    _fields_ = [("seed", C.c_uint64), ("n_trials", C.c_int32), ("n_cycles", C.c_int32), ("period_lo_ns", C.c_int64),
                ("period_hi_ns", C.c_int64), ("period_step_ns", C.c_int64), ("period_sigma_ns", C.c_int64),
                ("discard_sigma_ns", C.c_int64), ("flat_top_sigma_ns", C.c_int64), ("spot_switch_sigma_ns", C.c_int64),
                ("layer_switch_sigma_ns", C.c_int64), ("spill_protons_sigma", C.c_int64),
                ("protons_per_s_sigma", C.c_int64)]


class TrialResult(C.Structure):
    _fields_ = [("histories", C.c_uint64), ("delivery_ns", C.c_int64), ("fills", C.c_int64), ("phases_run", C.c_int32),
                ("pad", C.c_int32), ("transport_ms", C.c_float), ("accumulate_ms", C.c_float)]

    def as_dict(self):
        return {n: getattr(self, n) for n, _ in self._fields_ if n != "pad"}


class McStats(C.Structure):
    _fields_ = [("histories", C.c_uint64), ("steps", C.c_uint64), ("q_incident", C.c_int64),
                ("q_deposited", C.c_int64), ("q_escaped", C.c_int64), ("fixed_shift", C.c_int32), ("pad", C.c_int32),
                ("kernel_ms", C.c_float), ("aborted", C.c_int32), ("scoring_atomics", C.c_uint64)]

    def as_dict(self):
        return {n: getattr(self, n) for n, _ in self._fields_ if not n.startswith("pad")}


class AccStats(C.Structure):
    _fields_ = [("subvoxels", C.c_uint64), ("dropped_outside_ref", C.c_uint64), ("dropped_outside_dvf", C.c_uint64),
                ("push_ms", C.c_float), ("finalize_ms", C.c_float)]

    def as_dict(self):
        return {n: getattr(self, n) for n, _ in self._fields_}


_lib = None


def load():
    """dlopen libpbs4d.so; fails loudly if it has not been built (python -m paper_1809_03927_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_1809_03927_b200.build` "
                               "(there is no CPU fallback)")
        lib = C.CDLL(LIB_PATH)
        for name in EXPORTS:
            getattr(lib, name)                                   # AttributeError if a symbol is not exported
        lib.pbs4d_last_error.restype = C.c_char_p
        lib.pbs4d_last_error.argtypes = [C.c_void_p]
        lib.pbs4d_destroy.restype = None
        lib.pbs4d_destroy.argtypes = [C.c_void_p]
        _lib = lib
    return _lib


def _np(a):
    return a.ctypes.data_as(C.c_void_p)


def _ptr_array(tensors):
    arr = (C.c_void_p * len(tensors))()
    for i, t in enumerate(tensors):
        arr[i] = None if t is None else t.data_ptr()
    return arr


def shard_window(n_hist, rank, world):
    """Device-free: (begin, count) of rank's slice of n_hist histories (pbs4d_shard_window)."""
    b, c = C.c_int64(0), C.c_int64(0)
    rc = load().pbs4d_shard_window(C.c_int64(int(n_hist)), C.c_int32(int(rank)), C.c_int32(int(world)), C.byref(b),
                                   C.byref(c))
    if rc != 0:
        raise RuntimeError(f"pbs4d_shard_window: error {rc}")
    return int(b.value), int(c.value)


NOALLOC_MAX_TABLE_PTS, NOALLOC_MAX_VOXELS, NOALLOC_SCRATCH_BYTES = 64, 2_000_000_000, 524288


def hu_to_density_noalloc(hu, out, hu_pts=(-1000.0, 0.0, 1000.0), rho_pts=(0.001, 1.0, 1.6), stream=None):
    """pbs4d_hu_to_density_noalloc: HU -> density for callers that must not allocate device memory (a process whose
    memory pool owns the GPU, a latency-bound loop); no context, no cudaMalloc / cudaFree inside.  `hu` (int16) and `out`
    (float32, same element count) are the caller's contiguous CUDA tensors on the current device; the call only
    enqueues on `stream` (default: torch's current stream) -- synchronise before reading `out`.  The 512 KiB scratch
    is a static device array shared by all calls on a device: calls on one stream may follow each other, calls that
    overlap on the GPU race.  The first call on a device also does the one-time set-up (make it before any stream
    capture).  Without tensors (`hu`, `out` = None) the call runs with n_voxels = 0: argument checks and set-up only.
    Raises RuntimeError with the library's message on failure (too many table points, too many voxels, ...)."""
    import torch
    if hu is None:
        n, hu_ptr, out_ptr = 0, None, None
    else:
        if hu.dtype != torch.int16 or out.dtype != torch.float32 or not hu.is_cuda or not out.is_cuda or \
                not hu.is_contiguous() or not out.is_contiguous() or hu.numel() != out.numel():
            raise ValueError("hu_to_density_noalloc: hu int16 / out float32 contiguous CUDA tensors of one size")
        n, hu_ptr, out_ptr = hu.numel(), C.c_void_p(hu.data_ptr()), C.c_void_p(out.data_ptr())
    hp = np.ascontiguousarray(hu_pts, np.float32)
    rp = np.ascontiguousarray(rho_pts, np.float32)
    if hp.ndim != 1 or hp.shape != rp.shape:
        raise ValueError("hu_to_density_noalloc: hu_pts and rho_pts must be 1-D and of one length")
    if stream is None:
        stream = torch.cuda.current_stream().cuda_stream if torch.cuda.is_available() else 0
    err = C.create_string_buffer(256)
    rc = load().pbs4d_hu_to_density_noalloc(hu_ptr, C.c_int64(n), C.c_int32(len(hp)), _np(hp), _np(rp), out_ptr,
                                            C.c_void_p(stream), err, C.c_int32(len(err)))
    if rc != 0:
        raise RuntimeError(f"pbs4d error {rc}: {err.value.decode()}")
    return out


class _DevView:
    """a device buffer owned by the context, exposed through __cuda_array_interface__ (no copy)"""

    def __init__(self, ptr, shape, typestr):
        self.__cuda_array_interface__ = {"shape": tuple(shape), "typestr": typestr, "data": (int(ptr), False),
                                         "version": 2, "strides": None}


def sample_delivery_trial(spec, trial, n_fields, prm, **ext_kw):
    """Device-free: pbs4d_sample_delivery_trial.  spec: dict of TrialSpec fields.  Returns dict(start_phase, prm (DELIV_DT
    record), ext (keyword arguments of simulate_delivery_ext*))."""
    sp = TrialSpec(**spec)
    p = np.ascontiguousarray(prm, DELIV_DT)
    x, keep = make_delivery_ext(**ext_kw)
    start = np.zeros(n_fields, np.int32)
    cyc = np.zeros(max(sp.n_cycles, 1), np.int64)
    lsw = np.zeros(max(x.n_layer_switch, 1), np.int64)
    p_out = np.zeros(1, DELIV_DT)
    x_out = DeliveryExt()
    rc = load().pbs4d_sample_delivery_trial(C.byref(sp), C.c_int32(trial), C.c_int32(n_fields), _np(p), C.byref(x),
                                            _np(start), _np(cyc), _np(lsw), _np(p_out), C.byref(x_out))
    if rc != 0:
        raise RuntimeError(f"pbs4d_sample_delivery_trial: error {rc}")
    ext = dict(cycle_period_ns=cyc[:sp.n_cycles].copy() if sp.n_cycles > 0 else None, discard_ns=x_out.discard_ns,
               spill_protons_max=x_out.spill_protons_max, flat_top_ns=x_out.flat_top_ns,
               spot_switch_fixed_ns=x_out.spot_switch_fixed_ns,
               layer_switch_ns=lsw[:x.n_layer_switch].copy() if x.n_layer_switch > 0 and x.layer_switch_ns else None,
               max_protons_per_paint=x_out.max_protons_per_paint)
    return dict(start_phase=start, prm=p_out, ext=ext)


def simulate_delivery_host(fields, spots, prm, total_histories):
    """Device-free entry: the host delivery simulator alone (same code path as Context.simulate_delivery)."""
    lib = load()
    f = np.ascontiguousarray(fields, FIELD_DT)
    s = np.ascontiguousarray(spots, SPOT_DT)
    p = np.ascontiguousarray(prm, DELIV_DT)
    n = C.c_int64(0)
    args = [C.c_int32(len(f)), _np(f), C.c_int64(len(s)), _np(s), _np(p), C.c_uint64(int(total_histories))]
    rc = lib.pbs4d_simulate_delivery_host(*args, None, C.c_int64(0), C.byref(n), None, None, None)
    if rc != 0:
        raise RuntimeError(f"pbs4d_simulate_delivery_host: error {rc}")
    segs = np.zeros(n.value, SEG_DT)
    times = np.zeros(len(f), np.int64)
    dropped = C.c_int64(0)
    shift = C.c_int32(0)
    rc = lib.pbs4d_simulate_delivery_host(*args, _np(segs), C.c_int64(n.value), C.byref(n), _np(times),
                                          C.byref(dropped), C.byref(shift))
    if rc != 0:
        raise RuntimeError(f"pbs4d_simulate_delivery_host: error {rc}")
    return dict(segments=segs, field_time_ns=times, dropped_protons=int(dropped.value), fixed_shift=int(shift.value))


def simulate_delivery_ext_host(fields, spots, prm, total_histories, **ext_kw):
    """Device-free entry of the extended delivery model (pbs4d_simulate_delivery_ext_host)."""
    lib = load()
    f = np.ascontiguousarray(fields, FIELD_DT)
    s = np.ascontiguousarray(spots, SPOT_DT)
    p = np.ascontiguousarray(prm, DELIV_DT)
    x, keep = make_delivery_ext(**ext_kw)
    n = C.c_int64(0)
    args = [C.c_int32(len(f)), _np(f), C.c_int64(len(s)), _np(s), _np(p), C.byref(x), C.c_uint64(int(total_histories))]
    rc = lib.pbs4d_simulate_delivery_ext_host(*args, None, C.c_int64(0), C.byref(n), None, None, None, None)
    if rc != 0:
        raise RuntimeError(f"pbs4d_simulate_delivery_ext_host: error {rc}")
    segs = np.zeros(n.value, SEG_DT)
    times = np.zeros(len(f), np.int64)
    dropped = C.c_int64(0); shift = C.c_int32(0); fills = C.c_int64(0)
    rc = lib.pbs4d_simulate_delivery_ext_host(*args, _np(segs), C.c_int64(n.value), C.byref(n), _np(times),
                                              C.byref(dropped), C.byref(shift), C.byref(fills))
    if rc != 0:
        raise RuntimeError(f"pbs4d_simulate_delivery_ext_host: error {rc}")
    return dict(segments=segs, field_time_ns=times, dropped_protons=int(dropped.value), fixed_shift=int(shift.value),
                fills=int(fills.value))


class Context:
    """One pbs4d_ctx on a CUDA device, enqueueing on torch's current stream of that device."""

    def __init__(self, device=0):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("pbs4d needs a CUDA device (no CPU fallback)")
        self.torch = torch
        self.device = torch.device("cuda", device)
        self.lib = load()
        self.h = C.c_void_p()
        stream = torch.cuda.current_stream(self.device).cuda_stream
        rc = self.lib.pbs4d_create(C.byref(self.h), C.c_int(device), C.c_void_p(stream))
        if rc != 0:
            raise RuntimeError(f"pbs4d_create failed with code {rc}")
        self.dose_shape = None

    def close(self):
        if getattr(self, "h", None):
            self.lib.pbs4d_destroy(self.h)
            self.h = None

    __del__ = close

    def _check(self, rc):
        if rc != 0:
            raise RuntimeError(f"pbs4d error {rc}: {self.lib.pbs4d_last_error(self.h).decode()}")

    def _dev(self, t, dtype):
        assert t.is_cuda and t.dtype == dtype and t.is_contiguous(), "expected a contiguous CUDA tensor of " + str(dtype)
        return t

    # ---- a1 ----
    def set_ct_phases(self, ct_grid, hu, dose_grid=None, hu_pts=(-1000.0, 0.0, 1000.0), rho_pts=(0.001, 1.0, 1.6)):
        t = self.torch
        phases = [self._dev(hu[p], t.int16) for p in range(len(hu))]
        ct = np.ascontiguousarray(ct_grid, GRID_DT)
        dg = None if dose_grid is None else np.ascontiguousarray(dose_grid, GRID_DT)
        hp, rp = np.asarray(hu_pts, np.float32), np.asarray(rho_pts, np.float32)
        self._check(self.lib.pbs4d_set_ct_phases(self.h, C.c_int32(len(phases)), _np(ct), _ptr_array(phases),
                                                 None if dg is None else _np(dg), C.c_int32(len(hp)), _np(hp), _np(rp)))
        g = ct if dg is None else dg
        self.dose_shape = (int(g["nz"][0]), int(g["ny"][0]), int(g["nx"][0]))
        self.n_phases = len(phases)

    def set_density_phases(self, dose_grid, rho):
        t = self.torch
        phases = [self._dev(rho[p], t.float32) for p in range(len(rho))]
        g = np.ascontiguousarray(dose_grid, GRID_DT)
        self._check(self.lib.pbs4d_set_density_phases(self.h, C.c_int32(len(phases)), _np(g), _ptr_array(phases)))
        self.dose_shape = (int(g["nz"][0]), int(g["ny"][0]), int(g["nx"][0]))
        self.n_phases = len(phases)

    # ---- a2 ----
    def set_dvf(self, src_phase, ref_phase, dvf_grid, disp):
        g = np.ascontiguousarray(dvf_grid, GRID_DT)
        self._dev(disp, self.torch.float32)
        self._check(self.lib.pbs4d_set_dvf(self.h, C.c_int32(src_phase), C.c_int32(ref_phase), _np(g),
                                           C.c_void_p(disp.data_ptr())))

    def set_dvf_pull(self, src_phase, ref_phase, dvf_grid, disp):
        """T^{R->S} displacement field in the reference frame (dose-interpolation method)"""
        g = np.ascontiguousarray(dvf_grid, GRID_DT)
        self._dev(disp, self.torch.float32)
        self._check(self.lib.pbs4d_set_dvf_pull(self.h, C.c_int32(src_phase), C.c_int32(ref_phase), _np(g),
                                                C.c_void_p(disp.data_ptr())))

    def set_plan_spots(self, fields, spots):
        f = np.ascontiguousarray(fields, FIELD_DT)
        s = np.ascontiguousarray(spots, SPOT_DT)
        self._check(self.lib.pbs4d_set_plan_spots(self.h, C.c_int32(len(f)), _np(f), C.c_int64(len(s)), _np(s)))

    def set_mc_flags(self, flags):
        self._check(self.lib.pbs4d_set_mc_flags(self.h, C.c_uint32(flags)))

    # ---- a3 ----
    def simulate_delivery(self, prm, total_histories):
        p = np.ascontiguousarray(prm, DELIV_DT)
        out = PhaseLists()
        self._check(self.lib.pbs4d_simulate_delivery(self.h, _np(p), C.c_uint64(int(total_histories)), C.byref(out)))
        segs = np.zeros(out.n_segments, SEG_DT)
        if out.n_segments:
            C.memmove(segs.ctypes.data, out.segments, segs.nbytes)
        times = np.array([out.field_time_ns[i] for i in range(out.n_fields)], np.int64)
        return dict(segments=segs, field_time_ns=times, dropped_protons=int(out.dropped_protons),
                    fixed_shift=int(out.fixed_shift))

    def simulate_delivery_ext(self, prm, total_histories, **ext_kw):
        p = np.ascontiguousarray(prm, DELIV_DT)
        x, keep = make_delivery_ext(**ext_kw)
        out = PhaseLists(); fills = C.c_int64(0)
        self._check(self.lib.pbs4d_simulate_delivery_ext(self.h, _np(p), C.byref(x), C.c_uint64(int(total_histories)),
                                                         C.byref(out), C.byref(fills)))
        segs = np.zeros(out.n_segments, SEG_DT)
        if out.n_segments:
            C.memmove(segs.ctypes.data, out.segments, segs.nbytes)
        times = np.array([out.field_time_ns[i] for i in range(out.n_fields)], np.int64)
        return dict(segments=segs, field_time_ns=times, dropped_protons=int(out.dropped_protons),
                    fixed_shift=int(out.fixed_shift), fills=int(fills.value))

    # ---- uncertainty trials ----
    def simulate_delivery_trial(self, spec, trial, prm, total_histories, **ext_kw):
        sp = TrialSpec(**spec)
        p = np.ascontiguousarray(prm, DELIV_DT)
        x, keep = make_delivery_ext(**ext_kw)
        out = PhaseLists(); fills = C.c_int64(0)
        self._check(self.lib.pbs4d_simulate_delivery_trial(self.h, C.byref(sp), C.c_int32(trial), _np(p), C.byref(x),
                                                           C.c_uint64(int(total_histories)), C.byref(out),
                                                           C.byref(fills)))
        segs = np.zeros(out.n_segments, SEG_DT)
        if out.n_segments:
            C.memmove(segs.ctypes.data, out.segments, segs.nbytes)
        times = np.array([out.field_time_ns[i] for i in range(out.n_fields)], np.int64)
        return dict(segments=segs, field_time_ns=times, dropped_protons=int(out.dropped_protons),
                    fixed_shift=int(out.fixed_shift), fills=int(fills.value))

    def run_trials(self, spec, first, count, prm, total_histories, seed, ref_phase, ns_xyz, **ext_kw):
        """-> (list of `count` 4D-dose tensors, list of per-trial result dicts)"""
        t = self.torch
        sp = TrialSpec(**spec)
        p = np.ascontiguousarray(prm, DELIV_DT)
        x, keep = make_delivery_ext(**ext_kw)
        outs = [t.empty(self.dose_shape, dtype=t.float32, device=self.device) for _ in range(count)]
        res = (TrialResult * count)()
        self._check(self.lib.pbs4d_run_trials(self.h, C.byref(sp), C.c_int32(first), C.c_int32(count), _np(p),
                                              C.byref(x), C.c_uint64(int(total_histories)), C.c_uint64(int(seed)),
                                              C.c_int32(ref_phase), C.c_int32(ns_xyz[0]), C.c_int32(ns_xyz[1]),
                                              C.c_int32(ns_xyz[2]), _ptr_array(outs), res))
        return outs, [r.as_dict() for r in res]

    # ---- a4-a7 ----
    def mc_dose_phase(self, phase, seed, per_protons=0.0, want_dose=True, want_rho=False):
        t = self.torch
        dose = t.empty(self.dose_shape, dtype=t.float32, device=self.device) if want_dose else None
        rho = t.empty(self.dose_shape, dtype=t.float32, device=self.device) if want_rho else None
        st = McStats()
        self._check(self.lib.pbs4d_mc_dose_phase(self.h, C.c_int32(phase), C.c_uint64(int(seed)),
                                                 C.c_double(float(per_protons)),
                                                 C.c_void_p(dose.data_ptr() if want_dose else None),
                                                 C.c_void_p(rho.data_ptr() if want_rho else None), C.byref(st)))
        return dose, rho, st.as_dict()

    def mc_dose_phases(self, phases, seed, per_protons=0.0):
        """all listed phases in one call (concurrent launches); -> (list of stats dicts, device ms fork..join);
        the doses stay in the context (accumulate_subvoxel / get_phase_energy)"""
        n = len(phases)
        arr = (C.c_int32 * n)(*[int(p) for p in phases])
        st = (McStats * n)()
        ms = C.c_float(0.0)
        self._check(self.lib.pbs4d_mc_dose_phases(self.h, C.c_int32(n), arr, C.c_uint64(int(seed)),
                                                  C.c_double(float(per_protons)), st, C.byref(ms)))
        return [s.as_dict() for s in st], float(ms.value)

    # ---- sharding over GPUs (one context per rank) ----
    def set_shard(self, rank, world):
        self._check(self.lib.pbs4d_set_shard(self.h, C.c_int32(int(rank)), C.c_int32(int(world))))

    def phase_energy_view(self, phase):
        """int64 tensor aliasing the context's energy grid of `phase` (for an in-place all_reduce)"""
        q = C.c_void_p()
        self._check(self.lib.pbs4d_phase_energy_ptr(self.h, C.c_int32(phase), C.byref(q)))
        return self.torch.as_tensor(_DevView(q.value, self.dose_shape, "<i8"), device=self.device)

    def finalize_phase_dose(self, phase, per_protons=0.0):
        self._check(self.lib.pbs4d_finalize_phase_dose(self.h, C.c_int32(phase), C.c_double(float(per_protons))))

    def accumulate_push(self, ref_phase, ns_xyz, src_mask, phase_doses=None):
        t = self.torch
        ptrs = None
        if phase_doses is not None:
            ptrs = _ptr_array([None if d is None else self._dev(d, t.float32) for d in phase_doses])
        st = AccStats()
        self._check(self.lib.pbs4d_accumulate_push(self.h, C.c_int32(ref_phase), C.c_int32(ns_xyz[0]),
                                                   C.c_int32(ns_xyz[1]), C.c_int32(ns_xyz[2]), ptrs,
                                                   C.c_uint32(int(src_mask)), C.byref(st)))
        return st.as_dict()

    def accumulator_views(self, src_phase):
        """(E, M) int64 tensors aliasing the context's sums of one source phase"""
        e, m = C.c_void_p(), C.c_void_p()
        self._check(self.lib.pbs4d_accumulator_ptrs(self.h, C.c_int32(src_phase), C.byref(e), C.byref(m)))
        t = self.torch
        return (t.as_tensor(_DevView(e.value, self.dose_shape, "<i8"), device=self.device),
                t.as_tensor(_DevView(m.value, self.dose_shape, "<i8"), device=self.device))

    def accumulate_finalize(self, ref_phase, phase_doses=None):
        t = self.torch
        out = t.empty(self.dose_shape, dtype=t.float32, device=self.device)
        ptrs = None
        if phase_doses is not None:
            ptrs = _ptr_array([None if d is None else self._dev(d, t.float32) for d in phase_doses])
        st = AccStats()
        self._check(self.lib.pbs4d_accumulate_finalize(self.h, C.c_int32(ref_phase), ptrs, C.c_void_p(out.data_ptr()),
                                                       C.byref(st)))
        return out, st.as_dict()

    def get_phase_energy(self, phase):
        t = self.torch
        q = t.empty(self.dose_shape, dtype=t.int64, device=self.device)
        self._check(self.lib.pbs4d_get_phase_energy(self.h, C.c_int32(phase), C.c_void_p(q.data_ptr())))
        return q

    # ---- a8-a9 ----
    def accumulate_subvoxel(self, ref_phase, ns_xyz, phase_doses=None):
        t = self.torch
        out = t.empty(self.dose_shape, dtype=t.float32, device=self.device)
        ptrs = None
        if phase_doses is not None:
            ptrs = _ptr_array([None if d is None else self._dev(d, t.float32) for d in phase_doses])
        st = AccStats()
        self._check(self.lib.pbs4d_accumulate_subvoxel(self.h, C.c_int32(ref_phase), C.c_int32(ns_xyz[0]),
                                                       C.c_int32(ns_xyz[1]), C.c_int32(ns_xyz[2]), ptrs,
                                                       C.c_void_p(out.data_ptr()), C.byref(st)))
        return out, st.as_dict()

    def accumulate_dim(self, ref_phase, ns_xyz, phase_doses=None):
        t = self.torch
        out = t.empty(self.dose_shape, dtype=t.float32, device=self.device)
        ptrs = None
        if phase_doses is not None:
            ptrs = _ptr_array([None if d is None else self._dev(d, t.float32) for d in phase_doses])
        st = AccStats()
        self._check(self.lib.pbs4d_accumulate_dim(self.h, C.c_int32(ref_phase), C.c_int32(ns_xyz[0]),
                                                  C.c_int32(ns_xyz[1]), C.c_int32(ns_xyz[2]), ptrs,
                                                  C.c_void_p(out.data_ptr()), C.byref(st)))
        return out, st.as_dict()

    def get_accumulators(self, src_phase):
        t = self.torch
        E = t.empty(self.dose_shape, dtype=t.int64, device=self.device)
        M = t.empty(self.dose_shape, dtype=t.int64, device=self.device)
        self._check(self.lib.pbs4d_get_accumulators(self.h, C.c_int32(src_phase), C.c_void_p(E.data_ptr()),
                                                    C.c_void_p(M.data_ptr())))
        return E, M

    # ---- DVF construction (App. B) ----
    def build_dvf(self, info, delta, want_grid=False):
        """info: DICOM_DVF_DT record; delta: CUDA fp32 [3, nz, ny, nx] -> (r_f, r_f - r_0[, axis-aligned grid])"""
        t = self.torch
        r = np.ascontiguousarray(info, DICOM_DVF_DT)
        self._dev(delta, t.float32)
        rf = t.empty_like(delta); disp = t.empty_like(delta)
        g = np.zeros(1, GRID_DT)
        self._check(self.lib.pbs4d_build_dvf(self.h, _np(r), C.c_void_p(delta.data_ptr()), C.c_void_p(rf.data_ptr()),
                                             C.c_void_p(disp.data_ptr()), _np(g) if want_grid else None))
        return (rf, disp, g) if want_grid else (rf, disp)

    # ---- in-run roofline probes ----
    PROBES = {"fp32_issue": 0, "red_random": 1, "red_hot": 2, "hbm_copy": 3}

    def roofline_probe(self, kind):
        """kind: 'fp32_issue' (lane-instr/s), 'red_random' / 'red_hot' (lane-atomics/s), 'hbm_copy' (B/s)"""
        v = C.c_double(0.0)
        self._check(self.lib.pbs4d_roofline_probe(self.h, C.c_int32(self.PROBES[kind]), C.byref(v)))
        return float(v.value)

    # ---- whole path, host buffers ----
    def run_plan_host(self, ct_grid, hu_host, dose_grid, dvf_grid, disp_host, ref_phase, fields, spots, prm,
                      total_histories, seed, ns_xyz, out_host, hu_pts=(-1000.0, 0.0, 1000.0),
                      rho_pts=(0.001, 1.0, 1.6)):
        """hu_host: list of int16 numpy arrays (or pinned CPU tensors' numpy views); disp_host: list (None = no DVF);
        out_host: float32 numpy array [z,y,x] written in place.  Returns (histories_run, seconds[4], h2d_bytes)."""
        ct = np.ascontiguousarray(ct_grid, GRID_DT)
        dg = None if dose_grid is None else np.ascontiguousarray(dose_grid, GRID_DT)
        vg = None if dvf_grid is None else np.ascontiguousarray(dvf_grid, GRID_DT)
        hp, rp = np.asarray(hu_pts, np.float32), np.asarray(rho_pts, np.float32)
        n = len(hu_host)
        hu_ptrs = (C.c_void_p * n)(*[a.ctypes.data for a in hu_host])
        dp = None
        if disp_host is not None:
            dp = (C.c_void_p * n)(*[None if a is None else a.ctypes.data for a in disp_host])
        f = np.ascontiguousarray(fields, FIELD_DT)
        s = np.ascontiguousarray(spots, SPOT_DT)
        p = np.ascontiguousarray(prm, DELIV_DT)
        run = C.c_uint64(0)
        h2d = C.c_uint64(0)
        secs = (C.c_double * 4)()
        self._check(self.lib.pbs4d_run_plan_host(
            self.h, C.c_int32(n), _np(ct), hu_ptrs, None if dg is None else _np(dg), C.c_int32(len(hp)), _np(hp),
            _np(rp), None if vg is None else _np(vg), dp, C.c_int32(ref_phase), C.c_int32(len(f)), _np(f),
            C.c_int64(len(s)), _np(s), _np(p), C.c_uint64(int(total_histories)), C.c_uint64(int(seed)),
            C.c_int32(ns_xyz[0]), C.c_int32(ns_xyz[1]), C.c_int32(ns_xyz[2]), _np(out_host), C.byref(run), C.byref(h2d),
            secs))
        g = ct if dg is None else dg
        self.dose_shape = (int(g["nz"][0]), int(g["ny"][0]), int(g["nx"][0]))
        self.n_phases = n
        return int(run.value), list(secs), int(h2d.value)
