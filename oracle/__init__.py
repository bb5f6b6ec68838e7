"""CPU ORACLE for the pbs4d hot path -- TEST INFRASTRUCTURE ONLY.

ctypes wrapper (argument marshalling only) around oracle/liborc.so, the plain double-precision C restatement of
SURVEY.md 8(c) steps D1-D7 / T1-T12 / A1-A6 written from PAPER.md (arxiv 1809.03927) and BASELINE.json.
Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this package;
it imports nothing from paper_1809_03927_b200 and shares no code with the CUDA path.
"""
import ctypes as C
import numpy as np

from . import build as _build

# ---- plain-C struct mirrors (orc.h) ----
GRID_DT = np.dtype([("nx", "i4"), ("ny", "i4"), ("nz", "i4"), ("hx", "f4"), ("hy", "f4"), ("hz", "f4"),
                    ("ox", "f4"), ("oy", "f4"), ("oz", "f4")])
FIELD_DT = np.dtype([("dir", "f4", 3), ("eu", "f4", 3), ("ev", "f4", 3), ("ref", "f4", 3), ("start_phase", "i4")])
SPOT_DT = np.dtype([("field", "i4"), ("layer", "i4"), ("x_mm", "f4"), ("y_mm", "f4"), ("energy_mev", "f4"),
                    ("sigma_mm", "f4"), ("weight", "f4")])
SEG_DT = np.dtype([("field", "i4"), ("phase", "i4"), ("spot", "i4"), ("pad", "i4"), ("protons", "i8"),
                   ("first_history", "i8"), ("n_hist", "i8"), ("weight", "f8")])
DELIV_DT = np.dtype([("n_phases", "i4"), ("period_ns", "i8"), ("protons_per_weight", "i8"), ("protons_per_s", "i8"),
                     ("ns_per_um", "i4"), ("layer_switch_ns", "i8"), ("repaints", "i4"), ("gate_mask", "u4")],
                    align=True)
MCSTAT_DT = np.dtype([("histories", "u8"), ("steps", "u8"), ("q_incident", "i8"), ("q_deposited", "i8"),
                      ("q_escaped", "i8"), ("fixed_shift", "i4"), ("pad", "i4")])
ACCSTAT_DT = np.dtype([("subvoxels", "u8"), ("dropped_outside_ref", "u8"), ("dropped_outside_dvf", "u8")])

NO_MCS, NO_STRAGGLE, NO_ESPREAD, NO_SPOTSIZE = 1, 2, 4, 8

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.orc_bethe_S.restype = C.c_double
        _lib.orc_bethe_S.argtypes = [C.c_double]
        _lib.orc_range_water.restype = C.c_double
        _lib.orc_range_water.argtypes = [C.c_double]
        _lib.orc_bohr_var_per_t.restype = C.c_double
        _lib.orc_bohr_var_per_t.argtypes = [C.c_double]
        _lib.orc_theta0_sq_per_t.restype = C.c_double
        _lib.orc_theta0_sq_per_t.argtypes = [C.c_double]
        _lib.orc_simulate_delivery.restype = C.c_int64
        _lib.orc_fixed_shift.restype = C.c_int32
        _lib.orc_simulate_delivery_ext.restype = C.c_int64
        _lib.orc_transport.restype = C.c_int
        _lib.orc_finalize_dose.restype = None
        _lib.orc_hu_to_density.restype = C.c_int
        _lib.orc_emtm_push.restype = C.c_int
        _lib.orc_emtm_finalize.restype = C.c_int
        _lib.orc_dim_pull.restype = C.c_int
        _lib.orc_dim_finalize.restype = C.c_int
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def make_grid(shape_zyx, h_xyz, o_xyz=(0.0, 0.0, 0.0)):
    g = np.zeros(1, GRID_DT)
    g["nz"], g["ny"], g["nx"] = shape_zyx
    g["hx"], g["hy"], g["hz"] = h_xyz
    g["ox"], g["oy"], g["oz"] = o_xyz
    return g


def grid_shape(g):
    return int(g["nz"][0]), int(g["ny"][0]), int(g["nx"][0])


def philox4x32_10(ctr, key):
    c = np.asarray(ctr, np.uint32).copy()
    k = np.asarray(key, np.uint32).copy()
    o = np.zeros(4, np.uint32)
    lib().orc_philox4x32_10(_p(c), _p(k), _p(o))
    return o


def bethe_S(E):
    return lib().orc_bethe_S(float(E))


def range_water(E):
    return lib().orc_range_water(float(E))


def bohr_var_per_t(E):
    return lib().orc_bohr_var_per_t(float(E))


def theta0_sq_per_t(E):
    return lib().orc_theta0_sq_per_t(float(E))


def simulate_delivery(fields, spots, prm, total_histories):
    """D1-D7.  Returns (segments[SEG_DT], total_time_ns[n_fields], dropped_protons)."""
    fields = np.ascontiguousarray(fields, FIELD_DT)
    spots = np.ascontiguousarray(spots, SPOT_DT)
    prm = np.ascontiguousarray(prm, DELIV_DT)
    L = lib()
    args = [C.c_int32(len(fields)), _p(fields), C.c_int64(len(spots)), _p(spots), _p(prm),
            C.c_uint64(int(total_histories))]
    n = L.orc_simulate_delivery(*args, None, C.c_int64(0), None, None)
    if n < 0:
        raise ValueError(f"orc_simulate_delivery: error {n}")
    segs = np.zeros(n, SEG_DT)
    tt = np.zeros(len(fields), np.int64)
    dropped = np.zeros(1, np.int64)
    n2 = L.orc_simulate_delivery(*args, _p(segs), C.c_int64(n), _p(tt), _p(dropped))
    assert n2 == n
    return segs, tt, int(dropped[0])


def fixed_shift(segs, spots):
    segs = np.ascontiguousarray(segs, SEG_DT)
    spots = np.ascontiguousarray(spots, SPOT_DT)
    return int(lib().orc_fixed_shift(C.c_int64(len(segs)), _p(segs), _p(spots)))


def threads():
    """threads the oracle's history loop runs on (OpenMP)"""
    return int(lib().orc_threads())


def transport(grid, rho, fields, spots, segs, seed, shift, flags=0, probe_faces=None, trace=None):
    """T1-T12 over the given segments.  Returns (Q int64 [z,y,x], stats record, probe_xy or None, stop_xyz or None).
    trace = (hist_base, hist_count) enables stop_xyz (and probe_xy when probe_faces is given)."""
    rho = np.ascontiguousarray(rho, np.float32)
    fields = np.ascontiguousarray(fields, FIELD_DT)
    spots = np.ascontiguousarray(spots, SPOT_DT)
    segs = np.ascontiguousarray(segs, SEG_DT)
    Q = np.zeros(grid_shape(grid), np.int64)
    st = np.zeros(1, MCSTAT_DT)
    pf = pxy = sxyz = None
    base = cnt = 0
    if trace is not None:
        base, cnt = int(trace[0]), int(trace[1])
        sxyz = np.full((cnt, 3), np.nan)
        if probe_faces is not None:
            pf = np.ascontiguousarray(probe_faces, np.int32)
            pxy = np.full((len(pf), cnt, 2), np.nan)
    rc = lib().orc_transport(_p(grid), _p(rho), C.c_int32(len(fields)), _p(fields), _p(spots),
                             C.c_int64(len(segs)), _p(segs), C.c_uint64(int(seed)), C.c_int32(int(shift)),
                             C.c_uint32(int(flags)), _p(Q), _p(st),
                             C.c_int32(0 if pf is None else len(pf)), _p(pf), C.c_int64(base), C.c_int64(cnt),
                             _p(pxy), _p(sxyz))
    if rc != 0:
        raise ValueError(f"orc_transport: error {rc}")
    return Q, st[0], pxy, sxyz


def finalize_dose(grid, rho, Q, shift, per_protons=0.0):
    rho = np.ascontiguousarray(rho, np.float32)
    Q = np.ascontiguousarray(Q, np.int64)
    out = np.zeros(grid_shape(grid), np.float32)
    lib().orc_finalize_dose(_p(grid), _p(rho), _p(Q), C.c_int32(int(shift)), C.c_double(float(per_protons)), _p(out))
    return out


def hu_to_density(ct_grid, hu, dose_grid=None, hu_pts=(-1000.0, 0.0, 1000.0), rho_pts=(0.001, 1.0, 1.6)):
    hu = np.ascontiguousarray(hu, np.int16)
    hp = np.asarray(hu_pts, np.float32)
    rp = np.asarray(rho_pts, np.float32)
    out = np.zeros(grid_shape(ct_grid if dose_grid is None else dose_grid), np.float32)
    rc = lib().orc_hu_to_density(_p(ct_grid), _p(hu), _p(dose_grid), C.c_int32(len(hp)), _p(hp), _p(rp), _p(out))
    if rc != 0:
        raise ValueError(f"orc_hu_to_density: error {rc}")
    return out


def emtm_push(src_grid, dose, rho, dvf_grid, disp, ref_grid, ns_xyz):
    """A1-A5 for one source phase.  Returns (E, M int64 on ref grid, stats record)."""
    dose = np.ascontiguousarray(dose, np.float32)
    rho = np.ascontiguousarray(rho, np.float32)
    disp = np.ascontiguousarray(disp, np.float32)
    E = np.zeros(grid_shape(ref_grid), np.int64)
    M = np.zeros(grid_shape(ref_grid), np.int64)
    st = np.zeros(1, ACCSTAT_DT)
    rc = lib().orc_emtm_push(_p(src_grid), _p(dose), _p(rho), _p(dvf_grid), _p(disp), _p(ref_grid),
                             C.c_int32(ns_xyz[0]), C.c_int32(ns_xyz[1]), C.c_int32(ns_xyz[2]), _p(E), _p(M), _p(st))
    if rc != 0:
        raise ValueError(f"orc_emtm_push: error {rc}")
    return E, M, st[0]


def emtm_finalize(ref_grid, dose_ref, E_list, M_list, dvf_grids):
    """A6.  E_list/M_list: per source phase int64 grids in ascending phase order."""
    dose_ref = np.ascontiguousarray(dose_ref, np.float32)
    n = len(E_list)
    E = np.ascontiguousarray(np.stack(E_list), np.int64) if n else None
    M = np.ascontiguousarray(np.stack(M_list), np.int64) if n else None
    dg = np.ascontiguousarray(np.concatenate(dvf_grids), GRID_DT) if n else None
    out = np.zeros(grid_shape(ref_grid), np.float32)
    rc = lib().orc_emtm_finalize(_p(ref_grid), _p(dose_ref), C.c_int32(n), _p(E), _p(M), _p(dg), _p(out))
    if rc != 0:
        raise ValueError(f"orc_emtm_finalize: error {rc}")
    return out


def accumulate_subvoxel(grid, doses, rhos, disps, dvf_grids, ref_phase, ns_xyz):
    """Whole a8+a9 path: doses/rhos lists per phase, disps[p] S->R displacement (None for the reference)."""
    Es, Ms, dgs = [], [], []
    stats = np.zeros(1, ACCSTAT_DT)[0]
    for p in range(len(doses)):
        if p == ref_phase or disps[p] is None:
            continue
        E, M, st = emtm_push(grid, doses[p], rhos[p], dvf_grids[p], disps[p], grid, ns_xyz)
        Es.append(E); Ms.append(M); dgs.append(dvf_grids[p])
        for k in ACCSTAT_DT.names:
            stats[k] += st[k]
    return emtm_finalize(grid, doses[ref_phase], Es, Ms, dgs), stats


def dim_pull(ref_grid, ns_xyz, dvf_grid, disp, src_grid, dose_src):
    """P1-P5 (Eq. 3) for one source phase.  disp = T^{R->S} on dvf_grid (reference frame).
    Returns (D_i^S float64 on the reference grid, stats record)."""
    disp = np.ascontiguousarray(disp, np.float32)
    dose_src = np.ascontiguousarray(dose_src, np.float32)
    out = np.zeros(grid_shape(ref_grid), np.float64)
    st = np.zeros(1, ACCSTAT_DT)
    rc = lib().orc_dim_pull(_p(ref_grid), C.c_int32(ns_xyz[0]), C.c_int32(ns_xyz[1]), C.c_int32(ns_xyz[2]),
                            _p(dvf_grid), _p(disp), _p(src_grid), _p(dose_src), _p(out), _p(st))
    if rc != 0:
        raise ValueError(f"orc_dim_pull: error {rc}")
    return out, st[0]


def accumulate_dim(grid, doses, disps_pull, dvf_grids, ref_phase, ns_xyz):
    """Whole DIM path: doses per phase on `grid`; disps_pull[p] = T^{R->S_p} displacement (None: phase not pulled)."""
    pulled, dgs = [], []
    stats = np.zeros(1, ACCSTAT_DT)[0]
    for p in range(len(doses)):
        if p == ref_phase or disps_pull[p] is None:
            continue
        d, st = dim_pull(grid, ns_xyz, dvf_grids[p], disps_pull[p], grid, doses[p])
        pulled.append(d); dgs.append(dvf_grids[p])
        for k in ACCSTAT_DT.names:
            stats[k] += st[k]
    n = len(pulled)
    P = np.ascontiguousarray(np.stack(pulled), np.float64) if n else None
    dg = np.ascontiguousarray(np.concatenate(dgs), GRID_DT) if n else None
    out = np.zeros(grid_shape(grid), np.float32)
    rc = lib().orc_dim_finalize(_p(grid), _p(np.ascontiguousarray(doses[ref_phase], np.float32)), C.c_int32(n), _p(P),
                                _p(dg), _p(out))
    if rc != 0:
        raise ValueError(f"orc_dim_finalize: error {rc}")
    return out, stats


class DeliveryExt(C.Structure):
    """orc_delivery_ext (orc.h): extended delivery model, all zero / None = base model"""
    _fields_ = [("n_cycles", C.c_int32), ("cycle_period_ns", C.c_void_p), ("discard_ns", C.c_int64),
                ("spill_protons_max", C.c_int64), ("flat_top_ns", C.c_int64), ("spot_switch_fixed_ns", C.c_int64),
                ("n_layer_switch", C.c_int32), ("layer_switch_ns", C.c_void_p), ("max_protons_per_paint", C.c_int64)]


def simulate_delivery_ext(fields, spots, prm, total_histories, cycle_period_ns=None, discard_ns=0, spill_protons_max=0,
                          flat_top_ns=0, spot_switch_fixed_ns=0, layer_switch_ns=None, max_protons_per_paint=0):
    """E1-E5 + D6-D7.  Returns (segments, per-field end time [ns], dropped protons, synchrotron fills)."""
    f = np.ascontiguousarray(fields, FIELD_DT); s = np.ascontiguousarray(spots, SPOT_DT)
    p = np.ascontiguousarray(prm, DELIV_DT)
    cyc = None if cycle_period_ns is None else np.ascontiguousarray(cycle_period_ns, np.int64)
    lsw = None if layer_switch_ns is None else np.ascontiguousarray(layer_switch_ns, np.int64)
    x = DeliveryExt(0 if cyc is None else len(cyc), None if cyc is None else cyc.ctypes.data, int(discard_ns),
                    int(spill_protons_max), int(flat_top_ns), int(spot_switch_fixed_ns),
                    0 if lsw is None else len(lsw), None if lsw is None else lsw.ctypes.data, int(max_protons_per_paint))
    args = [C.c_int32(len(f)), _p(f), C.c_int64(len(s)), _p(s), _p(p), C.byref(x), C.c_uint64(int(total_histories))]
    n = lib().orc_simulate_delivery_ext(*args, None, C.c_int64(0), None, None, None)
    if n < 0:
        raise ValueError(f"orc_simulate_delivery_ext: error {n}")
    segs = np.zeros(n, SEG_DT); tt = np.zeros(len(f), np.int64)
    dropped = C.c_int64(0); fills = C.c_int64(0)
    n2 = lib().orc_simulate_delivery_ext(*args, _p(segs), C.c_int64(n), _p(tt), C.byref(dropped), C.byref(fills))
    assert n2 == n
    return segs, tt, int(dropped.value), int(fills.value)


DICOM_DVF_DT = np.dtype([("nx", "i4"), ("ny", "i4"), ("nz", "i4"), ("pad", "i4"), ("start", "f8", 3), ("delta", "f8", 3),
                         ("row_cos", "f8", 3), ("col_cos", "f8", 3), ("pre", "f8", 16), ("post", "f8", 16)])


def build_dvf(info, delta):
    """Eq. 7-8: info = DICOM_DVF_DT record, delta [3, nz, ny, nx] fp32 -> (r_f, r_f - r_0) fp32"""
    info = np.ascontiguousarray(info, DICOM_DVF_DT)
    delta = np.ascontiguousarray(delta, np.float32)
    rf = np.zeros_like(delta); disp = np.zeros_like(delta)
    lib().orc_build_dvf.restype = C.c_int
    rc = lib().orc_build_dvf(_p(info), _p(delta), _p(rf), _p(disp))
    if rc != 0:
        raise ValueError(f"orc_build_dvf: error {rc}")
    return rf, disp


class TrialSpec(C.Structure):
    """orc_trial_spec (orc.h): distributions of the uncertainty trials, PAPER.md:53-65"""
    _fields_ = [("seed", C.c_uint64), ("n_trials", C.c_int32), ("n_cycles", C.c_int32), ("period_lo_ns", C.c_int64),
                ("period_hi_ns", C.c_int64), ("period_step_ns", C.c_int64), ("period_sigma_ns", C.c_int64),
                ("discard_sigma_ns", C.c_int64), ("flat_top_sigma_ns", C.c_int64), ("spot_switch_sigma_ns", C.c_int64),
                ("layer_switch_sigma_ns", C.c_int64), ("spill_protons_sigma", C.c_int64),
                ("protons_per_s_sigma", C.c_int64)]


def sample_trial(spec, trial, n_fields, prm, cycle_period_ns=None, discard_ns=0, spill_protons_max=0, flat_top_ns=0,
                 spot_switch_fixed_ns=0, layer_switch_ns=None, max_protons_per_paint=0):
    """U0-U5 for one trial.  spec: dict of TrialSpec fields.  Returns dict(start_phase, prm (DELIV_DT record), ext
    (keyword arguments for simulate_delivery_ext))."""
    sp = TrialSpec(**spec)
    p = np.ascontiguousarray(prm, DELIV_DT)
    lsw = None if layer_switch_ns is None else np.ascontiguousarray(layer_switch_ns, np.int64)
    x = DeliveryExt(0, None, int(discard_ns), int(spill_protons_max), int(flat_top_ns), int(spot_switch_fixed_ns),
                    0 if lsw is None else len(lsw), None if lsw is None else lsw.ctypes.data, int(max_protons_per_paint))
    start = np.zeros(n_fields, np.int32)
    cyc = np.zeros(max(sp.n_cycles, 1), np.int64)
    lsw_out = np.zeros(max(1, 0 if lsw is None else len(lsw)), np.int64)
    p_out = np.zeros(1, DELIV_DT)
    x_out = DeliveryExt()
    lib().orc_sample_trial.restype = C.c_int
    rc = lib().orc_sample_trial(C.byref(sp), C.c_int32(trial), C.c_int32(n_fields), _p(p), C.byref(x), _p(start), _p(cyc),
                                _p(lsw_out), _p(p_out), C.byref(x_out))
    if rc != 0:
        raise ValueError(f"orc_sample_trial: error {rc}")
    ext = dict(cycle_period_ns=cyc[:sp.n_cycles].copy() if sp.n_cycles > 0 else None, discard_ns=x_out.discard_ns,
               spill_protons_max=x_out.spill_protons_max, flat_top_ns=x_out.flat_top_ns,
               spot_switch_fixed_ns=x_out.spot_switch_fixed_ns,
               layer_switch_ns=None if lsw is None else lsw_out[:len(lsw)].copy(),
               max_protons_per_paint=x_out.max_protons_per_paint)
    return dict(start_phase=start, prm=p_out, ext=ext)
