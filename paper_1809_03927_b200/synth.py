"""Seeded synthetic inputs for the pbs4d hot path (shared by the CUDA path's tests/bench and the oracle's tests).

This module holds NO arithmetic of the method (no transport, delivery or accumulation step): it only builds input
arrays -- phantoms (HU), plans (fields/spots), delivery parameters, dose blobs and displacement fields -- with
numpy.random.default_rng(seed).  The recipes are those of SURVEY.md 8(d), which make BASELINE.json's five configs
concrete; they stand in for the paper's three private patient cases (Table I).
Struct dtypes mirror include/pbs4d.h (layout only).
"""
import numpy as np

GRID_DT = np.dtype([("nx", "i4"), ("ny", "i4"), ("nz", "i4"), ("hx", "f4"), ("hy", "f4"), ("hz", "f4"),
                    ("ox", "f4"), ("oy", "f4"), ("oz", "f4")])
FIELD_DT = np.dtype([("dir", "f4", 3), ("eu", "f4", 3), ("ev", "f4", 3), ("ref", "f4", 3), ("start_phase", "i4")])
SPOT_DT = np.dtype([("field", "i4"), ("layer", "i4"), ("x_mm", "f4"), ("y_mm", "f4"), ("energy_mev", "f4"),
                    ("sigma_mm", "f4"), ("weight", "f4")])
DELIV_DT = np.dtype([("n_phases", "i4"), ("period_ns", "i8"), ("protons_per_weight", "i8"), ("protons_per_s", "i8"),
                     ("ns_per_um", "i4"), ("layer_switch_ns", "i8"), ("repaints", "i4"), ("gate_mask", "u4")],
                    align=True)

HU_PTS = np.array([-1000.0, 0.0, 1000.0], np.float32)     # BASELINE.json config 2
RHO_PTS = np.array([0.001, 1.0, 1.6], np.float32)


def make_grid(shape_zyx, h_xyz, o_xyz=(0.0, 0.0, 0.0)):
    g = np.zeros(1, GRID_DT)
    g["nz"], g["ny"], g["nx"] = shape_zyx
    g["hx"], g["hy"], g["hz"] = h_xyz
    g["ox"], g["oy"], g["oz"] = o_xyz
    return g


def grid_shape(g):
    return int(g["nz"][0]), int(g["ny"][0]), int(g["nx"][0])


def centres(g):
    """voxel-centre coordinate vectors (x, y, z) in mm, float64"""
    nz, ny, nx = grid_shape(g)
    x = float(g["ox"][0]) + (np.arange(nx) + 0.5) * float(g["hx"][0])
    y = float(g["oy"][0]) + (np.arange(ny) + 0.5) * float(g["hy"][0])
    z = float(g["oz"][0]) + (np.arange(nz) + 0.5) * float(g["hz"][0])
    return x, y, z


def make_field(direction, eu, ev, ref, start_phase=0):
    f = np.zeros(1, FIELD_DT)
    f["dir"], f["eu"], f["ev"], f["ref"], f["start_phase"] = direction, eu, ev, ref, start_phase
    return f


def make_delivery(n_phases=1, period_s=4.0, protons_per_weight=10**7, protons_per_s=10**9, ns_per_um=100,
                  layer_switch_s=1.0, repaints=1, gate_mask=None):
    d = np.zeros(1, DELIV_DT)
    d["n_phases"] = n_phases
    d["period_ns"] = int(round(period_s * 1e9))
    d["protons_per_weight"] = protons_per_weight
    d["protons_per_s"] = protons_per_s
    d["ns_per_um"] = ns_per_um
    d["layer_switch_ns"] = int(round(layer_switch_s * 1e9))
    d["repaints"] = repaints
    d["gate_mask"] = (1 << n_phases) - 1 if gate_mask is None else gate_mask
    return d


def disc_lattice(radius_mm, pitch_mm=5.0):
    """lattice points inside a disc, row-serpentine order -> (n,2) float array"""
    m = int(np.floor(radius_mm / pitch_mm))
    pts = []
    for r, j in enumerate(range(-m, m + 1)):
        row = [(i * pitch_mm, j * pitch_mm) for i in range(-m, m + 1)
               if (i * pitch_mm) ** 2 + (j * pitch_mm) ** 2 <= radius_mm ** 2 + 1e-9]
        if r % 2:
            row.reverse()
        pts.extend(row)
    return np.array(pts, np.float64)


# --------------------------------------------------------------------------------------------------------------
# config 1 (BASELINE.json:7): water cube, one pencil beam; "1b" = energy 100 MeV so the Bragg peak is inside
# --------------------------------------------------------------------------------------------------------------
def config1(energy_mev=150.0, n_hist=100_000, n=50, h=2.0, sigma_mm=5.0, seed=1):
    g = make_grid((n, n, n), (h, h, h))
    hu = np.zeros((1, n, n, n), np.int16)
    c = 0.5 * n * h
    fields = make_field((0, 0, 1), (1, 0, 0), (0, 1, 0), (c, c, 0.0))
    spots = np.zeros(1, SPOT_DT)
    spots[0] = (0, 0, 0.0, 0.0, energy_mev, sigma_mm, 1.0)
    deliv = make_delivery(n_phases=1, protons_per_weight=n_hist)      # weight 1 -> n_hist protons, w = 1
    return dict(name="config1", ct_grid=g, dose_grid=None, hu=hu, fields=fields, spots=spots, deliv=deliv,
                histories=n_hist, seed=seed, per_proton=True)


# --------------------------------------------------------------------------------------------------------------
# config 2 (BASELINE.json:8): slab phantom, 3 layers x 9x9 spots; "2b" = energies (90,100,110)
# --------------------------------------------------------------------------------------------------------------
def config2(energies=(120.0, 135.0, 150.0), n_hist=1_000_000, n=64, h=2.0, seed=2):
    rng = np.random.default_rng(seed)
    g = make_grid((n, n, n), (h, h, h))
    _, _, z = centres(g)
    hu = np.zeros((n, n, n), np.float64)
    lung = (z >= 40.0) & (z < 80.0)
    hu[lung] = rng.uniform(-850.0, -750.0, size=(int(lung.sum()), n, n))
    hu[(z >= 80.0) & (z < 90.0)] = 700.0
    hu = np.rint(hu).astype(np.int16)[None]
    c = 0.5 * n * h
    fields = make_field((0, 0, 1), (1, 0, 0), (0, 1, 0), (c, c, 0.0))
    spots = []
    for li, e in enumerate(energies):
        for j in range(9):
            xs = range(9) if j % 2 == 0 else range(8, -1, -1)
            for i in xs:
                spots.append((0, li, (i - 4) * 5.0, (j - 4) * 5.0, e, 4.0, 1.0))
    spots = np.array(spots, SPOT_DT)
    ppw = max(1, n_hist // len(spots))
    deliv = make_delivery(n_phases=1, protons_per_weight=ppw)
    return dict(name="config2", ct_grid=g, dose_grid=None, hu=hu, fields=fields, spots=spots, deliv=deliv,
                histories=n_hist, seed=seed, per_proton=False)


# --------------------------------------------------------------------------------------------------------------
# 4DCT phantoms (configs 3 and 5): tumour sphere moving SI as A cos^4(pi k / N); analytic DVF decaying with distance
# --------------------------------------------------------------------------------------------------------------
def _tumour_offsets(n_phases, amplitude_mm):
    k = np.arange(n_phases)
    return amplitude_mm * np.cos(np.pi * k / n_phases) ** 4


def _analytic_dvf(grid, centre_k, delta_k, r_t, decay_mm=30.0):
    """S->R displacement (source frame): u = (0, 0, -delta_k g(dist)), g = 1 inside the tumour, Gaussian outside."""
    x, y, z = centres(grid)
    dist = np.sqrt((z[:, None, None] - centre_k[2]) ** 2 + (y[None, :, None] - centre_k[1]) ** 2
                   + (x[None, None, :] - centre_k[0]) ** 2)
    gfun = np.where(dist <= r_t, 1.0, np.exp(-((dist - r_t) ** 2) / (2.0 * decay_mm ** 2)))
    u = np.zeros((3,) + grid_shape(grid), np.float32)
    u[2] = (-delta_k * gfun).astype(np.float32)
    return u


def _plan(field_defs, e_lo, e_hi, n_layers, disc_r, sig_lo_e, sig_hi_e, rng):
    """layers highest energy first; 5 mm lattice in a disc, serpentine; sigma linear in energy; weights U(0.5,1.5)"""
    lat = disc_lattice(disc_r)
    energies = np.linspace(e_hi, e_lo, n_layers)
    spots = []
    for f in range(len(field_defs)):
        for li, e in enumerate(energies):
            sig = sig_lo_e + (sig_hi_e - sig_lo_e) * (e - e_lo) / max(e_hi - e_lo, 1e-9)
            w = rng.uniform(0.5, 1.5, size=len(lat))
            for (px, py), wi in zip(lat, w):
                spots.append((f, li, px, py, e, sig, wi))
    return np.array(spots, SPOT_DT)


def config3(div=1, n_hist=10_000_000, n_phases=10, seed=3, e_range=(70.0, 180.0)):
    """Synthetic lung 4DCT (BASELINE.json:9).  div > 1 shrinks every voxel count and length by that factor."""
    rng = np.random.default_rng(seed)
    ct = make_grid((128 // div, 256 // div, 256 // div), (1.0, 1.0, 2.5))
    dg = make_grid((160 // div, 128 // div, 128 // div), (2.0, 2.0, 2.0))
    x, y, z = centres(ct)
    ext = np.array([256.0, 256.0, 320.0]) / div
    cen = 0.5 * ext
    L = 1.0 / div
    base = rng.normal(40.0, 20.0, size=grid_shape(ct))
    lung_noise = rng.uniform(-850.0, -750.0, size=grid_shape(ct))
    lung = np.zeros(grid_shape(ct), bool)
    for sx in (-1.0, 1.0):
        lung |= (((x[None, None, :] - (cen[0] + sx * 65.0 * L)) / (45.0 * L)) ** 2
                 + ((y[None, :, None] - cen[1]) / (70.0 * L)) ** 2
                 + ((z[:, None, None] - cen[2]) / (100.0 * L)) ** 2) <= 1.0
    static = np.where(lung, lung_noise, base)
    r_t = 15.0 * L
    offs = _tumour_offsets(n_phases, 10.0 * L)
    ref_phase = n_phases // 2
    c0 = np.array([cen[0] + 65.0 * L, cen[1], cen[2]])
    hu = np.empty((n_phases,) + grid_shape(ct), np.int16)
    dvf = []
    for k in range(n_phases):
        ck = c0 + np.array([0.0, 0.0, offs[k]])
        tum = ((x[None, None, :] - ck[0]) ** 2 + (y[None, :, None] - ck[1]) ** 2
               + (z[:, None, None] - ck[2]) ** 2) <= r_t ** 2
        hu[k] = np.rint(np.clip(np.where(tum, 40.0, static), -1000, 3000)).astype(np.int16)
        dvf.append(None if k == ref_phase else _analytic_dvf(dg, ck, offs[k] - offs[ref_phase], r_t, 30.0 * L))
    cref = c0 + np.array([0.0, 0.0, offs[ref_phase]])
    fields = make_field((0, 1, 0), (1, 0, 0), (0, 0, 1), cref)
    spots = _plan([0], e_range[0], e_range[1], 20, 35.0 * L, 6.0, 3.0, rng)
    deliv = make_delivery(n_phases=n_phases, period_s=4.0, protons_per_weight=10**7, layer_switch_s=1.0)
    return dict(name="config3", ct_grid=ct, dose_grid=dg, hu=hu, fields=fields, spots=spots, deliv=deliv,
                histories=n_hist, seed=seed, per_proton=False, dvf=dvf, dvf_grid=dg, ref_phase=ref_phase,
                subvox=(2, 2, 2))


def config5(div=1, n_hist=100_000_000, n_phases=10, seed=5, e_range=(90.0, 200.0)):
    """Synthetic liver 4DCT, 3 fields, 4x repainting, gating on phases 3..7 (BASELINE.json:11)."""
    rng = np.random.default_rng(seed)
    ct = make_grid((160 // div, 512 // div, 512 // div), (0.98, 0.98, 2.5))
    x, y, z = centres(ct)
    ext = np.array([512 * 0.98, 512 * 0.98, 400.0]) / div
    cen = 0.5 * ext
    L = 1.0 / div
    shape = grid_shape(ct)
    static = rng.normal(40.0, 20.0, size=shape).astype(np.float32)
    X, Y, Z = x[None, None, :], y[None, :, None], z[:, None, None]
    lc = cen + np.array([-60.0, 0.0, 0.0]) * L
    liver = (((X - lc[0]) / (90.0 * L)) ** 2 + ((Y - lc[1]) / (70.0 * L)) ** 2 + ((Z - lc[2]) / (80.0 * L)) ** 2) <= 1.0
    static = np.where(liver, rng.normal(60.0, 15.0, size=shape).astype(np.float32), static)
    # rib shell segments: elliptical shell, 8 mm thick, 10 mm ribs every 25 mm in z
    rr = np.sqrt(((X - cen[0]) / (200.0 * L)) ** 2 + ((Y - cen[1]) / (150.0 * L)) ** 2)
    ribs = (np.abs(rr - 1.0) <= 0.03) & (np.mod(Z / L, 25.0) < 10.0)
    static = np.where(ribs, np.float32(700.0), static)
    r_t = 25.0 * L
    offs = _tumour_offsets(n_phases, 15.0 * L)
    ref_phase = n_phases // 2
    hu = np.empty((n_phases,) + shape, np.int16)
    dvf = []
    gate = [p for p in range(n_phases) if 3 * n_phases // 10 <= p <= 7 * n_phases // 10]
    for k in range(n_phases):
        ck = lc + np.array([0.0, 0.0, offs[k]])
        tum = ((X - ck[0]) ** 2 + (Y - ck[1]) ** 2 + (Z - ck[2]) ** 2) <= r_t ** 2
        hu[k] = np.rint(np.clip(np.where(tum, np.float32(60.0), static), -1000, 3000)).astype(np.int16)
        dvf.append(_analytic_dvf(ct, ck, offs[k] - offs[ref_phase], r_t, 30.0 * L)
                   if (k in gate and k != ref_phase) else None)
    cref = lc + np.array([0.0, 0.0, offs[ref_phase]])
    fdefs = []
    for ang in (0.0, 45.0, 315.0):
        th = np.deg2rad(ang)
        fdefs.append(make_field((np.sin(th), np.cos(th), 0.0), (np.cos(th), -np.sin(th), 0.0), (0, 0, 1), cref))
    fields = np.concatenate(fdefs)
    spots = _plan(fdefs, e_range[0], e_range[1], 25, 30.0 * L, 6.0, 3.0, rng)
    gm = 0
    for p in gate:
        gm |= 1 << p
    deliv = make_delivery(n_phases=n_phases, period_s=4.5, protons_per_weight=10**7, layer_switch_s=1.0,
                          repaints=4, gate_mask=gm)
    return dict(name="config5", ct_grid=ct, dose_grid=None, hu=hu, fields=fields, spots=spots, deliv=deliv,
                histories=n_hist, seed=seed, per_proton=False, dvf=dvf, dvf_grid=ct, ref_phase=ref_phase,
                subvox=(2, 2, 5), gate_phases=gate)


# --------------------------------------------------------------------------------------------------------------
# config 4 (BASELINE.json:10): accumulation stress -- smooth dose blobs, phantom densities, random smooth DVFs
# --------------------------------------------------------------------------------------------------------------
def config4(n=128, n_phases=10, h=2.0, seed=4, max_disp_mm=20.0, dvf_div=1):
    """Returns doses [P,z,y,x] f32 (peak 2 Gy), rhos [P,z,y,x] f32, disps list ([3,z,y,x] f32 or None for phase 0).
    dvf_div > 1 stores the DVF on a coarser grid (as the paper's Table I deformation grids are)."""
    rng = np.random.default_rng(seed)
    g = make_grid((n, n, n), (h, h, h))
    nd = n // dvf_div
    dg = make_grid((nd, nd, nd), (h * dvf_div,) * 3)
    x, y, z = centres(g)
    ext = n * h
    # densities: config-3-like phantom rebuilt on this grid (tissue ~1.04, lung ellipsoids ~0.2) via the HU table
    hu = rng.normal(40.0, 20.0, size=(n, n, n))
    lung = np.zeros((n, n, n), bool)
    for sx in (-1.0, 1.0):
        lung |= (((x[None, None, :] - ext * (0.5 + sx * 0.25)) / (0.18 * ext)) ** 2
                 + ((y[None, :, None] - 0.5 * ext) / (0.27 * ext)) ** 2
                 + ((z[:, None, None] - 0.5 * ext) / (0.39 * ext)) ** 2) <= 1.0
    hu = np.where(lung, rng.uniform(-850.0, -750.0, size=(n, n, n)), hu)
    rho1 = np.interp(hu, HU_PTS.astype(np.float64), RHO_PTS.astype(np.float64)).astype(np.float32)
    rhos = np.broadcast_to(rho1, (n_phases, n, n, n)).copy()
    doses = np.zeros((n_phases, n, n, n), np.float32)
    disps = []
    xd, yd, zd = centres(dg)
    for p in range(n_phases):
        d = np.zeros((n, n, n), np.float64)
        for _ in range(6):
            c = rng.uniform(0.2 * ext, 0.8 * ext, 3)
            s = rng.uniform(10.0, 30.0) * ext / 256.0
            d += (np.exp(-((z - c[2]) ** 2) / (2 * s * s))[:, None, None]
                  * np.exp(-((y - c[1]) ** 2) / (2 * s * s))[None, :, None]
                  * np.exp(-((x - c[0]) ** 2) / (2 * s * s))[None, None, :])
        doses[p] = (2.0 * d / d.max()).astype(np.float32)
        if p == 0:
            disps.append(None)
            continue
        u = np.zeros((3, nd, nd, nd), np.float64)
        for _ in range(8):
            c = rng.uniform(0.0, ext, 3)
            s = rng.uniform(20.0, 60.0) * ext / 256.0
            amp = rng.normal(0.0, 1.0, 3)
            mode = (np.exp(-((zd - c[2]) ** 2) / (2 * s * s))[:, None, None]
                    * np.exp(-((yd - c[1]) ** 2) / (2 * s * s))[None, :, None]
                    * np.exp(-((xd - c[0]) ** 2) / (2 * s * s))[None, None, :])
            u += amp[:, None, None, None] * mode[None]
        u *= max_disp_mm / np.sqrt((u ** 2).sum(0)).max()
        disps.append(u.astype(np.float32))
    return dict(name="config4", grid=g, dvf_grid=dg, doses=doses, rhos=rhos, disps=disps, ref_phase=0, seed=seed)
