"""Pins of the DVF-construction oracle (oracle/orc_dvf.c; Eq. 7-8): numpy's 4x4 matrix algebra in
float64 (a library routine evaluating the same two equations), the identity special case of the paper ("for DIR
between 4DCT phases, these are both the 4 x 4 identity matrix") and rigid-motion invariants.  CPU only."""
import numpy as np

import oracle as orc


def info(shape, start, delta, U=(1, 0, 0), V=(0, 1, 0), pre=None, post=None):
    r = np.zeros(1, orc.DICOM_DVF_DT)
    r["nz"], r["ny"], r["nx"] = shape
    r["start"], r["delta"], r["row_cos"], r["col_cos"] = start, delta, U, V
    r["pre"] = (np.eye(4) if pre is None else pre).ravel()
    r["post"] = (np.eye(4) if post is None else post).ravel()
    return r


def rigid(rng):
    q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
    if np.linalg.det(q) < 0:
        q[:, 0] = -q[:, 0]
    M = np.eye(4); M[:3, :3] = q; M[:3, 3] = rng.uniform(-30, 30, 3)
    return M


def numpy_reference(r, delta):
    nz, ny, nx = int(r["nz"][0]), int(r["ny"][0]), int(r["nx"][0])
    U, V = r["row_cos"][0], r["col_cos"][0]; W = np.cross(U, V)
    A = np.zeros((4, 4)); A[:3, 0] = U * r["delta"][0][0]; A[:3, 1] = V * r["delta"][0][1]
    A[:3, 2] = W * r["delta"][0][2]; A[:3, 3] = r["start"][0]; A[3, 3] = 1.0            # Eq. 8 as a 4x4 matrix
    k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    idx = np.stack([i, j, k, np.ones_like(i)]).reshape(4, -1).astype(np.float64)
    r0 = A @ idx
    d = np.concatenate([delta.reshape(3, -1).astype(np.float64), np.zeros((1, idx.shape[1]))])
    rf = r["post"][0].reshape(4, 4) @ (r["pre"][0].reshape(4, 4) @ r0 + d)               # Eq. 7
    return r0[:3].reshape(3, nz, ny, nx), rf[:3].reshape(3, nz, ny, nx)


def test_matches_numpy_matrix_algebra_on_an_oblique_grid_with_rigid_pre_and_post():
    rng = np.random.default_rng(31)
    q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
    r = info((5, 6, 7), (-100.5, 20.25, 3.0), (2.5, 2.55, 3.0), U=q[:, 0], V=q[:, 1], pre=rigid(rng), post=rigid(rng))
    delta = rng.uniform(-8, 8, size=(3, 5, 6, 7)).astype(np.float32)
    rf, disp = orc.build_dvf(r, delta)
    r0_np, rf_np = numpy_reference(r, delta)
    assert np.abs(rf - rf_np).max() < 2e-5                                              # fp32 output of |r| ~ 150 mm
    assert np.abs(disp - (rf_np - r0_np)).max() < 2e-5
    # the rigid post transformation preserves distances between the points M_Pre r_0 + Delta
    pre = r["pre"][0].reshape(4, 4)
    a = (pre[:3, :3] @ r0_np.reshape(3, -1) + pre[:3, 3:4]) + delta.reshape(3, -1); b = rf.reshape(3, -1).astype(np.float64)
    assert abs(np.linalg.norm(a[:, 0] - a[:, -1]) - np.linalg.norm(b[:, 0] - b[:, -1])) < 1e-4


def test_identity_matrices_and_axis_aligned_cosines_give_the_stored_translations():
    rng = np.random.default_rng(32)
    r = info((4, 5, 6), (1.0, -2.0, 3.5), (2.0, 2.5, 3.0))
    delta = rng.uniform(-5, 5, size=(3, 4, 5, 6)).astype(np.float32)
    rf, disp = orc.build_dvf(r, delta)
    k, j, i = np.meshgrid(np.arange(4), np.arange(5), np.arange(6), indexing="ij")
    r0 = np.stack([1.0 + 2.0 * i, -2.0 + 2.5 * j, 3.5 + 3.0 * k])
    assert np.abs(disp - delta).max() < 1e-6 and (rf == (r0 + delta.astype(np.float64)).astype(np.float32)).all()
    # zero translation: r_f = r_0 exactly, displacement exactly 0
    rf0, d0 = orc.build_dvf(r, np.zeros_like(delta))
    assert (d0 == 0).all() and (rf0 == r0.astype(np.float32)).all()


def test_pure_translation_post_matrix_and_flipped_axes():
    rng = np.random.default_rng(33)
    post = np.eye(4); post[:3, 3] = (10.0, -4.0, 0.5)
    r = info((3, 4, 5), (0.0, 0.0, 0.0), (1.0, 1.0, 2.0), U=(0, -1, 0), V=(1, 0, 0), post=post)   # W = U x V = (0,0,1)
    delta = rng.uniform(-1, 1, size=(3, 3, 4, 5)).astype(np.float32)
    rf, disp = orc.build_dvf(r, delta)
    k, j, i = np.meshgrid(np.arange(3), np.arange(4), np.arange(5), indexing="ij")
    r0 = np.stack([1.0 * j, -1.0 * i, 2.0 * k]).astype(np.float64)
    want = r0 + delta + np.array([10.0, -4.0, 0.5])[:, None, None, None]
    assert np.abs(rf - want).max() < 1e-5 and np.abs(disp - (want - r0)).max() < 1e-5
