"""Pins of oracle/scan_image.py.  All CPU (-m "not gpu")."""
from __future__ import annotations

import numpy as np

from oracle import scan_image as si
from helpers import beam, make_sensor


def _grid_points(S, ranges):
    H, W = S.H, S.W
    jj, ii = np.meshgrid(np.arange(H), np.arange(W), indexing="ij")
    d = beam(S, jj, ii)                                          # the renderer's beams (R1), helpers.py
    return (d * ranges[..., None]).reshape(-1, 3).astype(np.float32), jj.ravel(), ii.ravel()


def test_grid_beams_fall_into_their_own_pixels_with_their_ranges():
    """One point on every beam of the rasteriser's grid: the image is exactly those ranges (ties the projection
    to the renderer's (row, column) convention: a swapped axis, sign or half-pixel offset fails)."""
    for H, W, fov in ((8, 32, (-22.5, 22.5)), (16, 64, (-24.8, 2.0))):
        S = make_sensor(H, W, fov)
        rng = np.random.default_rng(0)
        R = rng.uniform(2, 60, (H, W))
        pts, jj, ii = _grid_points(S, R)
        row, col, r32, valid = si.pixel_of(pts, S)
        assert valid.all() and np.array_equal(row, jj) and np.array_equal(col, ii)
        img, nrm, idx = si.scan_to_range_image(pts, None, S)
        expect = np.linalg.norm(pts.astype(np.float64), axis=1).astype(np.float32).reshape(H, W)
        assert np.array_equal(img, expect) and (idx.ravel() == np.arange(H * W)).all() and not nrm.any()
        assert np.abs(img - R).max() < 1e-4


def test_nearest_return_wins_ties_by_index_and_normals_follow():
    S = make_sensor(4, 16)
    d = beam(S, 2, 5)
    pts = np.stack([d * 10.0, d * 4.0, d * 7.0, d * 4.0]).astype(np.float32)      # same pixel; 1 and 3 tie
    nrm = np.eye(4, 3, dtype=np.float32) + 0.5
    img, n, idx = si.scan_to_range_image(pts, nrm, S)
    assert idx[2, 5] == 1 and np.count_nonzero(img) == 1
    assert img[2, 5] == np.float32(np.linalg.norm(pts[1].astype(np.float64)))
    assert np.array_equal(n[:, 2, 5], nrm[1])
    img2, _, idx2 = si.scan_to_range_image(pts[::-1].copy(), None, S)              # order reversed: index 0 now ties with 2
    assert idx2[2, 5] == 0 and img2[2, 5] == img[2, 5]


def test_seam_field_of_view_and_gates():
    S = make_sensor(8, 64, (-20.0, 20.0), r_min=1.0, r_max=50.0)
    eps = 1e-4
    def at(phi, th, r):
        return [r * np.cos(th) * np.cos(phi), r * np.cos(th) * np.sin(phi), r * np.sin(th)]
    pts = np.array([at(np.pi - eps, 0.01, 5.0),          # last column
                    at(-np.pi + eps, 0.01, 6.0),         # first column
                    [-7.0, 0.0, 0.1],                    # y = +0: phi = +pi exactly -> wraps to column 0
                    at(0.3, np.deg2rad(20.5), 5.0),      # above the field of view
                    at(0.3, np.deg2rad(-20.5), 5.0),     # below
                    at(0.3, 0.0, 0.5),                   # inside r_min
                    at(0.3, 0.0, 60.0),                  # beyond r_max
                    [np.nan, 0, 0], [0, 0, 0],           # not finite / zero range
                    at(0.3, np.deg2rad(20.0) - 1e-6, 5.0),    # just inside the top row
                    at(0.3, np.deg2rad(-20.0) + 1e-6, 5.0)],  # just inside the bottom row
                   dtype=np.float32)
    row, col, r32, valid = si.pixel_of(pts, S)
    assert valid.tolist() == [True, True, True, False, False, False, False, False, False, True, True]
    assert col[0] == 63 and col[1] == 0 and col[2] == 0
    assert row[9] == 0 and row[10] == 7
    img, _, idx = si.scan_to_range_image(pts, None, S)
    assert np.count_nonzero(img) == 4 and idx[row[1], 0] == 1      # the 6 m and the 7 m return share column 0: nearest


def test_yaw_by_whole_columns_shifts_the_image():
    S = make_sensor(16, 128)
    rng = np.random.default_rng(4)
    M = 4000
    v = rng.normal(size=(M, 3)); v[:, 2] *= 0.2
    pts = (v / np.linalg.norm(v, axis=1, keepdims=True) * rng.uniform(2, 40, (M, 1)))
    k = 5
    a = k * 2 * np.pi / S.W
    Rz = np.array([[np.cos(a), -np.sin(a), 0], [np.sin(a), np.cos(a), 0], [0, 0, 1]])
    # keep points away from cell borders so that the fp32 rounding of the rotated copy cannot move them
    row, col, r32, valid = si.pixel_of(pts.astype(np.float32), S)
    phi = np.arctan2(pts[:, 1], pts[:, 0]); th = np.arctan2(pts[:, 2], np.hypot(pts[:, 0], pts[:, 1]))
    fx = (phi + np.pi) / (2 * np.pi / S.W) % 1.0
    e_min, e_max = float(np.float32(S.elev_min)), float(np.float32(S.elev_max))
    fy = (e_max - th) / ((e_max - e_min) / S.H) % 1.0
    keep = valid & (np.abs(fx - 0.5) < 0.45) & (np.abs(fy - 0.5) < 0.45)
    p0 = pts[keep].astype(np.float32)
    p1 = (pts[keep] @ Rz.T).astype(np.float32)
    img0, _, idx0 = si.scan_to_range_image(p0, None, S)
    img1, _, idx1 = si.scan_to_range_image(p1, None, S)
    assert np.array_equal(np.roll(idx0, k, axis=1), idx1)
    assert np.allclose(np.roll(img0, k, axis=1), img1, rtol=1e-6)


def test_round_trip_with_the_rasterisers_input_scan():
    """The synthetic scan of the bench workload (ranges on the grid's beams) back-projected to points and re-imaged
    reproduces the scan's valid mask and ranges."""
    from workloads import make_newer_college, simulate_scan
    w = make_newer_college(n_surfels=1000, H=16, W=128)
    S = w.sensors[0]
    tgt, tn = simulate_scan(w.scene, S, w.scan_seed)
    jj, ii = np.meshgrid(np.arange(S.H), np.arange(S.W), indexing="ij")
    pts = (beam(S, jj, ii) * tgt[..., None].astype(np.float64)).reshape(-1, 3).astype(np.float32)
    nrm = tn.reshape(3, -1).T.copy()
    img, n, idx = si.scan_to_range_image(pts, nrm, S)
    assert np.array_equal(img > 0, tgt > 0)
    assert np.allclose(img, tgt, rtol=2e-7, atol=0)
    assert np.array_equal(n[:, tgt > 0], tn[:, tgt > 0])
