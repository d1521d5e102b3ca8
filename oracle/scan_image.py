"""ORACLE -- test infrastructure only (see oracle/__init__.py).

Plain fp64 numpy definition of the step just before the loss stage: building a LiDAR scan
into a spherical range image, "we build each scan as a spherical range image and render the Gaussian map under
the same spherical projection pi_s", with the valid mask M_D = [D > 0] and the image of
the tracker's normals N_g-icp.

Readings (R25-R27; the paper gives no formula): the grid is the renderer's (R1): pixel (j, i) owns the
directions with azimuth in [-pi + i dphi, -pi + (i+1) dphi) and elevation in (theta_max - (j+1) dtheta,
theta_max - j dtheta]; phi = atan2(y, x), theta = atan2(z, hypot(x, y)); azimuth +pi wraps to column 0; points
are given in the SENSOR frame (a deskewed scan); the nearest return of a pixel wins (z-buffer), equal fp32 ranges
break by the lower point index; points that are not finite, have range 0 or outside [r_min, r_max], or fall
outside the elevation field of view are dropped; pixels without a return are 0 (so M_D = [D > 0]).

Parity with the authors' projection is unpinned (the paper prints no value); pinned by tests/test_oracle_scan_image.py.
Nothing here is imported by the CUDA path.
"""
from __future__ import annotations

import numpy as np


def pixel_of(points, sensor):
    """(row, col, range fp32, valid) of every point, in fp64 from the fp32 inputs."""
    p = np.asarray(points, dtype=np.float64).reshape(-1, 3)
    H, W = int(sensor.H), int(sensor.W)
    e_min, e_max = float(np.float32(sensor.elev_min)), float(np.float32(sensor.elev_max))
    dphi = (2.0 * np.pi) / W
    dth = (e_max - e_min) / H
    x, y, z = p[:, 0], p[:, 1], p[:, 2]
    r = np.sqrt(x * x + y * y + z * z)
    r32 = r.astype(np.float32)
    with np.errstate(invalid="ignore"):
        phi = np.arctan2(y, x)
        th = np.arctan2(z, np.sqrt(x * x + y * y))
        col = np.floor((phi + np.pi) / dphi)
        row = np.floor((e_max - th) / dth)
    valid = np.isfinite(r) & (r32 > 0) & (r32 >= np.float32(sensor.r_min)) & (r32 <= np.float32(sensor.r_max))
    valid &= np.isfinite(col) & np.isfinite(row) & (row >= 0) & (row < H)
    col = np.where(valid, col, 0).astype(np.int64)
    col = np.where(col >= W, col - W, col)                       # phi = +pi -> column 0
    row = np.where(valid, row, 0).astype(np.int64)
    return row, col, r32, valid


def scan_to_range_image(points, normals, sensor):
    """Returns (range [H,W] f32, normal [3,H,W] f32, index [H,W] i64 of the winning point or -1)."""
    H, W = int(sensor.H), int(sensor.W)
    row, col, r32, valid = pixel_of(points, sensor)
    rng = np.zeros((H, W), dtype=np.float32)
    idx = np.full((H, W), -1, dtype=np.int64)
    for k in np.nonzero(valid)[0]:                               # plain z-buffer loop, point by point
        j, i = row[k], col[k]
        if idx[j, i] < 0 or r32[k] < rng[j, i]:                  # (equal range: the earlier, lower index stays)
            rng[j, i] = r32[k]
            idx[j, i] = k
    nrm = np.zeros((3, H, W), dtype=np.float32)
    if normals is not None:
        n = np.asarray(normals, dtype=np.float32).reshape(-1, 3)
        hit = idx >= 0
        nrm[:, hit] = n[idx[hit]].T
    return rng, nrm, idx
