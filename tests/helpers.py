"""Small test-side helpers (pose / frame construction only; no rasteriser arithmetic)."""
from __future__ import annotations

import numpy as np

from workloads.generators import Sensor, _mat_to_quat, _pose, _rot_zyx  # noqa: F401


def make_sensor(H, W, fov_deg=(-22.5, 22.5), T_ws=None, r_min=0.0, r_max=float("inf"), f64_pose=False):
    if T_ws is None:
        T_ws = np.concatenate([np.eye(3), np.zeros((3, 1))], 1)
    T = np.asarray(T_ws, dtype=np.float64 if f64_pose else np.float32).reshape(3, 4)
    s = Sensor(H, W, float(np.deg2rad(fov_deg[0])), float(np.deg2rad(fov_deg[1])), r_min, r_max, T)
    return s


def beam(sensor, j, i):
    """Unit beam of pixel (row j, col i): the grid convention of DESIGN.md reading R1."""
    W, H = sensor.W, sensor.H
    phi = -np.pi + (np.asarray(i) + 0.5) * (2 * np.pi / W)
    em, eM = float(np.float32(sensor.elev_min)), float(np.float32(sensor.elev_max))
    th = eM - (np.asarray(j) + 0.5) * ((eM - em) / H)
    return np.stack([np.cos(th) * np.cos(phi), np.cos(th) * np.sin(phi), np.sin(th) * np.ones_like(phi)], -1)


def frame_quat(n, tu_hint=None):
    """Unit quaternion (w,x,y,z) whose third column is n (first column orthogonal to n near tu_hint)."""
    n = np.asarray(n, dtype=np.float64)
    n = n / np.linalg.norm(n)
    if tu_hint is None:
        tu_hint = np.array([0.0, 0.0, 1.0]) if abs(n[2]) < 0.9 else np.array([1.0, 0.0, 0.0])
    tu = tu_hint - n * (tu_hint @ n)
    tu /= np.linalg.norm(tu)
    tv = np.cross(n, tu)
    R = np.stack([tu, tv, n], 1)
    return _mat_to_quat(R[None])[0], R


def quat_mul(a, b):
    aw, ax, ay, az = a
    bw, bx, by, bz = b
    return np.array([aw * bw - ax * bx - ay * by - az * bz,
                     aw * bx + ax * bw + ay * bz - az * by,
                     aw * by - ax * bz + ay * bw + az * bx,
                     aw * bz + ax * by - ay * bx + az * bw])


def quat_to_mat(q):
    w, x, y, z = q / np.linalg.norm(q)
    return np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - w * z), 2 * (x * z + w * y)],
                     [2 * (x * y + w * z), 1 - 2 * (x * x + z * z), 2 * (y * z - w * x)],
                     [2 * (x * z - w * y), 2 * (y * z + w * x), 1 - 2 * (x * x + y * y)]])
