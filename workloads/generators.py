"""Seeded synthetic workloads shaped like the paper's maps and scans.

Stand-ins for Newer College / KITTI / Oxford Spires, which are
not available: only the sensors' image shapes (64x1024, 64x2048, 128x2048), the
paper's map sizes and the range-proportional scale law
of Eq. 6 are reproduced.  numpy `default_rng(seed)` (PCG64),
fp32 outputs.  No rasteriser arithmetic lives here: the only geometry is the
scan simulator (ray / plane and ray / box intersection of the synthetic scene),
i.e. the production of the *input* range image D and normal image N_g-icp.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Optional

import numpy as np

# ----------------------------------------------------------------------------
# containers
# ----------------------------------------------------------------------------


@dataclass
class Sensor:
    """Spherical LiDAR image grid + rigid pose (sensor -> world)."""

    H: int
    W: int
    elev_min: float  # radians
    elev_max: float  # radians; row 0 is at elev_max
    r_min: float
    r_max: float
    T_ws: np.ndarray  # (3, 4) float32, p_world = R p_sensor + t

    def with_pose(self, T_ws: np.ndarray) -> "Sensor":
        return Sensor(self.H, self.W, self.elev_min, self.elev_max, self.r_min, self.r_max,
                      np.asarray(T_ws, dtype=np.float32).reshape(3, 4))


@dataclass
class Workload:
    name: str
    mean: np.ndarray      # (N, 3) float32, world
    quat: np.ndarray      # (N, 4) float32, (w, x, y, z), not necessarily unit
    scale: np.ndarray     # (N, 2) float32, metres
    opacity: np.ndarray   # (N,)  float32 in [0, 1]
    sensors: List[Sensor]
    scene: Optional[dict] = None            # for simulate_scan
    perturbed_mean: Optional[np.ndarray] = None  # tiny: target = render of these
    keep_masks: Optional[List[np.ndarray]] = None  # per frame (H, W) uint8, 0 = drop pixel
    lambdas: dict = field(default_factory=lambda: dict(lambda_n=1.0, lambda_ng=0.05, lambda_ns=0.01))
    scan_seed: int = 0

    @property
    def N(self) -> int:
        return int(self.mean.shape[0])


# ----------------------------------------------------------------------------
# small helpers (pose / frame construction: input generation only)
# ----------------------------------------------------------------------------

def _rot_zyx(yaw: float, pitch: float, roll: float) -> np.ndarray:
    cy, sy = np.cos(yaw), np.sin(yaw)
    cp, sp = np.cos(pitch), np.sin(pitch)
    cr, sr = np.cos(roll), np.sin(roll)
    Rz = np.array([[cy, -sy, 0], [sy, cy, 0], [0, 0, 1.0]])
    Ry = np.array([[cp, 0, sp], [0, 1, 0], [-sp, 0, cp]])
    Rx = np.array([[1, 0, 0], [0, cr, -sr], [0, sr, cr]])
    return Rz @ Ry @ Rx


def _pose(R: np.ndarray, t) -> np.ndarray:
    T = np.zeros((3, 4), dtype=np.float32)
    T[:, :3] = R.astype(np.float32)
    T[:, 3] = np.asarray(t, dtype=np.float32)
    return T


def _mat_to_quat(R: np.ndarray) -> np.ndarray:
    """(M, 3, 3) proper rotations -> (M, 4) unit quaternions (w, x, y, z)."""
    m00, m01, m02 = R[:, 0, 0], R[:, 0, 1], R[:, 0, 2]
    m10, m11, m12 = R[:, 1, 0], R[:, 1, 1], R[:, 1, 2]
    m20, m21, m22 = R[:, 2, 0], R[:, 2, 1], R[:, 2, 2]
    q = np.empty((R.shape[0], 4), dtype=np.float64)
    tr = m00 + m11 + m22
    # four candidate branches, pick the best conditioned one per row
    c0 = tr > 0
    c1 = (~c0) & (m00 >= m11) & (m00 >= m22)
    c2 = (~c0) & (~c1) & (m11 >= m22)
    c3 = ~(c0 | c1 | c2)
    with np.errstate(invalid="ignore"):
        s = np.sqrt(np.maximum(tr + 1.0, 1e-30)) * 2
        q[c0] = np.stack([0.25 * s, (m21 - m12) / s, (m02 - m20) / s, (m10 - m01) / s], 1)[c0]
        s = np.sqrt(np.maximum(1.0 + m00 - m11 - m22, 1e-30)) * 2
        q[c1] = np.stack([(m21 - m12) / s, 0.25 * s, (m01 + m10) / s, (m02 + m20) / s], 1)[c1]
        s = np.sqrt(np.maximum(1.0 + m11 - m00 - m22, 1e-30)) * 2
        q[c2] = np.stack([(m02 - m20) / s, (m01 + m10) / s, 0.25 * s, (m12 + m21) / s], 1)[c2]
        s = np.sqrt(np.maximum(1.0 + m22 - m00 - m11, 1e-30)) * 2
        q[c3] = np.stack([(m10 - m01) / s, (m02 + m20) / s, (m12 + m21) / s, 0.25 * s], 1)[c3]
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    return q


def _frames_from_normals(n: np.ndarray) -> np.ndarray:
    """Surfel frame [t_u t_v n] from unit plane normals (SURVEY 8(d) recipe)."""
    ref = np.where(np.abs(n[:, 2:3]) > 0.9, np.array([[1.0, 0, 0]]), np.array([[0, 0, 1.0]]))
    tu = np.cross(ref, n)
    tu /= np.linalg.norm(tu, axis=1, keepdims=True)
    tv = np.cross(n, tu)
    R = np.stack([tu, tv, n], axis=2)  # columns
    return _mat_to_quat(R)


def _deg(x: float) -> float:
    return float(np.deg2rad(x))


# ----------------------------------------------------------------------------
# scene sampling
# ----------------------------------------------------------------------------

def _make_boxes(rng, n_boxes: int, extent: float, ground_z: float) -> np.ndarray:
    """(B, 6): cx, cy, sx, sy, z0, z1 -- axis-aligned, standing on the ground."""
    cxy = rng.uniform(-0.9 * extent, 0.9 * extent, size=(n_boxes, 2))
    sxy = rng.uniform(3.0, 15.0, size=(n_boxes, 2))
    hgt = rng.uniform(3.0, 15.0, size=(n_boxes,))
    return np.concatenate([cxy, sxy, np.full((n_boxes, 1), ground_z), (ground_z + hgt)[:, None]], 1)


def _sample_ground(rng, n: int, kind: str, extent: float, ground_z: float):
    if kind == "disc":
        rad = extent * np.sqrt(rng.uniform(0, 1, n))
        ang = rng.uniform(-np.pi, np.pi, n)
        xy = np.stack([rad * np.cos(ang), rad * np.sin(ang)], 1)
    else:
        xy = rng.uniform(-extent, extent, size=(n, 2))
    pos = np.concatenate([xy, np.full((n, 1), ground_z)], 1)
    nrm = np.tile(np.array([[0.0, 0.0, 1.0]]), (n, 1))
    return pos, nrm


def _sample_facades(rng, n: int, boxes: np.ndarray):
    B = boxes.shape[0]
    cx, cy, sx, sy, z0, z1 = boxes.T
    h = z1 - z0
    # faces: +x, -x (width sy), +y, -y (width sx)
    area = np.stack([sy * h, sy * h, sx * h, sx * h], 1).reshape(-1)
    face = rng.choice(4 * B, size=n, p=area / area.sum())
    b, f = face // 4, face % 4
    a = rng.uniform(-0.5, 0.5, n)
    z = z0[b] + rng.uniform(0, 1, n) * h[b]
    pos = np.empty((n, 3))
    nrm = np.zeros((n, 3))
    fx = f < 2
    sgn = np.where(f % 2 == 0, 1.0, -1.0)
    pos[:, 0] = np.where(fx, cx[b] + sgn * 0.5 * sx[b], cx[b] + a * sx[b])
    pos[:, 1] = np.where(fx, cy[b] + a * sy[b], cy[b] + sgn * 0.5 * sy[b])
    pos[:, 2] = z
    nrm[:, 0] = np.where(fx, sgn, 0.0)
    nrm[:, 1] = np.where(fx, 0.0, sgn)
    return pos, nrm


def _range_aware_scales(rng, pos: np.ndarray, origin, W: int) -> np.ndarray:
    """s = 1.5 r (2 pi / W) U(0.8, 1.2), one jitter per component (shape of Eq. 6)."""
    r = np.linalg.norm(pos - np.asarray(origin)[None, :], axis=1)
    base = 1.5 * r * (2 * np.pi / W)
    return base[:, None] * rng.uniform(0.8, 1.2, size=(pos.shape[0], 2))


def _outside_boxes(p, boxes, margin=0.5) -> bool:
    cx, cy, sx, sy = boxes[:, 0], boxes[:, 1], boxes[:, 2], boxes[:, 3]
    inside = (np.abs(p[0] - cx) < 0.5 * sx + margin) & (np.abs(p[1] - cy) < 0.5 * sy + margin)
    return not bool(inside.any())


def _draw_pose(rng, boxes, span: float, tilt_deg: float = 2.0) -> np.ndarray:
    while True:
        p = np.array([rng.uniform(-span, span), rng.uniform(-span, span), 0.0])
        if boxes is None or _outside_boxes(p, boxes):
            break
    yaw = rng.uniform(-np.pi, np.pi)
    roll, pitch = rng.normal(0, _deg(tilt_deg), 2)
    return _pose(_rot_zyx(yaw, pitch, roll), p)


# ----------------------------------------------------------------------------
# scan simulator (input production; not the rasteriser)
# ----------------------------------------------------------------------------

def beam_grid(sensor: Sensor) -> np.ndarray:
    """(H, W, 3) unit beam directions in the sensor frame (x fwd, y left, z up).

    Grid convention (reading R1): azimuth phi_i = -pi + (i + 1/2) 2pi/W,
    elevation theta_j = elev_max - (j + 1/2) (elev_max - elev_min)/H.
    """
    H, W = sensor.H, sensor.W
    phi = -np.pi + (np.arange(W) + 0.5) * (2 * np.pi / W)
    th = sensor.elev_max - (np.arange(H) + 0.5) * ((sensor.elev_max - sensor.elev_min) / H)
    ct, st = np.cos(th)[:, None], np.sin(th)[:, None]
    d = np.stack([ct * np.cos(phi)[None, :], ct * np.sin(phi)[None, :], np.broadcast_to(st, (H, W))], -1)
    return d


def simulate_scan(scene: dict, sensor: Sensor, seed: int = 0, noise_sigma: float = 0.02):
    """Ray-cast the synthetic scene from the sensor pose.

    Returns (range (H, W) f32 with 0 = no return, normal (3, H, W) f32 in the
    sensor frame facing the sensor, zero where there is no return).  Gaussian
    range noise N(0, noise_sigma) stands in for LiDAR noise.
    """
    rng = np.random.default_rng(seed)
    H, W = sensor.H, sensor.W
    T = sensor.T_ws.astype(np.float64)
    R, o = T[:, :3], T[:, 3]
    d_s = beam_grid(sensor).reshape(-1, 3)
    d_w = d_s @ R.T
    P = d_w.shape[0]
    best_t = np.full(P, np.inf)
    best_n = np.zeros((P, 3))
    # ground
    gz = scene["ground_z"]
    with np.errstate(divide="ignore", invalid="ignore"):
        t = (gz - o[2]) / d_w[:, 2]
    hit = np.isfinite(t) & (t > 0)
    xy = o[None, :2] + t[:, None] * d_w[:, :2]
    if scene["ground_kind"] == "disc":
        hit &= (xy ** 2).sum(1) <= scene["ground_extent"] ** 2
    else:
        hit &= (np.abs(xy) <= scene["ground_extent"]).all(1)
    best_t[hit] = t[hit]
    best_n[hit] = np.array([0.0, 0.0, 1.0])
    # boxes (slab method), a few boxes at a time to bound memory
    boxes = scene.get("boxes")
    if boxes is not None and len(boxes):
        lo = np.stack([boxes[:, 0] - 0.5 * boxes[:, 2], boxes[:, 1] - 0.5 * boxes[:, 3], boxes[:, 4]], 1)
        hi = np.stack([boxes[:, 0] + 0.5 * boxes[:, 2], boxes[:, 1] + 0.5 * boxes[:, 3], boxes[:, 5]], 1)
        with np.errstate(divide="ignore", invalid="ignore"):
            inv = 1.0 / d_w
        for b in range(boxes.shape[0]):
            t0 = (lo[b][None, :] - o[None, :]) * inv
            t1 = (hi[b][None, :] - o[None, :]) * inv
            tn = np.minimum(t0, t1)
            tf = np.maximum(t0, t1)
            tnear = tn.max(1)
            tfar = tf.min(1)
            h = (tnear <= tfar) & (tnear > 0) & (tnear < best_t)
            if not h.any():
                continue
            ax = tn.argmax(1)
            nb = np.zeros((P, 3))
            nb[np.arange(P), ax] = -np.sign(d_w[np.arange(P), ax])
            best_t[h] = tnear[h]
            best_n[h] = nb[h]
    valid = np.isfinite(best_t) & (best_t >= max(sensor.r_min, 0.3))
    if np.isfinite(sensor.r_max):
        valid &= best_t <= sensor.r_max
    rng_img = np.where(valid, best_t + rng.normal(0, noise_sigma, P), 0.0)
    rng_img = np.where(valid & (rng_img > 0), rng_img, 0.0)
    n_s = best_n @ R  # R^T n, row form
    flip = (n_s * d_s).sum(1) > 0
    n_s[flip] *= -1
    n_s[~valid] = 0
    return (rng_img.reshape(H, W).astype(np.float32),
            np.ascontiguousarray(n_s.T.reshape(3, H, W)).astype(np.float32))


# ----------------------------------------------------------------------------
# the five BASELINE.json configs (+ a free-form random shell for tests)
# ----------------------------------------------------------------------------

def make_random_shell(seed: int, n: int, H: int, W: int, fov_deg=(-22.5, 22.5), r_lo=2.0, r_hi=20.0,
                      s_lo=0.05, s_hi=0.5, a_lo=0.1, a_hi=0.99, pose: Optional[np.ndarray] = None,
                      name: str = "shell") -> Workload:
    """Surfels uniform in a spherical shell around the origin, random frames."""
    rng = np.random.default_rng(seed)
    dirs = rng.normal(size=(n, 3))
    dirs /= np.linalg.norm(dirs, axis=1, keepdims=True)
    rad = rng.uniform(r_lo, r_hi, size=(n, 1))
    mean = dirs * rad
    quat = rng.normal(size=(n, 4))
    quat /= np.linalg.norm(quat, axis=1, keepdims=True)
    scale = rng.uniform(s_lo, s_hi, size=(n, 2))
    opacity = rng.uniform(a_lo, a_hi, size=(n,))
    pert = mean + rng.normal(0, 0.02, size=(n, 3))
    T = _pose(np.eye(3), [0, 0, 0]) if pose is None else np.asarray(pose, dtype=np.float32).reshape(3, 4)
    sensor = Sensor(H, W, _deg(fov_deg[0]), _deg(fov_deg[1]), 0.0, float("inf"), T)
    return Workload(name, mean.astype(np.float32), quat.astype(np.float32), scale.astype(np.float32),
                    opacity.astype(np.float32), [sensor], None, pert.astype(np.float32), None,
                    dict(lambda_n=0.0, lambda_ng=0.0, lambda_ns=0.0), seed)


def make_tiny(seed: int = 0) -> Workload:
    """BASELINE.json configs[0]: 64x256, 2,000 surfels in a 2-20 m shell, identity pose, L1 only."""
    w = make_random_shell(seed, 2000, 64, 256, name="tiny")
    return w


def _scene_workload(name, seed, n_surfels, H, W, fov_deg, ground_kind, extent, n_boxes, poses_fn,
                    a_lo, a_hi, r_max=float("inf"), clutter_frac=0.0, clutter_box=None,
                    clusters=None, cluster_frac=0.0) -> Workload:
    rng = np.random.default_rng(seed)
    ground_z = -1.7
    boxes = _make_boxes(rng, n_boxes, extent, ground_z)
    poses = poses_fn(rng, boxes)
    origin = poses[0][:, 3].astype(np.float64)
    n_clutter = int(round(clutter_frac * n_surfels))
    n_cluster = int(round(cluster_frac * n_surfels))
    n_plane = n_surfels - n_clutter - n_cluster
    n_ground = n_plane // 2
    n_fac = n_plane - n_ground
    gp, gn = _sample_ground(rng, n_ground, ground_kind, extent, ground_z)
    fp, fn = _sample_facades(rng, n_fac, boxes)
    pos = [gp, fp]
    nrm = [gn, fn]
    opa = [rng.uniform(a_lo, a_hi, n_ground + n_fac)]
    all_boxes = boxes
    if n_cluster:
        # 10 dense slabs: 50 parallel layers 0.05 m apart, facing the origin's x or y axis
        per = n_cluster // clusters
        cpos, cnrm, cbox = [], [], []
        for k in range(clusters):
            ang = rng.uniform(-np.pi, np.pi)
            dist = rng.uniform(10.0, 40.0)
            c = np.array([dist * np.cos(ang), dist * np.sin(ang)])
            along_x = bool(rng.integers(0, 2))  # layers stacked along x (normal +-x) or y
            m = per if k < clusters - 1 else n_cluster - per * (clusters - 1)
            layer = rng.integers(0, 50, m)
            u = rng.uniform(-3.0, 3.0, m)
            z = ground_z + rng.uniform(0, 4.0, m)
            off = (layer - 24.5) * 0.05
            p = np.empty((m, 3))
            nn = np.zeros((m, 3))
            if along_x:
                p[:, 0], p[:, 1] = c[0] + off, c[1] + u
                nn[:, 0] = 1.0
                cbox.append([c[0], c[1], 2.5, 6.0, ground_z, ground_z + 4.0])
            else:
                p[:, 0], p[:, 1] = c[0] + u, c[1] + off
                nn[:, 1] = 1.0
                cbox.append([c[0], c[1], 6.0, 2.5, ground_z, ground_z + 4.0])
            p[:, 2] = z
            cpos.append(p)
            cnrm.append(nn)
        pos.append(np.concatenate(cpos))
        nrm.append(np.concatenate(cnrm))
        opa.append(rng.uniform(0.05, 0.3, n_cluster))
        all_boxes = np.concatenate([boxes, np.array(cbox)], 0)
    if n_clutter:
        lo, hi = clutter_box
        cp = rng.uniform(lo, hi, size=(n_clutter, 3))
        cn = rng.normal(size=(n_clutter, 3))
        cn /= np.linalg.norm(cn, axis=1, keepdims=True)
        pos.append(cp)
        nrm.append(cn)
        opa.append(rng.uniform(a_lo, a_hi, n_clutter))
    pos = np.concatenate(pos)
    nrm = np.concatenate(nrm)
    opa = np.concatenate(opa)
    quat = _frames_from_normals(nrm)
    scale = _range_aware_scales(rng, pos, origin, W)
    if n_clutter:
        scale[-n_clutter:] = rng.uniform(0.02, 0.2, size=(n_clutter, 2))
    # shuffle so that map order carries no spatial structure (a SLAM map is insertion ordered,
    # the rasteriser may not rely on it)
    perm = rng.permutation(pos.shape[0])
    pos, quat, scale, opa = pos[perm], quat[perm], scale[perm], opa[perm]
    sensors = [Sensor(H, W, _deg(fov_deg[0]), _deg(fov_deg[1]), 0.0, r_max, T) for T in poses]
    scene = dict(ground_z=ground_z, ground_kind=ground_kind, ground_extent=extent, boxes=all_boxes)
    return Workload(name, pos.astype(np.float32), quat.astype(np.float32), scale.astype(np.float32),
                    opa.astype(np.float32), sensors, scene, None, None,
                    dict(lambda_n=1.0, lambda_ng=0.05, lambda_ns=0.01), seed + 1000)


def make_newer_college(seed: int = 1, n_surfels: int = 300_000, H: int = 64, W: int = 1024) -> Workload:
    """BASELINE.json configs[1] (graded): ground disc r=50 m at z=-1.7 + 40 boxes, range-aware scales."""
    return _scene_workload("newer_college", seed, n_surfels, H, W, (-22.5, 22.5), "disc", 50.0, 40,
                           lambda rng, boxes: [_draw_pose(rng, boxes, 20.0)], 0.3, 0.99)


def make_kitti(seed: int = 2, n_surfels: int = 1_000_000, H: int = 64, W: int = 2048, n_poses: int = 10) -> Workload:
    """BASELINE.json configs[2]: 64x2048, FOV -24.8..+2 deg, ground +-80 m + 200 boxes, 10 poses 1 m apart."""
    def poses(rng, boxes):
        return [_pose(np.eye(3), [float(k), 0.0, 0.0]) for k in range(n_poses)]
    return _scene_workload("kitti", seed, n_surfels, H, W, (-24.8, 2.0), "square", 80.0, 200, poses, 0.2, 0.99)


def make_large_map(seed: int = 3, n_surfels: int = 4_000_000, H: int = 128, W: int = 2048) -> Workload:
    """BASELINE.json configs[3]: 200 m x 200 m block, 5 % clutter, sensor at a corner, r_max = 100 m."""
    def poses(rng, boxes):
        return [_pose(_rot_zyx(np.pi / 4, 0.0, 0.0), [-100.0, -100.0, 0.0])]
    return _scene_workload("large_map", seed, n_surfels, H, W, (-22.5, 22.5), "square", 100.0, 400, poses,
                           0.3, 0.99, r_max=100.0, clutter_frac=0.05,
                           clutter_box=(np.array([-100.0, -100.0, -1.7]), np.array([100.0, 100.0, 8.0])))


def make_mapping_batch(seed: int = 4, n_surfels: int = 2_000_000, H: int = 64, W: int = 1024,
                       n_frames: int = 8) -> Workload:
    """BASELINE.json configs[4]: 8 keyframes vs a shared map, 30 % of surfels in 10 dense slabs, keep masks."""
    def poses(rng, boxes):
        return [_draw_pose(rng, boxes, 10.0) for _ in range(n_frames)]
    w = _scene_workload("mapping_batch", seed, n_surfels, H, W, (-22.5, 22.5), "disc", 80.0, 80, poses,
                        0.3, 0.99, clusters=10, cluster_frac=0.3)
    rng = np.random.default_rng(seed + 77)
    w.keep_masks = [(rng.uniform(size=(H, W)) >= 0.1).astype(np.uint8) for _ in range(n_frames)]
    return w


CONFIGS = {
    "tiny": make_tiny,
    "newer_college": make_newer_college,
    "kitti": make_kitti,
    "large_map": make_large_map,
    "mapping_batch": make_mapping_batch,
}
