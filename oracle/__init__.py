"""ORACLE -- test infrastructure only (see oracle/lgs_oracle.cpp header).

ctypes binding around the plain fp64 C++ oracle.  Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It imports nothing from paper_2607_04127_b200.

All array arguments are promoted to float64 ("inputs are the same fp32 arrays the
GPU gets, promoted to fp64"); float64 inputs are used as
they are (needed for finite differences).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lgs_oracle.cpp")
_LIB = os.path.join(_HERE, "liblgs_oracle.so")

BRUTE, BOUNDED = 0, 1


def build(force: bool = False) -> str:
    """Compile the oracle (g++, -ffp-contract=off so that fma appears only where written)."""
    if force or (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["g++", "-O2", "-std=c++17", "-fopenmp", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC",
               _SRC, "-o", _LIB]
        subprocess.check_call(cmd)
    return _LIB


class _CSensor(ctypes.Structure):
    _fields_ = [("H", ctypes.c_int32), ("W", ctypes.c_int32),
                ("elev_min", ctypes.c_double), ("elev_max", ctypes.c_double),
                ("r_min", ctypes.c_double), ("r_max", ctypes.c_double),
                ("T", ctypes.c_double * 12)]


_lib = None


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_LIB)
        _lib.lgs_oracle_tile_lists.restype = ctypes.c_int64
        _lib.lgs_oracle_num_threads.restype = ctypes.c_int
    return _lib


def num_threads() -> int:
    return int(_load().lgs_oracle_num_threads())


def _sensor(sensor) -> _CSensor:
    """`sensor` is any object with H, W, elev_min, elev_max, r_min, r_max, T_ws (3x4)."""
    s = _CSensor()
    s.H, s.W = int(sensor.H), int(sensor.W)
    # the C ABI of the CUDA library takes these as fp32: round the same way, then promote
    s.elev_min = float(np.float32(sensor.elev_min))
    s.elev_max = float(np.float32(sensor.elev_max))
    s.r_min = float(np.float32(sensor.r_min))
    s.r_max = float(np.float32(sensor.r_max))
    T = np.asarray(sensor.T_ws)
    if T.dtype != np.float64:
        T = T.astype(np.float32)
    T = T.astype(np.float64).reshape(12)
    for k in range(12):
        s.T[k] = float(T[k])
    return s


def _f64(a, shape=None):
    a = np.ascontiguousarray(np.asarray(a), dtype=np.float64)
    if shape is not None:
        a = a.reshape(shape)
    return a


def _p(a, ty=ctypes.c_double):
    if a is None:
        return None
    return a.ctypes.data_as(ctypes.POINTER(ty))


@dataclass
class ForwardResult:
    range: np.ndarray      # (H, W) f64, un-normalised sum_i w_i tau_i
    alpha: np.ndarray      # (H, W) f64
    normal: np.ndarray     # (3, H, W) f64, sensor frame, un-normalised
    ncontrib: np.ndarray   # (H, W) i32
    fragile: np.ndarray    # (H, W) bool
    stats: dict


def render_forward(mean, quat, scale, opacity, sensor, mode: int = BOUNDED, check_rects=None) -> ForwardResult:
    lib = _load()
    mean, quat, scale, opacity = _f64(mean), _f64(quat), _f64(scale), _f64(opacity)
    N = mean.shape[0]
    H, W = int(sensor.H), int(sensor.W)
    rng = np.empty((H, W)); alp = np.empty((H, W)); nrm = np.empty((3, H, W))
    ncon = np.empty((H, W), dtype=np.int32); frag = np.empty((H, W), dtype=np.uint8)
    stats = np.zeros(8, dtype=np.int64)
    cr = None
    if check_rects is not None:
        cr = np.ascontiguousarray(check_rects, dtype=np.int32).reshape(N, 4)
    cs = _sensor(sensor)
    rc = lib.lgs_oracle_forward(ctypes.c_int64(N), _p(mean), _p(quat), _p(scale), _p(opacity), ctypes.byref(cs),
                                ctypes.c_int(mode), _p(rng), _p(alp), _p(nrm), _p(ncon, ctypes.c_int32),
                                _p(frag, ctypes.c_uint8), _p(cr, ctypes.c_int32), _p(stats, ctypes.c_int64))
    assert rc == 0
    names = ["n_alive", "I_c", "I_3sigma", "I_visited", "n_fragile", "rect_violations", "n_stopped"]
    return ForwardResult(rng, alp, nrm, ncon, frag.astype(bool), {k: int(stats[i]) for i, k in enumerate(names)})


def render_backward(mean, quat, scale, opacity, sensor, gD, gA=None, gN=None, mode: int = BOUNDED,
                    with_cond: bool = False):
    """Returns (g_mean [N,3], g_quat [N,4], g_scale [N,2], g_opacity [N]) in fp64
    (+ cond [N,4], the conditioning diagnostic of lgs_oracle_backward, if with_cond)."""
    lib = _load()
    mean, quat, scale, opacity = _f64(mean), _f64(quat), _f64(scale), _f64(opacity)
    N = mean.shape[0]
    H, W = int(sensor.H), int(sensor.W)
    gD = _f64(gD, (H, W)) if gD is not None else None
    gA = _f64(gA, (H, W)) if gA is not None else None
    gN = _f64(gN, (3, H, W)) if gN is not None else None
    gm = np.empty((N, 3)); gq = np.empty((N, 4)); gs = np.empty((N, 2)); go = np.empty((N,))
    cs = _sensor(sensor)
    cond = np.empty((N, 4)) if with_cond else None
    rc = lib.lgs_oracle_backward(ctypes.c_int64(N), _p(mean), _p(quat), _p(scale), _p(opacity), ctypes.byref(cs),
                                 ctypes.c_int(mode), _p(gD), _p(gA), _p(gN), _p(gm), _p(gq), _p(gs), _p(go), _p(cond))
    assert rc == 0
    if with_cond:
        return gm, gq, gs, go, cond
    return gm, gq, gs, go


@dataclass
class LossResult:
    loss: float
    L_depth: float
    L_ng: float
    L_ns: float
    n_M: int
    n_N: int
    n_S: int
    gD: np.ndarray
    gA: np.ndarray
    gN: np.ndarray
    sign_fragile: np.ndarray


def loss_range_normal(sensor, range_, alpha, normal, target_range, target_normal=None, keep_mask=None,
                      lambda_n=1.0, lambda_ng=0.05, lambda_ns=0.01, detach_surf=False) -> LossResult:
    lib = _load()
    H, W = int(sensor.H), int(sensor.W)
    range_ = _f64(range_, (H, W)); alpha = _f64(alpha, (H, W)); normal = _f64(normal, (3, H, W))
    target_range = _f64(target_range, (H, W))
    tn = _f64(target_normal, (3, H, W)) if target_normal is not None else None
    km = np.ascontiguousarray(keep_mask, dtype=np.uint8).reshape(H, W) if keep_mask is not None else None
    gD = np.empty((H, W)); gA = np.empty((H, W)); gN = np.empty((3, H, W))
    sf = np.empty((H, W), dtype=np.uint8)
    losses = np.zeros(4); counts = np.zeros(3, dtype=np.int64)
    cs = _sensor(sensor)
    rc = lib.lgs_oracle_loss(ctypes.byref(cs), _p(range_), _p(alpha), _p(normal), _p(target_range), _p(tn),
                             _p(km, ctypes.c_uint8), ctypes.c_double(lambda_n), ctypes.c_double(lambda_ng),
                             ctypes.c_double(lambda_ns), ctypes.c_int(int(detach_surf)), _p(losses),
                             _p(counts, ctypes.c_int64), _p(gD), _p(gA), _p(gN), _p(sf, ctypes.c_uint8))
    assert rc == 0
    return LossResult(float(losses[0]), float(losses[1]), float(losses[2]), float(losses[3]),
                      int(counts[0]), int(counts[1]), int(counts[2]), gD, gA, gN, sf.astype(bool))


@dataclass
class TileLists:
    keys: np.ndarray         # (K,) u64 sorted
    vals: np.ndarray         # (K,) u32
    tile_ranges: np.ndarray  # (n_tiles, 2) u32
    rects: np.ndarray        # (N, 4) i32: col_min, ncols, row_min, row_max
    rkeys: np.ndarray        # (N,) f32


TILE_W, TILE_H = 8, 4     # list tiles of the CUDA path (include/lgs.h LGS_TILE_W / LGS_TILE_H)


def footprint_surfels(mean, quat, scale, opacity, sensor) -> np.ndarray:
    """bool [N]: surfels with a non-empty footprint (SURVEY.md 8(d)'s N_fp = its sum) -- some beam of the grid meets the
    surfel inside its 3 sigma ellipse (|den| >= den_min, tau > 0, rho2 <= 9), whatever lies in front of it."""
    lib = _load()
    lib.lgs_oracle_footprint.restype = ctypes.c_int64
    mean, quat, scale, opacity = _f64(mean), _f64(quat), _f64(scale), _f64(opacity)
    N = mean.shape[0]
    touched = np.zeros(max(N, 1), dtype=np.uint8)
    cs = _sensor(sensor)
    n = lib.lgs_oracle_footprint(ctypes.c_int64(N), _p(mean), _p(quat), _p(scale), _p(opacity), ctypes.byref(cs),
                                 _p(touched, ctypes.c_uint8))
    assert n == int(touched[:N].sum())
    return touched[:N].astype(bool)


def tile_lists(mean, quat, scale, opacity, sensor, tile=(TILE_W, TILE_H)) -> TileLists:
    """List reference for tiles of tile = (columns, rows) pixels (an int means a square tile)."""
    lib = _load()
    tile_w, tile_h = (tile, tile) if isinstance(tile, int) else (int(tile[0]), int(tile[1]))
    mean, quat, scale, opacity = _f64(mean), _f64(quat), _f64(scale), _f64(opacity)
    N = mean.shape[0]
    H, W = int(sensor.H), int(sensor.W)
    nt = ((H + tile_h - 1) // tile_h) * ((W + tile_w - 1) // tile_w)
    rects = np.zeros((N, 4), dtype=np.int32)
    rkeys = np.zeros((N,), dtype=np.float32)
    ranges = np.zeros((nt, 2), dtype=np.uint32)
    cs = _sensor(sensor)
    cap = max(1024, 4 * N)
    while True:
        keys = np.zeros((cap,), dtype=np.uint64)
        vals = np.zeros((cap,), dtype=np.uint32)
        K = lib.lgs_oracle_tile_lists(ctypes.c_int64(N), _p(mean), _p(quat), _p(scale), _p(opacity), ctypes.byref(cs),
                                      ctypes.c_int(tile_w), ctypes.c_int(tile_h), ctypes.c_int64(cap), _p(keys, ctypes.c_uint64),
                                      _p(vals, ctypes.c_uint32), _p(ranges, ctypes.c_uint32), _p(rects, ctypes.c_int32),
                                      _p(rkeys, ctypes.c_float))
        if K <= cap:
            break
        cap = int(K)
    return TileLists(keys[:K].copy(), vals[:K].copy(), ranges, rects, rkeys)
