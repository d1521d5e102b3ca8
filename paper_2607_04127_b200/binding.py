"""ctypes binding of include/lgs.h -- argument marshalling only.

Every function has the name of the C entry point it calls.  Tensors are torch CUDA
tensors (fp32, contiguous); torch is used for device memory and streams, nothing else:
every step of the path runs in the library's kernels.  There is no CPU fallback: if
liblgs.so cannot be loaded the call raises.
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIBPATH = os.path.join(_HERE, "liblgs.so")
LGS_TILE_W, LGS_TILE_H = 8, 4

_STATUS = {0: "LGS_OK", 1: "LGS_ERR_INVALID_ARG", 2: "LGS_ERR_WORKSPACE_TOO_SMALL", 3: "LGS_ERR_KEY_OVERFLOW",
           4: "LGS_ERR_CUDA", 5: "LGS_ERR_UNSUPPORTED_DEVICE", 6: "LGS_ERR_STATIC_LIMIT"}


class LgsError(RuntimeError):
    def __init__(self, code: int, where: str):
        super().__init__("%s returned %s" % (where, _STATUS.get(code, code)))
        self.code = code


class _CGaussians(ctypes.Structure):
    _fields_ = [("mean", ctypes.c_void_p), ("quat", ctypes.c_void_p), ("scale", ctypes.c_void_p),
                ("opacity", ctypes.c_void_p), ("N", ctypes.c_int64)]


class _CSensor(ctypes.Structure):
    _fields_ = [("H", ctypes.c_int32), ("W", ctypes.c_int32), ("elev_min", ctypes.c_float),
                ("elev_max", ctypes.c_float), ("r_min", ctypes.c_float), ("r_max", ctypes.c_float),
                ("T_ws", ctypes.c_float * 12)]


@dataclass
class Sensor:
    """Host-side mirror of lgs_sensor."""
    H: int
    W: int
    elev_min: float
    elev_max: float
    r_min: float
    r_max: float
    T_ws: np.ndarray  # (3, 4)

    @staticmethod
    def of(obj) -> "Sensor":
        return Sensor(int(obj.H), int(obj.W), float(obj.elev_min), float(obj.elev_max), float(obj.r_min),
                      float(obj.r_max), np.asarray(obj.T_ws, dtype=np.float32).reshape(3, 4))

    def c(self) -> _CSensor:
        s = _CSensor()
        s.H, s.W = self.H, self.W
        s.elev_min, s.elev_max, s.r_min, s.r_max = self.elev_min, self.elev_max, self.r_min, self.r_max
        T = np.asarray(self.T_ws, dtype=np.float32).reshape(12)
        for k in range(12):
            s.T_ws[k] = float(T[k])
        return s


_lib = None


def library_path() -> str:
    return _LIBPATH


def _load():
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIBPATH):
        # build in-tree if a toolchain is present; otherwise fail loudly (no fallback path exists)
        from . import build as _build
        _build.build()
    lib = ctypes.CDLL(_LIBPATH)
    lib.lgs_workspace_bytes.restype = ctypes.c_size_t
    lib.lgs_workspace_bytes.argtypes = [ctypes.c_int64, ctypes.c_int32, ctypes.c_int32, ctypes.c_int64]
    lib.lgs_loss_workspace_bytes.restype = ctypes.c_size_t
    lib.lgs_loss_workspace_bytes.argtypes = [ctypes.c_int32, ctypes.c_int32]
    lib.lgs_version.restype = ctypes.c_char_p
    vp, i64, i32, f32 = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int32, ctypes.c_float
    lib.lgs_render_forward.restype = ctypes.c_int
    lib.lgs_render_forward.argtypes = [ctypes.POINTER(_CGaussians), ctypes.POINTER(_CSensor), vp, ctypes.c_size_t, i64,
                                       vp, vp, vp, vp]
    lib.lgs_render_backward.restype = ctypes.c_int
    lib.lgs_render_backward.argtypes = [ctypes.POINTER(_CGaussians), ctypes.POINTER(_CSensor), vp, ctypes.c_size_t, i64,
                                        vp, vp, vp, vp, vp, vp, vp, ctypes.c_int, vp]
    lib.lgs_workspace_bytes_batch.restype = ctypes.c_size_t
    lib.lgs_workspace_bytes_batch.argtypes = [i64, i32, i32, i64, i32]
    lib.lgs_render_forward_batch.restype = ctypes.c_int
    lib.lgs_render_forward_batch.argtypes = [ctypes.POINTER(_CGaussians), ctypes.POINTER(_CSensor), i32, vp, ctypes.c_size_t,
                                             i64, vp, vp, vp, vp]
    lib.lgs_render_backward_batch.restype = ctypes.c_int
    lib.lgs_render_backward_batch.argtypes = [ctypes.POINTER(_CGaussians), ctypes.POINTER(_CSensor), i32, vp, ctypes.c_size_t,
                                              i64, vp, vp, vp, vp, vp, vp, vp, ctypes.c_int, vp]
    lib.lgs_loss_range_normal.restype = ctypes.c_int
    lib.lgs_loss_range_normal.argtypes = [ctypes.POINTER(_CSensor), vp, vp, vp, vp, vp, vp, f32, f32, f32, ctypes.c_int,
                                          vp, ctypes.c_size_t, vp, vp, vp, vp, vp]
    lib.lgs_loss_mapping.restype = ctypes.c_int
    lib.lgs_loss_mapping.argtypes = [ctypes.POINTER(_CSensor), vp, vp, vp, vp, vp, vp, f32, f32, f32, f32, f32, ctypes.c_int,
                                     vp, ctypes.c_size_t, vp, vp, vp, vp, vp]
    lib.lgs_adam_step.restype = ctypes.c_int
    lib.lgs_adam_step.argtypes = [i64, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, ctypes.POINTER(_CAdam), vp, vp]
    lib.lgs_prune_workspace_bytes.restype = ctypes.c_size_t
    lib.lgs_prune_workspace_bytes.argtypes = [i64]
    lib.lgs_prune_compact.restype = ctypes.c_int
    lib.lgs_prune_compact.argtypes = [i64, f32] + [vp] * 15 + [vp, ctypes.c_size_t, vp]
    lib.lgs_scan_to_range_image.restype = ctypes.c_int
    lib.lgs_scan_to_range_image.argtypes = [vp, vp, i64, ctypes.POINTER(_CSensor), vp, ctypes.c_size_t, vp, vp, vp]
    lib.lgs_scan_to_range_image_static.restype = ctypes.c_int
    lib.lgs_scan_to_range_image_static.argtypes = [vp, vp, i64, ctypes.POINTER(_CSensor), vp, vp, vp]
    lib.lgs_query.restype = ctypes.c_int
    lib.lgs_query.argtypes = [vp, i64, i32, i32, i64, ctypes.POINTER(i64), ctypes.POINTER(i64), ctypes.POINTER(i64), vp]
    lib.lgs_debug_tile_lists.restype = ctypes.c_int
    lib.lgs_debug_tile_lists.argtypes = [vp, ctypes.POINTER(_CSensor), i64, i64, vp, vp, ctypes.POINTER(vp), vp, vp]
    lib.lgs_debug_tile_lists_batch.restype = ctypes.c_int
    lib.lgs_debug_tile_lists_batch.argtypes = [vp, ctypes.POINTER(_CSensor), i32, i64, i64, vp, vp, ctypes.POINTER(vp), vp, vp]
    lib.lgs_debug_segmented_sort.restype = ctypes.c_int
    lib.lgs_debug_segmented_sort.argtypes = [vp, vp, vp, vp, vp, i32, vp]
    _lib = lib
    return lib


def _ptr(t, dtype=None, numel=None, name="tensor"):
    """Device pointer of a contiguous CUDA tensor (None -> NULL)."""
    import torch
    if t is None:
        return None
    if not isinstance(t, torch.Tensor) or not t.is_cuda or not t.is_contiguous():
        raise TypeError("%s must be a contiguous CUDA tensor" % name)
    if dtype is not None and t.dtype != dtype:
        raise TypeError("%s must be %s, got %s" % (name, dtype, t.dtype))
    if numel is not None and t.numel() != numel:
        raise ValueError("%s has %d elements, expected %d" % (name, t.numel(), numel))
    return ctypes.c_void_p(t.data_ptr())


def _stream(stream):
    import torch
    if stream is None:
        stream = torch.cuda.current_stream()
    return ctypes.c_void_p(stream.cuda_stream)


def _gauss(mean, quat, scale, opacity) -> _CGaussians:
    import torch
    N = int(opacity.numel())
    g = _CGaussians()
    g.mean = _ptr(mean, torch.float32, 3 * N, "mean").value if N else None
    g.quat = _ptr(quat, torch.float32, 4 * N, "quat").value if N else None
    g.scale = _ptr(scale, torch.float32, 2 * N, "scale").value if N else None
    g.opacity = _ptr(opacity, torch.float32, N, "opacity").value if N else None
    g.N = N
    return g


def _check(code: int, where: str):
    if code != 0:
        raise LgsError(code, where)


def lgs_version() -> str:
    return _load().lgs_version().decode()


def lgs_workspace_bytes(N: int, H: int, W: int, max_keys: int) -> int:
    return int(_load().lgs_workspace_bytes(N, H, W, max_keys))


def lgs_loss_workspace_bytes(H: int, W: int) -> int:
    return int(_load().lgs_loss_workspace_bytes(H, W))


def lgs_render_forward(mean, quat, scale, opacity, sensor: Sensor, workspace, max_keys: int, out_range, out_alpha,
                       out_normal=None, stream=None) -> None:
    import torch
    lib = _load()
    HW = sensor.H * sensor.W
    g = _gauss(mean, quat, scale, opacity)
    cs = sensor.c()
    _check(lib.lgs_render_forward(ctypes.byref(g), ctypes.byref(cs), _ptr(workspace, torch.uint8, None, "workspace"),
                                  workspace.numel(), max_keys, _ptr(out_range, torch.float32, HW, "out_range"),
                                  _ptr(out_alpha, torch.float32, HW, "out_alpha"),
                                  _ptr(out_normal, torch.float32, 3 * HW, "out_normal"), _stream(stream)),
           "lgs_render_forward")


def lgs_render_backward(mean, quat, scale, opacity, sensor: Sensor, workspace, max_keys: int, dL_drange,
                        dL_dalpha, dL_dnormal, g_mean, g_quat, g_scale, g_opacity, accumulate: bool = False,
                        stream=None) -> None:
    import torch
    lib = _load()
    HW = sensor.H * sensor.W
    g = _gauss(mean, quat, scale, opacity)
    N = g.N
    cs = sensor.c()
    _check(lib.lgs_render_backward(ctypes.byref(g), ctypes.byref(cs), _ptr(workspace, torch.uint8, None, "workspace"),
                                   workspace.numel(), max_keys, _ptr(dL_drange, torch.float32, HW, "dL_drange"),
                                   _ptr(dL_dalpha, torch.float32, HW, "dL_dalpha"),
                                   _ptr(dL_dnormal, torch.float32, 3 * HW, "dL_dnormal"),
                                   _ptr(g_mean, torch.float32, 3 * N, "g_mean"), _ptr(g_quat, torch.float32, 4 * N, "g_quat"),
                                   _ptr(g_scale, torch.float32, 2 * N, "g_scale"),
                                   _ptr(g_opacity, torch.float32, N, "g_opacity"), int(bool(accumulate)), _stream(stream)),
           "lgs_render_backward")


LGS_MAX_FRAMES = 16


def _sensor_array(sensors):
    arr = (_CSensor * len(sensors))()
    for k, sn in enumerate(sensors):
        arr[k] = sn.c()
    return arr


def lgs_workspace_bytes_batch(N: int, H: int, W: int, max_keys: int, F: int) -> int:
    return int(_load().lgs_workspace_bytes_batch(N, H, W, max_keys, F))


def lgs_render_forward_batch(mean, quat, scale, opacity, sensors, workspace, max_keys: int, out_range, out_alpha,
                             out_normal=None, stream=None) -> None:
    """F keyframes (list of Sensor: same grid, one pose each) against one map in one sequence of kernels;
    out_range / out_alpha [F,H,W], out_normal [F,3,H,W]."""
    import torch
    lib = _load()
    F = len(sensors)
    HW = sensors[0].H * sensors[0].W
    g = _gauss(mean, quat, scale, opacity)
    arr = _sensor_array(sensors)
    _check(lib.lgs_render_forward_batch(ctypes.byref(g), arr, F, _ptr(workspace, torch.uint8, None, "workspace"),
                                        workspace.numel(), max_keys, _ptr(out_range, torch.float32, F * HW, "out_range"),
                                        _ptr(out_alpha, torch.float32, F * HW, "out_alpha"),
                                        _ptr(out_normal, torch.float32, 3 * F * HW, "out_normal"), _stream(stream)),
           "lgs_render_forward_batch")


def lgs_render_backward_batch(mean, quat, scale, opacity, sensors, workspace, max_keys: int, dL_drange, dL_dalpha,
                              dL_dnormal, g_mean, g_quat, g_scale, g_opacity, accumulate: bool = False,
                              stream=None) -> None:
    import torch
    lib = _load()
    F = len(sensors)
    HW = sensors[0].H * sensors[0].W
    g = _gauss(mean, quat, scale, opacity)
    N = g.N
    arr = _sensor_array(sensors)
    _check(lib.lgs_render_backward_batch(ctypes.byref(g), arr, F, _ptr(workspace, torch.uint8, None, "workspace"),
                                         workspace.numel(), max_keys, _ptr(dL_drange, torch.float32, F * HW, "dL_drange"),
                                         _ptr(dL_dalpha, torch.float32, F * HW, "dL_dalpha"),
                                         _ptr(dL_dnormal, torch.float32, 3 * F * HW, "dL_dnormal"),
                                         _ptr(g_mean, torch.float32, 3 * N, "g_mean"),
                                         _ptr(g_quat, torch.float32, 4 * N, "g_quat"),
                                         _ptr(g_scale, torch.float32, 2 * N, "g_scale"),
                                         _ptr(g_opacity, torch.float32, N, "g_opacity"), int(bool(accumulate)),
                                         _stream(stream)),
           "lgs_render_backward_batch")


def lgs_loss_range_normal(sensor: Sensor, range_, alpha, normal, target_range, target_normal, keep_mask,
                          lambda_n: float, lambda_ng: float, lambda_ns: float, detach_surf: bool, loss_workspace,
                          loss, dL_drange, dL_dalpha, dL_dnormal, stream=None) -> None:
    import torch
    lib = _load()
    HW = sensor.H * sensor.W
    cs = sensor.c()
    _check(lib.lgs_loss_range_normal(ctypes.byref(cs), _ptr(range_, torch.float32, HW, "range"),
                                     _ptr(alpha, torch.float32, HW, "alpha"), _ptr(normal, torch.float32, 3 * HW, "normal"),
                                     _ptr(target_range, torch.float32, HW, "target_range"),
                                     _ptr(target_normal, torch.float32, 3 * HW, "target_normal"),
                                     _ptr(keep_mask, torch.uint8, HW, "keep_mask"), lambda_n, lambda_ng, lambda_ns,
                                     int(bool(detach_surf)), _ptr(loss_workspace, torch.uint8, None, "loss_workspace"),
                                     loss_workspace.numel(), _ptr(loss, torch.float32, 4, "loss"),
                                     _ptr(dL_drange, torch.float32, HW, "dL_drange"),
                                     _ptr(dL_dalpha, torch.float32, HW, "dL_dalpha"),
                                     _ptr(dL_dnormal, torch.float32, 3 * HW, "dL_dnormal"), _stream(stream)),
           "lgs_loss_range_normal")


def lgs_loss_mapping(sensor: Sensor, range_, alpha, normal, target_range, target_normal, keep_mask,
                     lambda_alpha: float, alpha_eps: float, lambda_n: float, lambda_ng: float, lambda_ns: float,
                     detach_surf: bool, loss_workspace, loss, dL_drange, dL_dalpha, dL_dnormal, stream=None) -> None:
    """Image side of Eq. 13 (adds lambda_alpha L_alpha, Eq. 10 right); loss is a float[5] tensor."""
    import torch
    lib = _load()
    HW = sensor.H * sensor.W
    cs = sensor.c()
    _check(lib.lgs_loss_mapping(ctypes.byref(cs), _ptr(range_, torch.float32, HW, "range"),
                                _ptr(alpha, torch.float32, HW, "alpha"), _ptr(normal, torch.float32, 3 * HW, "normal"),
                                _ptr(target_range, torch.float32, HW, "target_range"),
                                _ptr(target_normal, torch.float32, 3 * HW, "target_normal"),
                                _ptr(keep_mask, torch.uint8, HW, "keep_mask"), lambda_alpha, alpha_eps, lambda_n,
                                lambda_ng, lambda_ns, int(bool(detach_surf)),
                                _ptr(loss_workspace, torch.uint8, None, "loss_workspace"), loss_workspace.numel(),
                                _ptr(loss, torch.float32, 5, "loss"), _ptr(dL_drange, torch.float32, HW, "dL_drange"),
                                _ptr(dL_dalpha, torch.float32, HW, "dL_dalpha"),
                                _ptr(dL_dnormal, torch.float32, 3 * HW, "dL_dnormal"), _stream(stream)),
           "lgs_loss_mapping")


class _CAdam(ctypes.Structure):
    _fields_ = [("lr_mean", ctypes.c_float), ("lr_quat", ctypes.c_float), ("lr_scale", ctypes.c_float),
                ("lr_opacity", ctypes.c_float), ("beta1", ctypes.c_float), ("beta2", ctypes.c_float),
                ("eps", ctypes.c_float), ("step", ctypes.c_int32), ("lambda_s", ctypes.c_float),
                ("s_max", ctypes.c_float), ("alpha_lo", ctypes.c_float), ("alpha_hi", ctypes.c_float),
                ("step_device", ctypes.c_void_p)]


def lgs_adam_step(mean, quat, log_scale, opacity, scale, g_mean, g_quat, g_scale, g_opacity, m, v, step: int,
                  lr_mean: float, lr_quat: float, lr_scale: float, lr_opacity: float, beta1: float = 0.9,
                  beta2: float = 0.999, eps: float = 1e-15, lambda_s: float = 10.0, s_max: float = 1.0,
                  alpha_lo: float = 0.0, alpha_hi: float = 1.0, loss_scale=None, stream=None, step_device=None) -> None:
    """One fused Adam step on {mu, q, log s, alpha} with the Eq. 12 regulariser (include/lgs.h: lgs_adam_step).
    step_device: optional int32 CUDA tensor holding t (then `step` is ignored; for CUDA-graph replays)."""
    import torch
    lib = _load()
    N = int(mean.shape[0])
    sd = _ptr(step_device, torch.int32, 1, "step_device")
    h = _CAdam(lr_mean, lr_quat, lr_scale, lr_opacity, beta1, beta2, eps, int(step), lambda_s, s_max, alpha_lo, alpha_hi,
               sd.value if sd is not None else None)
    _check(lib.lgs_adam_step(N, _ptr(mean, torch.float32, 3 * N, "mean"), _ptr(quat, torch.float32, 4 * N, "quat"),
                             _ptr(log_scale, torch.float32, 2 * N, "log_scale"),
                             _ptr(opacity, torch.float32, N, "opacity"), _ptr(scale, torch.float32, 2 * N, "scale"),
                             _ptr(g_mean, torch.float32, 3 * N, "g_mean"), _ptr(g_quat, torch.float32, 4 * N, "g_quat"),
                             _ptr(g_scale, torch.float32, 2 * N, "g_scale"),
                             _ptr(g_opacity, torch.float32, N, "g_opacity"), _ptr(m, torch.float32, 10 * N, "m"),
                             _ptr(v, torch.float32, 10 * N, "v"), ctypes.byref(h),
                             _ptr(loss_scale, torch.float32, 1, "loss_scale"), _stream(stream)),
           "lgs_adam_step")


def lgs_prune_workspace_bytes(N: int) -> int:
    return int(_load().lgs_prune_workspace_bytes(N))


def lgs_prune_compact(alpha_min: float, mean, quat, log_scale, opacity, scale=None, m=None, v=None, stream=None,
                      out=None):
    """Opacity prune + compaction (include/lgs.h).  Returns (n_out, [compacted tensors in the order of the inputs that
    were given]); the outputs are new tensors of N rows of capacity whose first n_out rows are valid.  Synchronises
    (reads n_out).
    out = (outputs, n_out, workspace) -- a list of 7 pre-allocated output tensors (None where the input is None), a
    device int64 tensor [1] and a uint8 workspace of lgs_prune_workspace_bytes(N): the call then allocates nothing,
    does not synchronise, and returns (n_out tensor, outputs)."""
    import torch
    lib = _load()
    N = int(opacity.numel())
    ins = [mean, quat, log_scale, opacity, scale, m, v]
    widths = [3, 4, 2, 1, 2, 10, 10]
    if out is not None:
        outs, n_out, ws = out
        pin = [None if t is None else _ptr(t, torch.float32, w * N, "in") for t, w in zip(ins, widths)]
        pout = [None if t is None else _ptr(t, torch.float32, w * N, "out") for t, w in zip(outs, widths)]
        _check(lib.lgs_prune_compact(N, alpha_min, *pin, *pout, ctypes.c_void_p(n_out.data_ptr()),
                                     ctypes.c_void_p(ws.data_ptr()), ws.numel(), _stream(stream)), "lgs_prune_compact")
        return n_out, [t for t in outs if t is not None]
    outs = [None if t is None else torch.empty_like(t) for t in ins]
    n_out = torch.zeros(1, dtype=torch.int64, device=opacity.device)
    ws = torch.empty(max(lgs_prune_workspace_bytes(N), 4), dtype=torch.uint8, device=opacity.device)
    pin = [None if t is None else _ptr(t, torch.float32, w * N, "in") for t, w in zip(ins, widths)]
    pout = [None if t is None else _ptr(t, torch.float32, w * N, "out") for t, w in zip(outs, widths)]
    _check(lib.lgs_prune_compact(N, alpha_min, *pin, *pout, ctypes.c_void_p(n_out.data_ptr()),
                                 ctypes.c_void_p(ws.data_ptr()), ws.numel(), _stream(stream)), "lgs_prune_compact")
    # the kernels run on `stream`, which need not be torch's current stream: order the read-back (and the allocator's
    # reuse of ws) behind THAT stream
    (stream if stream is not None else torch.cuda.current_stream()).synchronize()
    n = int(n_out.item())
    return n, [t for t in outs if t is not None]


def lgs_scan_to_range_image(points, normals, sensor: Sensor, zbuf, out_range, out_normal=None, stream=None) -> None:
    """Scan (sensor-frame points [M,3], optional normals [M,3]) -> range image [H,W] and normal image [3,H,W]."""
    import torch
    lib = _load()
    HW = sensor.H * sensor.W
    M = int(points.shape[0])
    cs = sensor.c()
    _check(lib.lgs_scan_to_range_image(_ptr(points, torch.float32, 3 * M, "points") if M else None,
                                       _ptr(normals, torch.float32, 3 * M, "normals") if M else None, M,
                                       ctypes.byref(cs), _ptr(zbuf, torch.uint8, None, "zbuf"), zbuf.numel(),
                                       _ptr(out_range, torch.float32, HW, "out_range"),
                                       _ptr(out_normal, torch.float32, 3 * HW, "out_normal"), _stream(stream)),
           "lgs_scan_to_range_image")


LGS_SCAN_STATIC_MAX_PIXELS = 1 << 18


def lgs_scan_to_range_image_static(points, normals, sensor: Sensor, out_range, out_normal=None, stream=None) -> None:
    """lgs_scan_to_range_image without a `zbuf` argument, for callers that cannot allocate device memory where they run
    (a real-time scan callback that must not enter cudaMalloc, a process whose device memory is all in a pool it does not
    own, a plugin in a host program that does all allocation).  The z-buffer is a fixed 2 MiB array inside liblgs.so,
    one per GPU, so: H * W must be <= LGS_SCAN_STATIC_MAX_PIXELS (else LgsError LGS_ERR_STATIC_LIMIT, nothing is
    launched); make the first call on each device at start-up, outside any stream capture (it looks the array up);
    calls that can overlap on one GPU race on the array -- order them.  Outputs equal lgs_scan_to_range_image's bit for
    bit.  This wrapper itself creates no tensor."""
    import torch
    lib = _load()
    HW = sensor.H * sensor.W
    M = int(points.shape[0])
    cs = sensor.c()
    _check(lib.lgs_scan_to_range_image_static(_ptr(points, torch.float32, 3 * M, "points") if M else None,
                                              _ptr(normals, torch.float32, 3 * M, "normals") if M else None, M,
                                              ctypes.byref(cs), _ptr(out_range, torch.float32, HW, "out_range"),
                                              _ptr(out_normal, torch.float32, 3 * HW, "out_normal"), _stream(stream)),
           "lgs_scan_to_range_image_static")


def lgs_query(workspace, N: int, H: int, W: int, max_keys: int, stream=None):
    """Returns (n_visible, n_keys, n_contrib, overflowed). Synchronises the stream."""
    import torch
    lib = _load()
    a, b, c = ctypes.c_int64(0), ctypes.c_int64(0), ctypes.c_int64(0)
    code = lib.lgs_query(_ptr(workspace, torch.uint8, None, "workspace"), N, H, W, max_keys, ctypes.byref(a),
                         ctypes.byref(b), ctypes.byref(c), _stream(stream))
    if code not in (0, 3):
        raise LgsError(code, "lgs_query")
    return int(a.value), int(b.value), int(c.value), code == 3


def lgs_debug_tile_lists(workspace, sensor: Sensor, N: int, max_keys: int, stream=None, frames: int = 1):
    """Test-only: (keys u64 [K], vals u32 [K], tile_ranges u32 [F n_tiles,2], rects i32 [F N,4]) as numpy arrays
    (frames > 1: of a batched forward; keys then carry the global tile id f * n_tiles + tile)."""
    import torch
    lib = _load()
    H, W = sensor.H, sensor.W
    n_vis, K, _, ovf = lgs_query(workspace, N, H, W, max_keys, stream)
    if ovf:
        raise LgsError(3, "lgs_debug_tile_lists")
    rp = ctypes.c_void_p()
    dev = workspace.device
    keys_d = torch.zeros(max(K, 1), dtype=torch.int64, device=dev)
    vals_d = torch.zeros(max(K, 1), dtype=torch.int32, device=dev)
    rects = torch.zeros((max(N * frames, 1), 4), dtype=torch.int32, device=dev)
    cs = sensor.c()
    _check(lib.lgs_debug_tile_lists_batch(_ptr(workspace, torch.uint8, None, "workspace"), ctypes.byref(cs), frames, N,
                                          max_keys, _ptr(keys_d), _ptr(vals_d), ctypes.byref(rp), _ptr(rects),
                                          _stream(stream)),
           "lgs_debug_tile_lists")
    nt = frames * ((H + LGS_TILE_H - 1) // LGS_TILE_H) * ((W + LGS_TILE_W - 1) // LGS_TILE_W)
    off = rp.value - workspace.data_ptr()
    ranges = workspace[off:off + 8 * nt].cpu().numpy().view(np.uint32).reshape(nt, 2).copy()
    keys = keys_d[:K].cpu().numpy().view(np.uint64).copy()
    vals = vals_d[:K].cpu().numpy().view(np.uint32).copy()
    return keys, vals, ranges, rects[:N * frames].cpu().numpy()


def lgs_debug_tile_lists_batch(workspace, sensor: Sensor, frames: int, N: int, max_keys: int, stream=None):
    """Test-only: the sorted lists of a batched forward (see lgs_debug_tile_lists)."""
    return lgs_debug_tile_lists(workspace, sensor, N, max_keys, stream, frames=frames)


def lgs_debug_segmented_sort(keys, vals, seg_ranges, stream=None):
    """Test-only: sorts every segment of (keys int32-as-u32, vals int32-as-u32) CUDA tensors in place by
    (key, val); seg_ranges int32 [n_segments, 2] = [start, end)."""
    import torch
    lib = _load()
    n = keys.numel()
    tk, tv = torch.empty_like(keys), torch.empty_like(vals)
    _check(lib.lgs_debug_segmented_sort(_ptr(keys, torch.int32, None, "keys"), _ptr(vals, torch.int32, n, "vals"),
                                        _ptr(tk), _ptr(tv), _ptr(seg_ranges, torch.int32, None, "seg_ranges"),
                                        seg_ranges.numel() // 2, _stream(stream)),
           "lgs_debug_segmented_sort")
    (stream if stream is not None else torch.cuda.current_stream()).synchronize()


def lgs_debug_set_pdl(enabled: bool) -> None:
    """Test-only: False launches every kernel in plain stream order (no programmatic dependent launch)."""
    lib = _load()
    lib.lgs_debug_set_pdl.restype = ctypes.c_int
    _check(lib.lgs_debug_set_pdl(ctypes.c_int(int(bool(enabled)))), "lgs_debug_set_pdl")


# ---- map management ---------------------------------------------------------------------------
class _CCover(ctypes.Structure):
    _fields_ = [("axis_a", ctypes.c_int32), ("axis_b", ctypes.c_int32), ("origin_a", ctypes.c_float),
                ("origin_b", ctypes.c_float), ("cell", ctypes.c_float), ("dim_a", ctypes.c_int32), ("dim_b", ctypes.c_int32),
                ("alpha_min", ctypes.c_float), ("kappa", ctypes.c_float), ("q_cover", ctypes.c_float),
                ("s_max", ctypes.c_float), ("max_removed", ctypes.c_int64)]


def _ws(nbytes, device):
    import torch
    return torch.empty(max(int(nbytes), 256), dtype=torch.uint8, device=device)


def _alloc_on(stream):
    """Context in which torch allocates (and zero-fills) on the stream the kernels of the call will run on.  A tensor made
    on torch's current stream and used only on another one could be handed out again by the caching allocator, once it
    is dropped here, while those kernels still run; its zero fill would also race with them."""
    import torch
    return torch.cuda.stream(stream if stream is not None else torch.cuda.current_stream())


def lgs_manage_workspace_bytes(N: int) -> int:
    lib = _load()
    lib.lgs_manage_workspace_bytes.restype = ctypes.c_size_t
    return int(lib.lgs_manage_workspace_bytes(ctypes.c_int64(N)))


def lgs_cover_workspace_bytes(N: int, dim_a: int, dim_b: int) -> int:
    lib = _load()
    lib.lgs_cover_workspace_bytes.restype = ctypes.c_size_t
    return int(lib.lgs_cover_workspace_bytes(ctypes.c_int64(N), ctypes.c_int32(dim_a), ctypes.c_int32(dim_b)))


def lgs_control_score(sigma, res, bounds, weights=(0.55, 0.30, 0.15), eps: float = 1e-12, out=None, stream=None):
    """Eq. 9 (include/lgs.h).  bounds = ((lo_l, hi_l), (lo_c, hi_c), (lo_r, hi_r)).  Returns c [N]."""
    import torch
    lib = _load()
    N = int(res.numel())
    with _alloc_on(stream):
        c = torch.empty(N, dtype=torch.float32, device=res.device) if out is None else out
    b = (ctypes.c_float * 6)(*[float(x) for pair in bounds for x in pair])
    w = (ctypes.c_float * 3)(*[float(x) for x in weights])
    lib.lgs_control_score.restype = ctypes.c_int
    lib.lgs_control_score.argtypes = [ctypes.c_int64, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p,
                                      ctypes.c_float, ctypes.c_void_p, ctypes.c_void_p]
    _check(lib.lgs_control_score(N, _ptr(sigma, torch.float32, 3 * N, "sigma"), _ptr(res, torch.float32, N, "res"),
                                 ctypes.cast(b, ctypes.c_void_p), ctypes.cast(w, ctypes.c_void_p), eps,
                                 _ptr(c, torch.float32, N, "c"), _stream(stream)), "lgs_control_score")
    return c


def lgs_quantile(x, q: float, out=None, workspace=None, stream=None):
    """Q_q(x): device float tensor [1] holding the k-th smallest, k = clip(ceil(q N), 1, N)."""
    import torch
    lib = _load()
    N = int(x.numel())
    with _alloc_on(stream):
        out = torch.zeros(1, dtype=torch.float32, device=x.device) if out is None else out
        ws = _ws(lgs_manage_workspace_bytes(N), x.device) if workspace is None else workspace
    lib.lgs_quantile.restype = ctypes.c_int
    lib.lgs_quantile.argtypes = [ctypes.c_int64, ctypes.c_void_p, ctypes.c_double, ctypes.c_void_p, ctypes.c_void_p,
                                 ctypes.c_size_t, ctypes.c_void_p]
    _check(lib.lgs_quantile(N, _ptr(x, torch.float32, N, "x"), float(q), _ptr(out, torch.float32, 1, "out"),
                            _ptr(ws, torch.uint8, None, "workspace"), ws.numel(), _stream(stream)), "lgs_quantile")
    return out


def lgs_split(N: int, c, thr, alpha_min: float, max_splits: int, shift: float, shrink: float, mean, quat, log_scale,
              opacity, scale=None, m=None, v=None, flags_out=None, n_new=None, workspace=None, stream=None):
    """Adaptive split in place (include/lgs.h).  The parameter tensors hold >= N + max_splits rows, the first N valid.
    Returns n_new (device int64 tensor [1])."""
    import torch
    lib = _load()
    dev = mean.device
    with _alloc_on(stream):
        n_new = torch.zeros(1, dtype=torch.int64, device=dev) if n_new is None else n_new
        ws = _ws(lgs_manage_workspace_bytes(N), dev) if workspace is None else workspace
    cap_rows = N + max_splits
    for t, wdt, nm in ((mean, 3, "mean"), (quat, 4, "quat"), (log_scale, 2, "log_scale"), (opacity, 1, "opacity"),
                       (scale, 2, "scale"), (m, 10, "m"), (v, 10, "v")):
        if t is not None and t.numel() < wdt * cap_rows:
            raise ValueError("%s has room for %d rows, needs %d" % (nm, t.numel() // wdt, cap_rows))
    lib.lgs_split.restype = ctypes.c_int
    lib.lgs_split.argtypes = [ctypes.c_int64, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_float, ctypes.c_int64,
                              ctypes.c_float, ctypes.c_float] + [ctypes.c_void_p] * 9 + [ctypes.c_void_p, ctypes.c_size_t,
                                                                                       ctypes.c_void_p]
    _check(lib.lgs_split(N, _ptr(c, torch.float32, None, "c"), _ptr(thr, torch.float32, 1, "thr"), alpha_min, max_splits,
                         shift, shrink, _ptr(mean, torch.float32), _ptr(quat, torch.float32), _ptr(log_scale, torch.float32),
                         _ptr(opacity, torch.float32), _ptr(scale, torch.float32), _ptr(m, torch.float32),
                         _ptr(v, torch.float32), _ptr(flags_out, torch.uint8), ctypes.c_void_p(n_new.data_ptr()),
                         _ptr(ws, torch.uint8), ws.numel(), _stream(stream)), "lgs_split")
    return n_new


def lgs_cover_prune_pass(mean, quat, scale, log_scale, opacity, c, thr, axes, origin, cell: float, dims, alpha_min: float,
                         kappa: float, q_cover: float, s_max: float, max_removed: int, keep=None, n_removed=None,
                         workspace=None, stream=None):
    """One pass of planar cover-and-prune (include/lgs.h).  Updates scale / log_scale of the representatives in place;
    returns (keep uint8 [N], n_removed device int64 [1])."""
    import torch
    lib = _load()
    N = int(opacity.numel())
    dev = opacity.device
    with _alloc_on(stream):
        keep = torch.empty(N, dtype=torch.uint8, device=dev) if keep is None else keep
        n_removed = torch.zeros(1, dtype=torch.int64, device=dev) if n_removed is None else n_removed
        ws = _ws(lgs_cover_workspace_bytes(N, dims[0], dims[1]), dev) if workspace is None else workspace
    P = _CCover(int(axes[0]), int(axes[1]), float(origin[0]), float(origin[1]), float(cell), int(dims[0]), int(dims[1]),
                float(alpha_min), float(kappa), float(q_cover), float(s_max), int(max_removed))
    lib.lgs_cover_prune_pass.restype = ctypes.c_int
    lib.lgs_cover_prune_pass.argtypes = [ctypes.c_int64] + [ctypes.c_void_p] * 7 + [ctypes.POINTER(_CCover), ctypes.c_void_p,
                                                                                   ctypes.c_void_p, ctypes.c_void_p,
                                                                                   ctypes.c_size_t, ctypes.c_void_p]
    _check(lib.lgs_cover_prune_pass(N, _ptr(mean, torch.float32, 3 * N), _ptr(quat, torch.float32, 4 * N),
                                    _ptr(scale, torch.float32, 2 * N), _ptr(log_scale, torch.float32, 2 * N),
                                    _ptr(opacity, torch.float32, N), _ptr(c, torch.float32, N), _ptr(thr, torch.float32, 1),
                                    ctypes.byref(P), _ptr(keep, torch.uint8, N), ctypes.c_void_p(n_removed.data_ptr()),
                                    _ptr(ws, torch.uint8), ws.numel(), _stream(stream)), "lgs_cover_prune_pass")
    return keep, n_removed


def lgs_compact(keep, mean, quat, log_scale, opacity, scale=None, m=None, v=None, stream=None):
    """Order-preserving compaction by keep flags (include/lgs.h).  Returns (n_out, [compacted tensors]); synchronises."""
    import torch
    lib = _load()
    N = int(opacity.numel())
    ins = [mean, quat, log_scale, opacity, scale, m, v]
    widths = [3, 4, 2, 1, 2, 10, 10]
    st = stream if stream is not None else torch.cuda.current_stream()
    with torch.cuda.stream(st):
        outs = [None if t is None else torch.empty_like(t) for t in ins]
        n_out = torch.zeros(1, dtype=torch.int64, device=opacity.device)
        ws = _ws(lgs_prune_workspace_bytes(N), opacity.device)
    pin = [None if t is None else _ptr(t, torch.float32, w * N, "in") for t, w in zip(ins, widths)]
    pout = [None if t is None else _ptr(t, torch.float32, w * N, "out") for t, w in zip(outs, widths)]
    lib.lgs_compact.restype = ctypes.c_int
    lib.lgs_compact.argtypes = [ctypes.c_int64] + [ctypes.c_void_p] * 16 + [ctypes.c_void_p, ctypes.c_size_t, ctypes.c_void_p]
    _check(lib.lgs_compact(N, _ptr(keep, torch.uint8, N, "keep"), *pin, *pout, ctypes.c_void_p(n_out.data_ptr()),
                           ctypes.c_void_p(ws.data_ptr()), ws.numel(), _stream(stream)), "lgs_compact")
    st.synchronize()
    return int(n_out.item()), [t for t in outs if t is not None]


LGS_MB_FFMA, LGS_MB_MUFU_EX2, LGS_MB_RED_F32, LGS_MB_RED_F32X4 = 0, 1, 2, 3


def lgs_microbench(which: int, scratch, param: int = 1, stream=None):
    """Runs one of the library's micro-benchmarks (include/lgs.h).  Returns (rate per second, ms of the best launch).
    Synchronises."""
    import torch
    lib = _load()
    lib.lgs_microbench.restype = ctypes.c_int
    lib.lgs_microbench.argtypes = [ctypes.c_int, ctypes.c_void_p, ctypes.c_size_t, ctypes.c_int,
                                   ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_float), ctypes.c_void_p]
    rate, ms = ctypes.c_double(0.0), ctypes.c_float(0.0)
    _check(lib.lgs_microbench(which, _ptr(scratch, torch.uint8, None, "scratch"), scratch.numel(), int(param),
                              ctypes.byref(rate), ctypes.byref(ms), _stream(stream)), "lgs_microbench")
    return float(rate.value), float(ms.value)


LGS_PROF_SLOTS = 8


def lgs_profile_enable(on: bool) -> None:
    lib = _load()
    lib.lgs_profile_enable.restype = ctypes.c_int
    _check(lib.lgs_profile_enable(ctypes.c_int(int(bool(on)))), "lgs_profile_enable")


def lgs_profile_slot_name(slot: int) -> str:
    lib = _load()
    lib.lgs_profile_slot_name.restype = ctypes.c_char_p
    return lib.lgs_profile_slot_name(ctypes.c_int(slot)).decode()


def lgs_profile_read(stream=None) -> dict:
    """{slot name: milliseconds} of the kernels launched since the last read. Synchronises."""
    lib = _load()
    lib.lgs_profile_slot_name.restype = ctypes.c_char_p
    ms = (ctypes.c_float * LGS_PROF_SLOTS)()
    _check(lib.lgs_profile_read(ms, _stream(stream)), "lgs_profile_read")
    out = {lib.lgs_profile_slot_name(k).decode(): float(ms[k]) for k in range(LGS_PROF_SLOTS - 1)}
    if ms[LGS_PROF_SLOTS - 1] > 0:
        out[lib.lgs_profile_slot_name(LGS_PROF_SLOTS - 1).decode()] = float(ms[LGS_PROF_SLOTS - 1])
    return out


class Rasterizer:
    """Owns the device buffers of one (N, H, W, max_keys) problem; every method is one C-ABI call."""

    def __init__(self, N: int, sensor, max_keys: int, device="cuda:0"):
        import torch
        self.sensor = sensor if isinstance(sensor, Sensor) else Sensor.of(sensor)
        self.N, self.max_keys = int(N), int(max_keys)
        H, W = self.sensor.H, self.sensor.W
        self.device = torch.device(device)
        nbytes = lgs_workspace_bytes(self.N, H, W, self.max_keys)
        if nbytes == 0:
            raise ValueError("bad problem size")
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        self.loss_workspace = torch.empty(lgs_loss_workspace_bytes(H, W), dtype=torch.uint8, device=self.device)
        f = dict(dtype=torch.float32, device=self.device)
        self.range = torch.empty((H, W), **f)
        self.alpha = torch.empty((H, W), **f)
        self.normal = torch.empty((3, H, W), **f)
        self.dL_drange = torch.empty((H, W), **f)
        self.dL_dalpha = torch.empty((H, W), **f)
        self.dL_dnormal = torch.empty((3, H, W), **f)
        self.loss5 = torch.zeros(5, **f)            # lgs_loss_mapping: L, L_depth, L_ng, L_ns, L_alpha
        self.loss = self.loss5[:4]                  # lgs_loss_range_normal: L, L_depth, L_ng, L_ns
        n = max(self.N, 1)
        self.g_mean = torch.zeros((n, 3), **f)[:self.N]
        self.g_quat = torch.zeros((n, 4), **f)[:self.N]
        self.g_scale = torch.zeros((n, 2), **f)[:self.N]
        self.g_opacity = torch.zeros((n,), **f)[:self.N]

    def set_pose(self, T_ws):
        self.sensor = Sensor(self.sensor.H, self.sensor.W, self.sensor.elev_min, self.sensor.elev_max,
                             self.sensor.r_min, self.sensor.r_max, np.asarray(T_ws, dtype=np.float32).reshape(3, 4))

    def forward(self, mean, quat, scale, opacity, stream=None):
        lgs_render_forward(mean, quat, scale, opacity, self.sensor, self.workspace, self.max_keys, self.range,
                           self.alpha, self.normal, stream)

    def loss_stage(self, target_range, target_normal=None, keep_mask=None, lambda_n=1.0, lambda_ng=0.05,
                   lambda_ns=0.01, detach_surf=False, stream=None):
        lgs_loss_range_normal(self.sensor, self.range, self.alpha, self.normal, target_range, target_normal, keep_mask,
                              lambda_n, lambda_ng, lambda_ns, detach_surf, self.loss_workspace, self.loss,
                              self.dL_drange, self.dL_dalpha, self.dL_dnormal, stream)

    def loss_mapping(self, target_range, target_normal=None, keep_mask=None, lambda_alpha=0.1, alpha_eps=1e-6,
                     lambda_n=1.0, lambda_ng=0.05, lambda_ns=0.01, detach_surf=False, stream=None):
        lgs_loss_mapping(self.sensor, self.range, self.alpha, self.normal, target_range, target_normal, keep_mask,
                         lambda_alpha, alpha_eps, lambda_n, lambda_ng, lambda_ns, detach_surf, self.loss_workspace,
                         self.loss5, self.dL_drange, self.dL_dalpha, self.dL_dnormal, stream)

    def backward(self, mean, quat, scale, opacity, dL_drange=None, dL_dalpha=None, dL_dnormal=None, accumulate=False,
                 stream=None):
        # no upstream given: the images written by loss_stage(); otherwise exactly what was passed
        # (dL_dalpha / dL_dnormal = None mean zero, as in the C ABI)
        if dL_drange is None:
            dL_drange, dL_dalpha, dL_dnormal = self.dL_drange, self.dL_dalpha, self.dL_dnormal
        lgs_render_backward(mean, quat, scale, opacity, self.sensor, self.workspace, self.max_keys,
                            dL_drange, dL_dalpha, dL_dnormal,
                            self.g_mean, self.g_quat, self.g_scale, self.g_opacity, accumulate, stream)

    def query(self, stream=None):
        return lgs_query(self.workspace, self.N, self.sensor.H, self.sensor.W, self.max_keys, stream)

    def tile_lists(self, stream=None):
        return lgs_debug_tile_lists(self.workspace, self.sensor, self.N, self.max_keys, stream)


class BatchRasterizer:
    """F keyframes against one shared map: owns the device buffers of one
    (N, F, H, W, max_keys) problem; forward / backward are ONE C-ABI call each for all frames, the loss stage is one
    call per frame (each frame has its own 1/|Omega| normalisation, R18)."""

    def __init__(self, N: int, sensors, max_keys: int, device="cuda:0"):
        import torch
        self.sensors = [sn if isinstance(sn, Sensor) else Sensor.of(sn) for sn in sensors]
        self.F = len(self.sensors)
        self.N, self.max_keys = int(N), int(max_keys)
        H, W = self.sensors[0].H, self.sensors[0].W
        self.device = torch.device(device)
        nbytes = lgs_workspace_bytes_batch(self.N, H, W, self.max_keys, self.F)
        if nbytes == 0:
            raise ValueError("bad problem size")
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        self.loss_workspace = [torch.empty(lgs_loss_workspace_bytes(H, W), dtype=torch.uint8, device=self.device)
                               for _ in range(self.F)]
        f = dict(dtype=torch.float32, device=self.device)
        F = self.F
        self.range = torch.empty((F, H, W), **f)
        self.alpha = torch.empty((F, H, W), **f)
        self.normal = torch.empty((F, 3, H, W), **f)
        self.dL_drange = torch.empty((F, H, W), **f)
        self.dL_dalpha = torch.empty((F, H, W), **f)
        self.dL_dnormal = torch.empty((F, 3, H, W), **f)
        self.loss5 = torch.zeros((F, 8), **f)       # per frame: L, L_depth, L_ng, L_ns, L_alpha (8 floats: 16-byte rows)
        n = max(self.N, 1)
        self.g_mean = torch.zeros((n, 3), **f)[:self.N]
        self.g_quat = torch.zeros((n, 4), **f)[:self.N]
        self.g_scale = torch.zeros((n, 2), **f)[:self.N]
        self.g_opacity = torch.zeros((n,), **f)[:self.N]

    def forward(self, mean, quat, scale, opacity, stream=None):
        lgs_render_forward_batch(mean, quat, scale, opacity, self.sensors, self.workspace, self.max_keys, self.range,
                                 self.alpha, self.normal, stream)

    def loss_stage(self, target_range, target_normal=None, keep_mask=None, lambda_n=1.0, lambda_ng=0.05,
                   lambda_ns=0.01, detach_surf=False, stream=None):
        """lgs_loss_range_normal per frame; target_range [F,H,W], target_normal [F,3,H,W] or None, keep_mask [F,H,W]."""
        for k in range(self.F):
            lgs_loss_range_normal(self.sensors[k], self.range[k], self.alpha[k], self.normal[k], target_range[k],
                                  None if target_normal is None else target_normal[k],
                                  None if keep_mask is None else keep_mask[k], lambda_n, lambda_ng, lambda_ns,
                                  detach_surf, self.loss_workspace[k], self.loss5[k, :4], self.dL_drange[k],
                                  self.dL_dalpha[k], self.dL_dnormal[k], stream)

    def loss_mapping(self, target_range, target_normal=None, keep_mask=None, lambda_alpha=0.1, alpha_eps=1e-6,
                     lambda_n=1.0, lambda_ng=0.05, lambda_ns=0.01, detach_surf=False, stream=None):
        """target_range [F,H,W], target_normal [F,3,H,W] or None, keep_mask [F,H,W] uint8 or None."""
        for k in range(self.F):
            lgs_loss_mapping(self.sensors[k], self.range[k], self.alpha[k], self.normal[k], target_range[k],
                             None if target_normal is None else target_normal[k],
                             None if keep_mask is None else keep_mask[k], lambda_alpha, alpha_eps, lambda_n, lambda_ng,
                             lambda_ns, detach_surf, self.loss_workspace[k], self.loss5[k, :5], self.dL_drange[k],
                             self.dL_dalpha[k], self.dL_dnormal[k], stream)

    def backward(self, mean, quat, scale, opacity, dL_drange=None, dL_dalpha=None, dL_dnormal=None, accumulate=False,
                 stream=None):
        if dL_drange is None:
            dL_drange, dL_dalpha, dL_dnormal = self.dL_drange, self.dL_dalpha, self.dL_dnormal
        lgs_render_backward_batch(mean, quat, scale, opacity, self.sensors, self.workspace, self.max_keys, dL_drange,
                                  dL_dalpha, dL_dnormal, self.g_mean, self.g_quat, self.g_scale, self.g_opacity,
                                  accumulate, stream)

    def query(self, stream=None):
        return lgs_query(self.workspace, self.N, self.sensors[0].H, self.sensors[0].W, self.max_keys, stream)

    def tile_lists(self, stream=None):
        return lgs_debug_tile_lists(self.workspace, self.sensors[0], self.N, self.max_keys, stream, frames=self.F)
