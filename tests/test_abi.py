"""CPU-side checks of the boundary: liblgs.so loads without a GPU and exports every entry point that
include/lgs.h declares; the binding exposes the same names; argument errors are refused before any CUDA
call; the product path has no CPU fallback (it raises without the library / a CUDA tensor)."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "lgs.h")


def _declared():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = re.findall(r"\b(lgs_[a-z0-9_]+)\s*\(", src)
    return sorted(set(names))


@pytest.fixture(scope="module")
def lib():
    from paper_2607_04127_b200 import build
    return ctypes.CDLL(build.build())


def test_every_declared_symbol_is_exported(lib):
    names = _declared()
    assert {"lgs_render_forward", "lgs_render_backward", "lgs_loss_range_normal", "lgs_query",
            "lgs_workspace_bytes"} <= set(names)
    for n in names:
        assert hasattr(lib, n), "include/lgs.h declares %s but liblgs.so does not export it" % n


def test_binding_has_the_same_names():
    import paper_2607_04127_b200 as lgs
    for n in _declared():
        assert hasattr(lgs, n), "binding lacks %s" % n


def test_workspace_bytes_and_argument_validation(lib):
    lib.lgs_workspace_bytes.restype = ctypes.c_size_t
    lib.lgs_workspace_bytes.argtypes = [ctypes.c_int64, ctypes.c_int32, ctypes.c_int32, ctypes.c_int64]
    a = lib.lgs_workspace_bytes(300_000, 64, 1024, 500_000)
    b = lib.lgs_workspace_bytes(600_000, 64, 1024, 500_000)
    c = lib.lgs_workspace_bytes(300_000, 64, 1024, 1_000_000)
    assert 0 < a < b and a < c and a % 256 == 0
    assert lib.lgs_workspace_bytes(0, 1, 1, 0) > 0
    # out-of-range sizes are refused (0 bytes): N > 2^24, H/W > 32767, negative, max_keys >= 2^30
    for bad in ((-1, 64, 1024, 10), ((1 << 24) + 1, 64, 1024, 10), (10, 0, 1024, 10), (10, 64, 40000, 10),
                (10, 64, 1024, -1), (10, 64, 1024, 1 << 30)):
        assert lib.lgs_workspace_bytes(*bad) == 0, bad
    # NULL arguments are refused synchronously with LGS_ERR_INVALID_ARG (= 1), before any CUDA call
    lib.lgs_render_forward.restype = ctypes.c_int
    assert lib.lgs_render_forward(None, None, None, ctypes.c_size_t(0), ctypes.c_int64(0), None, None, None, None) == 1
    lib.lgs_render_backward.restype = ctypes.c_int
    assert lib.lgs_render_backward(None, None, None, ctypes.c_size_t(0), ctypes.c_int64(0), None, None, None, None,
                                   None, None, None, 0, None) == 1
    # batched calls: workspace grows with the number of frames, F outside [1, LGS_MAX_FRAMES] is refused, NULL arguments
    # are refused synchronously
    lib.lgs_workspace_bytes_batch.restype = ctypes.c_size_t
    lib.lgs_workspace_bytes_batch.argtypes = [ctypes.c_int64, ctypes.c_int32, ctypes.c_int32, ctypes.c_int64, ctypes.c_int32]
    w1 = lib.lgs_workspace_bytes_batch(300_000, 64, 1024, 500_000, 1)
    w8 = lib.lgs_workspace_bytes_batch(300_000, 64, 1024, 500_000, 8)
    assert w1 == a and w8 > w1 and w8 % 256 == 0
    assert lib.lgs_workspace_bytes_batch(300_000, 64, 1024, 500_000, 0) == 0
    assert lib.lgs_workspace_bytes_batch(300_000, 64, 1024, 500_000, 17) == 0
    lib.lgs_render_forward_batch.restype = ctypes.c_int
    assert lib.lgs_render_forward_batch(None, None, 4, None, ctypes.c_size_t(0), ctypes.c_int64(0), None, None, None, None) == 1
    lib.lgs_render_backward_batch.restype = ctypes.c_int
    assert lib.lgs_render_backward_batch(None, None, 4, None, ctypes.c_size_t(0), ctypes.c_int64(0), None, None, None, None,
                                         None, None, None, 0, None) == 1
    lib.lgs_version.restype = ctypes.c_char_p
    assert b"sm_100a" in lib.lgs_version()
    # loss workspace: counters + the per-column / per-row fp64 beam table
    lib.lgs_loss_workspace_bytes.restype = ctypes.c_size_t
    lib.lgs_loss_workspace_bytes.argtypes = [ctypes.c_int32, ctypes.c_int32]
    assert lib.lgs_loss_workspace_bytes(64, 1024) == 256 + (2 * 1024 + 2 * 64) * 8 + (64 * 1024 // 256) * 8
    assert lib.lgs_loss_workspace_bytes(0, 1024) == 0 and lib.lgs_loss_workspace_bytes(64, -1) == 0


def test_no_cpu_fallback():
    """Host tensors are refused: the binding marshals device pointers only and never computes."""
    torch = pytest.importorskip("torch")
    import paper_2607_04127_b200 as lgs
    from workloads import make_tiny
    w = make_tiny()
    cpu = [torch.from_numpy(np.ascontiguousarray(x)) for x in (w.mean, w.quat, w.scale, w.opacity)]
    S = w.sensors[0]
    ws = torch.zeros(1 << 20, dtype=torch.uint8)
    out = torch.zeros((S.H, S.W))
    with pytest.raises(Exception):
        lgs.lgs_render_forward(*cpu, S, ws, 1024, out, out.clone(), None)


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2607_04127_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in txt.replace("the oracle", "").replace("oracle's", "").lower() or \
                    not re.search(r"^\s*(import|from)\s+oracle|#include\s+\".*oracle", txt, flags=re.M), f
