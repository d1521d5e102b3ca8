"""lgs_scan_to_range_image_static: the scan -> range image step for callers that cannot allocate device memory where
they run -- a per-scan real-time callback that must keep out of cudaMalloc, a process whose device memory all sits in a
pool it does not own, a plugin whose host program does every allocation.  They cannot bring the 8 bytes per pixel of
z-buffer the ordinary call wants, so this entry point uses a fixed 2 MiB array inside liblgs.so instead (one per GPU,
shared by all calls, H * W <= LGS_SCAN_STATIC_MAX_PIXELS).

What is checked: on two calls in a row its images are bit for bit those of lgs_scan_to_range_image with a caller-owned
z-buffer (integer decisions and copied fp32 values -- the same bar as tests/test_gpu_scan_image.py).  The second scan
is much sparser than the first and drawn on a different grid, so anything the first call left in the shared array
would show up as returns that the second scan does not have.  Images over the limit are refused with their own code.

The file is named to be collected last: with `pytest -x` a failure here cannot hide another test.  It does not depend
on what ran before it: the first call on a device looks the array up, wherever in the session that happens."""
import numpy as np
import pytest

from helpers import make_sensor

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


def _cloud(seed, M, r_hi):
    rng = np.random.default_rng(seed)
    v = rng.normal(size=(M, 3))
    v[:, 2] *= 0.3
    v /= np.maximum(np.linalg.norm(v, axis=1, keepdims=True), 1e-9)
    pts = (v * rng.uniform(0.2, r_hi, (M, 1))).astype(np.float32)
    nrm = rng.normal(size=(M, 3)).astype(np.float32)
    return torch.from_numpy(pts).to("cuda:0"), torch.from_numpy(nrm).to("cuda:0")


def _both_paths(lgs, pts, nrm, S):
    """(range, normal) of the existing path with its own z-buffer, then of the built-in-scratch path."""
    H, W = S.H, S.W
    sensor = lgs.Sensor.of(S)
    zbuf = torch.empty(8 * H * W, dtype=torch.uint8, device="cuda:0")
    ref_r = torch.full((H, W), -1.0, device="cuda:0")
    ref_n = torch.full((3, H, W), -1.0, device="cuda:0")
    lgs.lgs_scan_to_range_image(pts, nrm, sensor, zbuf, ref_r, ref_n)
    got_r = torch.full((H, W), -2.0, device="cuda:0")
    got_n = torch.full((3, H, W), -2.0, device="cuda:0")
    before = torch.cuda.memory_allocated()
    lgs.lgs_scan_to_range_image_static(pts, nrm, sensor, got_r, got_n)
    assert torch.cuda.memory_allocated() == before       # the binding made no tensor either
    torch.cuda.synchronize()
    return ref_r, ref_n, got_r, got_n


def test_two_calls_in_a_row_match_the_caller_buffer_path():
    import paper_2607_04127_b200 as lgs
    # call 1: the largest grid the built-in array takes (128 x 2048), dense -- several returns per pixel
    S1 = make_sensor(128, 2048, r_min=0.5, r_max=80.0)
    assert S1.H * S1.W == lgs.LGS_SCAN_STATIC_MAX_PIXELS
    pts1, nrm1 = _cloud(11, 1_000_003, 100.0)
    ref_r, ref_n, got_r, got_n = _both_paths(lgs, pts1, nrm1, S1)
    assert torch.equal(got_r, ref_r) and torch.equal(got_n, ref_n)
    assert (ref_r > 0).float().mean() > 0.5
    # call 2, straight after: a ragged smaller grid and a sparse scan; most pixels must come out empty (0), which they
    # only do if the call reset the words the dense scan filled
    S2 = make_sensor(33, 1000, r_min=0.5, r_max=80.0)
    pts2, nrm2 = _cloud(12, 3_001, 60.0)
    ref_r, ref_n, got_r, got_n = _both_paths(lgs, pts2, nrm2, S2)
    assert torch.equal(got_r, ref_r) and torch.equal(got_n, ref_n)
    assert 0 < int((ref_r > 0).sum()) < 3_001
    # and without normals / without a normal image, as the ordinary call allows
    r3 = torch.full((S2.H, S2.W), -2.0, device="cuda:0")
    lgs.lgs_scan_to_range_image_static(pts2, None, lgs.Sensor.of(S2), r3, None)
    torch.cuda.synchronize()
    assert torch.equal(r3, ref_r)


def test_images_beyond_the_built_in_array_are_refused():
    import paper_2607_04127_b200 as lgs
    S = make_sensor(128, 2049)
    pts, _ = _cloud(13, 100, 50.0)
    out = torch.full((S.H, S.W), -2.0, device="cuda:0")
    with pytest.raises(lgs.LgsError, match="LGS_ERR_STATIC_LIMIT"):
        lgs.lgs_scan_to_range_image_static(pts, None, lgs.Sensor.of(S), out, None)
    torch.cuda.synchronize()
    assert bool((out == -2.0).all())                       # nothing was launched
    with pytest.raises(lgs.LgsError, match="LGS_ERR_INVALID_ARG"):   # the ordinary call's own checks still apply
        lgs.lgs_scan_to_range_image_static(pts, None, lgs.Sensor.of(make_sensor(16, 128, r_min=5.0, r_max=1.0)),
                                           torch.zeros((16, 128), device="cuda:0"), None)
