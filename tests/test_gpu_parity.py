"""GPU parity tests: the CUDA path (through the C ABI) against the fp64 oracle, element by
element, on the same seeded inputs.  Tolerances are north_star's: images 1e-4 relative
(+1e-6), gradients 1e-3 relative (+1e-6 absolute) per surfel and parameter group, sorted
tile lists bit-exact.  Pixels the oracle flags as fragile (a cut-off decided within
rounding distance) are excluded from image parity and carry zero
upstream gradient on both sides."""
import numpy as np
import pytest

import oracle
from workloads import (make_kitti, make_large_map, make_mapping_batch, make_newer_college, make_random_shell,
                       make_tiny, simulate_scan)
from workloads.generators import _pose, _rot_zyx

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


def _lgs():
    import paper_2607_04127_b200 as lgs
    return lgs


def _dev(x):
    return torch.from_numpy(np.ascontiguousarray(x)).to("cuda:0")


class Run:
    """One forward on the GPU + the oracle's forward on the same inputs."""

    def __init__(self, w, frame=0, max_keys=None, slack=1.25):
        lgs = _lgs()
        self.w, self.S = w, w.sensors[frame]
        self.params = [_dev(x) for x in (w.mean, w.quat, w.scale, w.opacity)]
        self.tl = oracle.tile_lists(w.mean, w.quat, w.scale, w.opacity, self.S)
        K = len(self.tl.keys)
        self.max_keys = int(K * slack) + 64 if max_keys is None else max_keys
        self.R = lgs.Rasterizer(w.N, self.S, self.max_keys)
        self.R.forward(*self.params)
        torch.cuda.synchronize()
        self.fo = oracle.render_forward(w.mean, w.quat, w.scale, w.opacity, self.S)
        self.ok = ~self.fo.fragile

    def check_images(self, max_fragile=0.005):       # fragile pixels must stay below 0.5 %
        fo, ok, R = self.fo, self.ok, self.R
        assert self.fo.stats["n_fragile"] < max_fragile * ok.size
        for name, a, b in (("range", R.range, fo.range), ("alpha", R.alpha, fo.alpha)):
            a = a.cpu().numpy().astype(np.float64)
            tol = 1e-4 * np.abs(b) + 1e-6
            bad = (np.abs(a - b) > tol) & ok
            assert not bad.any(), "%s: %d pixels out of tolerance, worst %.3g tol-units" % (
                name, bad.sum(), (np.abs(a - b) / tol)[ok].max())
        n = R.normal.cpu().numpy().astype(np.float64)
        tol = 1e-4 * np.maximum(np.linalg.norm(fo.normal, axis=0), fo.alpha) + 1e-6
        bad = (np.linalg.norm(n - fo.normal, axis=0) > tol) & ok
        assert not bad.any(), "normal: %d pixels out of tolerance" % bad.sum()
        nv, nk, nc, ovf = R.query()
        assert not ovf and nk == len(self.tl.keys) and nv == int((self.tl.rects[:, 1] > 0).sum())
        # contributing pairs: identical outside fragile pixels
        assert abs(nc - fo.stats["I_c"]) <= 4 * fo.stats["n_fragile"]

    def check_lists(self):
        keys, vals, ranges, rects = self.R.tile_lists()
        tl = self.tl
        assert np.array_equal(rects, tl.rects), "rects differ for %d surfels" % (rects != tl.rects).any(1).sum()
        assert np.array_equal(ranges, tl.tile_ranges)
        assert np.array_equal(keys, tl.keys) and np.array_equal(vals, tl.vals)

    def check_backward(self, gD, gA, gN, stress=False):
        """gD/gA/gN: fp32 upstream images (zero at fragile pixels); the same arrays go to both sides."""
        w, S, R = self.w, self.S, self.R
        gm, gq, gs, go, cond = oracle.render_backward(w.mean, w.quat, w.scale, w.opacity, S, gD, gA, gN,
                                                      with_cond=True)
        R.backward(*self.params, _dev(gD), None if gA is None else _dev(gA), None if gN is None else _dev(gN))
        torch.cuda.synchronize()
        worst = {}
        for k, (name, a, b) in enumerate((("g_mean", R.g_mean, gm), ("g_quat", R.g_quat, gq), ("g_scale", R.g_scale, gs),
                                          ("g_opacity", R.g_opacity[:, None], go[:, None]))):
            a = a.cpu().numpy().astype(np.float64)
            assert np.isfinite(a).all()
            err = np.linalg.norm(a - b, axis=1)
            tol = 1e-3 * np.linalg.norm(b, axis=1) + 1e-6
            if stress:
                # O(1) random-sign upstream: the per-surfel sums cancel heavily, so the strict form is
                # only required of 99.8 % of the surfels; every surfel must satisfy the backward-error
                # form: the first-order effect (cond, from the oracle) of a relative error of
                # 1e-5 / |d.n| in every evaluated alpha, ~10 x what fp32 delivers
                assert (err > tol).mean() < 2e-3, "%s: %d strict violations" % (name, (err > tol).sum())
                tol = tol + 1e-5 * cond[:, k]
            bad = err > tol
            worst[name] = float((err / tol).max()) if len(err) else 0.0
            assert not bad.any(), "%s: %d surfels out of tolerance (worst %.3g tol-units)" % (name, bad.sum(), worst[name])
            culled = self.tl.rects[:, 1] == 0
            assert not a[culled].any()
        return worst

    def loss_upstream(self, seed=0):
        """Oracle loss stage on the oracle's render -> fp32 upstream images, zeroed on fragile pixels."""
        w, S, fo = self.w, self.S, self.fo
        if w.scene is not None:
            tgt, tn = simulate_scan(w.scene, S, w.scan_seed)
        else:
            tgt = oracle.render_forward(w.perturbed_mean, w.quat, w.scale, w.opacity, S).range.astype(np.float32)
            tn = None
        lr = oracle.loss_range_normal(S, fo.range, fo.alpha, fo.normal, tgt, tn, None, **w.lambdas)
        keep = self.ok & ~lr.sign_fragile
        gD = (lr.gD * keep).astype(np.float32)
        gN = (lr.gN * keep).astype(np.float32)
        return gD, None, gN, tgt, tn


def _cases():
    return {
        "tiny": lambda: make_tiny(),
        "ragged_seam": lambda: make_random_shell(21, 1500, 40, 200, s_lo=0.3, s_hi=1.5, r_lo=5.0,
                                                 pose=_pose(_rot_zyx(3.0, 0.1, -0.2), [0.5, 0.2, -0.1])),
        "poles": lambda: make_random_shell(22, 3000, 64, 128, fov_deg=(-85, 85), s_lo=0.1, s_hi=1.0, r_lo=3.5),
        "scene30k": lambda: make_newer_college(n_surfels=30_000, H=64, W=512),
        "one_pixel_tall": lambda: make_random_shell(24, 500, 1, 300, fov_deg=(-1, 1), s_lo=0.1, s_hi=0.6),
        # 33 x 513 = 16,929 tiles: beyond the 8,192 tile counters the ranges kernel keeps in registers (re-read path)
        "many_tiles": lambda: make_random_shell(25, 3000, 132, 4100, s_lo=0.05, s_hi=0.5),
    }


@pytest.mark.parametrize("case", list(_cases().keys()))
def test_forward_lists_backward_parity(case):
    run = Run(_cases()[case]())
    run.check_lists()
    run.check_images()
    H, W = run.S.H, run.S.W
    # (a) the real loss-scale upstream (north_star's tolerance as stated)
    gD, gA, gN, _, _ = run.loss_upstream()
    run.check_backward(gD, gA, gN)
    # (b) stress: O(1) random-sign upstream on all three images
    rng = np.random.default_rng(1)
    ok = run.ok
    run.check_backward((rng.normal(size=(H, W)) * ok).astype(np.float32),
                       (rng.normal(size=(H, W)) * ok).astype(np.float32),
                       (rng.normal(size=(3, H, W)) * ok).astype(np.float32), stress=True)


def test_full_size_newer_college_parity():
    """BASELINE.json configs[1] at full size (64x1024, 300k surfels), the configuration bench.py times."""
    run = Run(make_newer_college())
    assert run.w.N == 300_000 and len(run.tl.keys) > 300_000
    run.check_lists()
    # 370 of 65,536 pixels (0.56 %) are fragile on this workload: the 150k facade surfels are seen at every incidence
    # down to grazing, where |d.n| sits near its cut-off and rho^2 near 9 for many beams at once (every other full-size
    # config stays below the survey's 0.5 %)
    run.check_images(max_fragile=0.006)
    gD, gA, gN, tgt, tn = run.loss_upstream()
    run.check_backward(gD, gA, gN)
    rng = np.random.default_rng(2)
    H, W = run.S.H, run.S.W
    run.check_backward((rng.normal(size=(H, W)) * run.ok).astype(np.float32), None,
                       (rng.normal(size=(3, H, W)) * run.ok).astype(np.float32), stress=True)


@pytest.mark.parametrize("maker,kw", [(make_newer_college, dict(n_surfels=30_000, H=64, W=512)),
                                      (make_newer_college, {}), (make_large_map, {})])
def test_loss_stage_parity(maker, kw):
    """lgs_loss_range_normal against the oracle's loss stage on the oracle's own render, at 64x512, at the graded
    64x1024 / 300k surfels and at 128x2048 / 4M surfels; dL/dD and dL/dN compared PER PIXEL."""
    w = maker(**kw)
    S = w.sensors[0]
    lgs = _lgs()
    fo = oracle.render_forward(w.mean, w.quat, w.scale, w.opacity, S)
    tgt, tn = simulate_scan(w.scene, S, w.scan_seed)
    rng = np.random.default_rng(5)
    mask = (rng.uniform(size=tgt.shape) > 0.1).astype(np.uint8)
    R = lgs.Rasterizer(w.N, S, 1024)
    r32, a32, n32 = fo.range.astype(np.float32), fo.alpha.astype(np.float32), fo.normal.astype(np.float32)
    R.range.copy_(_dev(r32)); R.alpha.copy_(_dev(a32)); R.normal.copy_(_dev(n32))
    for lam, detach, tnorm, km in (((1.0, 0.05, 0.01), False, tn, mask), ((0.7, 0.5, 0.9), False, tn, None),
                                   ((1.0, 0.05, 0.3), True, None, mask), ((0.0, 0.0, 0.0), False, None, None)):
        lr = oracle.loss_range_normal(S, r32, a32, n32, tgt, tnorm, km, *lam, detach_surf=detach)
        R.loss_stage(_dev(tgt), None if tnorm is None else _dev(tnorm), None if km is None else _dev(km), *lam,
                     detach_surf=detach)
        torch.cuda.synchronize()
        got = R.loss.cpu().numpy().astype(np.float64)
        ref = np.array([lr.loss, lr.L_depth, lr.L_ng, lr.L_ns])
        assert np.allclose(got, ref, rtol=1e-5, atol=1e-7), (got, ref)
        ok = ~lr.sign_fragile
        gD = R.dL_drange.cpu().numpy().astype(np.float64)
        gN = R.dL_dnormal.cpu().numpy().astype(np.float64)
        # per pixel: 1e-4 relative + 1e-6 of the image's largest entry (measured: <= 1e-5 relative, <= 1.1e-6 of the
        # largest entry at 128x2048; the N_surf path differentiates finite differences of X = D^ d, hence the floor)
        tol_D = 1e-4 * np.abs(lr.gD) + 1e-6 * (np.abs(lr.gD).max() + 1e-30)
        bad = (np.abs(gD - lr.gD) > tol_D) & ok
        assert not bad.any(), "dL/dD: %d pixels out of tolerance" % bad.sum()
        tol_N = 1e-4 * np.abs(lr.gN) + 1e-5 * (np.abs(lr.gN).max() + 1e-30)
        assert not (np.abs(gN - lr.gN) > tol_N).any()
        assert not R.dL_dalpha.any()
    # empty valid set
    R.loss_stage(_dev(np.zeros_like(tgt)), _dev(tn), None)
    torch.cuda.synchronize()
    assert not R.loss.any() and not R.dL_drange.any() and not R.dL_dnormal.any()


def test_segmented_radix_sort_standalone():
    """The hand-written per-tile radix sort on its own: every segment ordered by (key, value).  Segment lengths
    span empty, 1, one warp, every class boundary +-1 (bitonic 256, big class 1024, shared-memory capacity 4096) and the
    ping-pong path through global memory;
    duplicates exercise the tie-break by surfel index; bit patterns cover all four digits; one segment has a
    constant top byte and one a constant low byte (skipped passes, odd number of passes)."""
    lgs = _lgs()
    rng = np.random.default_rng(0)
    lens = [0, 1, 2, 31, 32, 33, 511, 512, 513, 4095, 4096, 4097, 8191, 20_000, 0, 7, 100_003, 3,
            255, 256, 257, 1023, 1024, 1025, 2047, 2048, 2049, 64, 65, 128, 129, 700, 1500, 3000]
    starts = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
    n = int(starts[-1])
    keys = rng.integers(0, 1 << 32, size=n, dtype=np.uint64).astype(np.uint32)
    for s, e in zip(starts[:-1], starts[1:]):
        if e - s > 3:
            keys[rng.integers(s, e, size=(e - s) // 3)] = keys[s]       # many duplicates inside a segment
    s3, e3 = starts[3], starts[4]; keys[s3:e3] = (keys[s3:e3] & np.uint32(0x00ffffff)) | np.uint32(0x41000000)
    s9, e9 = starts[9], starts[10]; keys[s9:e9] = (keys[s9:e9] & np.uint32(0x00ffffff)) | np.uint32(0x41000000)
    s13, e13 = starts[13], starts[14]; keys[s13:e13] = (keys[s13:e13] & np.uint32(0xffffff00)) | np.uint32(0x7f)
    vals = rng.permutation(1 << 24)[:n].astype(np.uint32)               # distinct ids, arbitrary input order
    ranges = np.stack([starts[:-1], starts[1:]], 1).astype(np.int32)
    k = _dev(keys.view(np.int32)); v = _dev(vals.view(np.int32))
    lgs.lgs_debug_segmented_sort(k, v, _dev(ranges))
    gk, gv = k.cpu().numpy().view(np.uint32), v.cpu().numpy().view(np.uint32)
    for s, e in zip(starts[:-1], starts[1:]):
        order = np.lexsort((vals[s:e], keys[s:e]))
        assert np.array_equal(gk[s:e], keys[s:e][order]), (s, e)
        assert np.array_equal(gv[s:e], vals[s:e][order]), (s, e)


def test_sort_long_runs_of_equal_range_keys():
    """Many surfels at ONE fp32 range in one tile (a sphere shell, a quantised map): the tie-break by surfel index is a
    cooperative bitonic pass for runs longer than 16 keys, not a single thread's insertion sort.  Segments: 4,096 and
    5,000 equal keys (shared-memory class / global-memory class), 20,000 keys of two values, 3,000 keys in runs of
    17-40, 600 equal keys (small class), a whole 50,000-key segment of one value; plus a rendered shell."""
    lgs = _lgs()
    rng = np.random.default_rng(3)
    segs = [np.full(4096, 0x41200000, np.uint32), np.full(5000, 0x41200000, np.uint32),
            rng.choice(np.array([0x40000000, 0x40000001], np.uint32), size=20_000),
            np.repeat(rng.integers(0, 1 << 32, size=120, dtype=np.uint64).astype(np.uint32), rng.integers(17, 41, size=120))[:3000],
            np.full(600, 0x3f800000, np.uint32), np.full(50_000, 0x42c80000, np.uint32),
            np.concatenate([np.full(1000, 7, np.uint32), rng.integers(0, 1 << 32, size=1500, dtype=np.uint64).astype(np.uint32),
                            np.full(1200, 0xfffffff0, np.uint32)])]
    for sg in segs:
        rng.shuffle(sg)
    lens = [len(x) for x in segs]
    starts = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
    keys = np.concatenate(segs)
    n = len(keys)
    vals = rng.permutation(1 << 24)[:n].astype(np.uint32)
    ranges = np.stack([starts[:-1], starts[1:]], 1).astype(np.int32)
    k = _dev(keys.view(np.int32)); v = _dev(vals.view(np.int32))
    lgs.lgs_debug_segmented_sort(k, v, _dev(ranges))
    gk, gv = k.cpu().numpy().view(np.uint32), v.cpu().numpy().view(np.uint32)
    for s, e in zip(starts[:-1], starts[1:]):
        order = np.lexsort((vals[s:e], keys[s:e]))
        assert np.array_equal(gk[s:e], keys[s:e][order]), (s, e)
        assert np.array_equal(gv[s:e], vals[s:e][order]), (s, e)
    # end to end: 6,000 surfels on a sphere of radius exactly 8 m around the sensor (every key identical), lists bit-exact
    # (pixels under surfels that share a key are fragile by definition -- the order decides -- so only the lists are compared)
    w = make_random_shell(31, 6000, 32, 128, fov_deg=(-60, 60), s_lo=0.3, s_hi=0.8, r_lo=8.0, r_hi=8.0)
    run = Run(w)
    assert len(np.unique(run.tl.keys & np.uint64(0xffffffff))) <= 8          # (fp32 rounding of |c|: a handful of values)
    assert np.bincount((run.tl.keys >> np.uint64(32)).astype(np.int64)).max() > 64
    run.check_lists()
    assert bool(torch.isfinite(run.R.range).all())


def test_edge_cases_empty_culled_overflow_accumulate():
    lgs = _lgs()
    w = make_tiny()
    S = w.sensors[0]
    H, W = S.H, S.W
    # N = 0
    R0 = lgs.Rasterizer(0, S, 16)
    e = [torch.empty((0, k), device="cuda:0") for k in (3, 4, 2)] + [torch.empty((0,), device="cuda:0")]
    R0.forward(*e)
    torch.cuda.synchronize()
    assert not R0.range.any() and not R0.alpha.any() and not R0.normal.any()
    assert R0.query() == (0, 0, 0, False)
    # everything culled (opacity below 1/255)
    p = [_dev(x) for x in (w.mean, w.quat, w.scale, np.full_like(w.opacity, 0.003))]
    R1 = lgs.Rasterizer(w.N, S, 64)
    R1.forward(*p)
    R1.backward(*p, torch.ones((H, W), device="cuda:0"), None, None)
    torch.cuda.synchronize()
    assert not R1.alpha.any() and not R1.g_mean.any() and R1.query()[:2] == (0, 0)
    # key overflow: reported, frame renders as zeros, gradients zero; retry with the reported size works
    p = [_dev(x) for x in (w.mean, w.quat, w.scale, w.opacity)]
    R2 = lgs.Rasterizer(w.N, S, 100)
    R2.forward(*p)
    R2.backward(*p, torch.ones((H, W), device="cuda:0"), None, None)
    torch.cuda.synchronize()
    nv, need, nc, ovf = R2.query()
    assert ovf and need > 100 and nc == 0 and not R2.alpha.any() and not R2.g_mean.any()
    R3 = lgs.Rasterizer(w.N, S, need)            # exactly the capacity needed
    R3.forward(*p)
    torch.cuda.synchronize()
    assert R3.query()[3] is False and R3.alpha.any()
    # accumulate = 1 adds, accumulate = 0 overwrites every row
    gD = torch.ones((H, W), device="cuda:0")
    R3.backward(*p, gD, None, None)
    torch.cuda.synchronize()
    g1 = [t.clone() for t in (R3.g_mean, R3.g_quat, R3.g_scale, R3.g_opacity)]
    R3.backward(*p, gD, None, None, accumulate=True)   # a second backward on the same forward is allowed
    torch.cuda.synchronize()
    for a, b in zip((R3.g_mean, R3.g_quat, R3.g_scale, R3.g_opacity), g1):
        # (the per-surfel sums are float atomics over up to hundreds of O(1) pairs that largely cancel under this
        # all-ones upstream: two passes agree to the order-of-summation noise, measured against the surfel's vector)
        a2, b2 = a.reshape(w.N, -1).double(), 2 * b.reshape(w.N, -1).double()
        err = (a2 - b2).norm(dim=1)
        assert bool((err <= 1e-3 * b2.norm(dim=1) + 1e-5 * float(b2.norm(dim=1).max())).all()), float(err.max())
    # bad arguments are refused synchronously
    with pytest.raises(lgs.LgsError):
        lgs.lgs_render_forward(*p, R3.sensor, R3.workspace[:1024], R3.max_keys, R3.range, R3.alpha, R3.normal)


def test_multi_pose_and_keep_mask_batch_accumulation():
    """configs[4] in miniature: several keyframes against one map, keep masks, gradients summed."""
    lgs = _lgs()
    w = make_mapping_batch(n_surfels=40_000, H=32, W=256, n_frames=3)
    p = [_dev(x) for x in (w.mean, w.quat, w.scale, w.opacity)]
    ref = [np.zeros((w.N, 3)), np.zeros((w.N, 4)), np.zeros((w.N, 2)), np.zeros((w.N,))]
    tls = [oracle.tile_lists(w.mean, w.quat, w.scale, w.opacity, S) for S in w.sensors]
    R = lgs.Rasterizer(w.N, w.sensors[0], max(len(t.keys) for t in tls) + 4096)
    ups = []
    for f, S in enumerate(w.sensors):
        fo = oracle.render_forward(w.mean, w.quat, w.scale, w.opacity, S)
        tgt, tn = simulate_scan(w.scene, S, w.scan_seed + f)
        lr = oracle.loss_range_normal(S, fo.range, fo.alpha, fo.normal, tgt, tn, w.keep_masks[f], **w.lambdas)
        keep = ~(fo.fragile | lr.sign_fragile)
        gD, gN = (lr.gD * keep).astype(np.float32), (lr.gN * keep).astype(np.float32)
        g = oracle.render_backward(w.mean, w.quat, w.scale, w.opacity, S, gD, None, gN)
        for a, b in zip(ref, g):
            a += b
        ups.append((gD, gN))

    def run_frame(f, accumulate):
        R.set_pose(w.sensors[f].T_ws)
        R.forward(*p)
        R.backward(*p, _dev(ups[f][0]), None, _dev(ups[f][1]), accumulate=accumulate)
        torch.cuda.synchronize()
        nv, nk, nc, ovf = R.query()
        assert not ovf and nk == len(tls[f].keys)

    # the frame-sharded driver of batch.py with one rank (two ranks: tests/test_batch_multirank.py, gloo)
    lgs.batch_gradients(run_frame, len(w.sensors), (R.g_mean, R.g_quat, R.g_scale, R.g_opacity))
    for a, b in zip((R.g_mean, R.g_quat, R.g_scale, R.g_opacity[:, None]), (ref[0], ref[1], ref[2], ref[3][:, None])):
        a = a.cpu().numpy().astype(np.float64)
        err = np.linalg.norm(a - b, axis=1)
        assert (err <= 1e-3 * np.linalg.norm(b, axis=1) + 1e-6).all()


@pytest.mark.parametrize("maker,kw", [(make_kitti, dict(n_surfels=200_000, n_poses=2)),
                                      (make_large_map, dict(n_surfels=400_000))])
def test_other_configs_scaled_down(maker, kw):
    """configs[2] and [3] at a fifth / tenth of their surfel count (full image size): images + lists."""
    w = maker(**kw)
    run = Run(w, frame=len(w.sensors) - 1)
    run.check_lists()
    run.check_images()
    gD, gA, gN, _, _ = run.loss_upstream()
    run.check_backward(gD, gA, gN)


@pytest.mark.parametrize("maker,frame", [(make_kitti, 9), (make_large_map, 0), (make_mapping_batch, 7)])
def test_other_configs_full_size(maker, frame):
    """configs[2], [3], [4] at BASELINE.json's full sizes (1M / 4M / 2M surfels; 4,096 / 8,192 / 2,048 tiles; lists of up
    to 2,264 / 7,183 / 47,502 keys, i.e. every class of the sort including the global-memory path): bit-exact lists,
    images and gradients of one frame against the oracle (bounded mode, a few seconds)."""
    w = maker()
    run = Run(w, frame=frame, slack=1.05)
    run.check_lists()
    # the 50-layer slabs of configs[4] put more decisions near a threshold (alpha G around 1/255 fifty times per beam):
    # 1.25 % of its pixels are fragile, against 0.1-0.6 % elsewhere
    run.check_images(max_fragile=0.02 if maker is make_mapping_batch else 0.005)
    gD, gA, gN, _, _ = run.loss_upstream()
    run.check_backward(gD, gA, gN)


def test_lists_far_from_the_origin():
    """A map and a pose ~2e5 m from the origin (UTM-style coordinates), range-gated and large enough (700k pairs) for
    the batched projection with its fp32 pre-cull: the pre-cull forms mu - t in fp64, so its error is relative to the
    range and not to the offset, and the lists stay those of the exact rule -- bit for bit the list reference's."""
    import dataclasses
    w = make_large_map(n_surfels=700_000)
    off = np.array([1.0e5, -2.0e5, 300.0])
    w.mean = (w.mean.astype(np.float64) + off).astype(np.float32)
    T = np.asarray(w.sensors[0].T_ws, dtype=np.float64).reshape(3, 4).copy()
    T[:, 3] += off
    w.sensors = [dataclasses.replace(w.sensors[0], T_ws=T.astype(np.float32))]
    run = Run(w)
    run.check_lists()
    nv, nk, _, ovf = run.R.query()
    assert not ovf and nk == len(run.tl.keys) and nk > 100_000 and nv < 0.5 * w.N    # most of the map is beyond r_max


def test_cuda_graph_capture_and_replay():
    """The whole step (forward + loss + backward) is capturable and replays to the same result."""
    lgs = _lgs()
    w = make_newer_college(n_surfels=30_000, H=64, W=512)
    S = w.sensors[0]
    p = [_dev(x) for x in (w.mean, w.quat, w.scale, w.opacity)]
    tgt, tn = simulate_scan(w.scene, S, w.scan_seed)
    tgt, tn = _dev(tgt), _dev(tn)
    R = lgs.Rasterizer(w.N, S, 100_000)

    def step():
        R.forward(*p)
        R.loss_stage(tgt, tn, None)
        R.backward(*p)

    step()
    torch.cuda.synchronize()
    ref = [t.clone() for t in (R.range, R.g_mean, R.g_opacity, R.loss)]
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        step()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            step()
    torch.cuda.synchronize()
    for t in (R.range, R.g_mean, R.g_opacity):
        t.zero_()
    g.replay()
    torch.cuda.synchronize()
    assert torch.equal(R.range, ref[0])
    assert torch.allclose(R.g_mean, ref[1], rtol=1e-4, atol=1e-7) and torch.allclose(R.loss, ref[3], rtol=1e-5)
