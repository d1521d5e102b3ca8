"""GPU parity of the one-launch batched keyframes (lgs_render_forward_batch /
lgs_render_backward_batch): F keyframes against one shared map, frame id folded into the tile id.

Oracle = the per-frame oracle, summed over the frames (reading R18: the sum of the per-frame losses, each
with its own 1/|Omega|).  Checked: the sorted lists of every frame bit for bit against the list reference, the images of
every frame element by element, the summed gradients per surfel and parameter group (north_star's tolerances), and that the
batch equals F single-frame calls with accumulate = 1 (images bit for bit)."""
import numpy as np
import pytest

import oracle
from workloads import make_kitti, make_mapping_batch, simulate_scan

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


def _lgs():
    import paper_2607_04127_b200 as lgs
    return lgs


def _dev(x):
    return torch.from_numpy(np.ascontiguousarray(x)).to("cuda:0")


def _oracle_batch(w, check_lists):
    """Per frame: list reference, forward, loss stage with the frame's keep mask, backward; gradients summed."""
    ref = [np.zeros((w.N, 3)), np.zeros((w.N, 4)), np.zeros((w.N, 2)), np.zeros((w.N,))]
    frames = []
    for f, S in enumerate(w.sensors):
        tl = oracle.tile_lists(w.mean, w.quat, w.scale, w.opacity, S) if check_lists else None
        fo = oracle.render_forward(w.mean, w.quat, w.scale, w.opacity, S)
        tgt, tn = simulate_scan(w.scene, S, w.scan_seed + f)
        km = None if w.keep_masks is None else w.keep_masks[f]
        lr = oracle.loss_range_normal(S, fo.range, fo.alpha, fo.normal, tgt, tn, km, **w.lambdas)
        keep = ~(fo.fragile | lr.sign_fragile)
        gD, gN = (lr.gD * keep).astype(np.float32), (lr.gN * keep).astype(np.float32)
        g = oracle.render_backward(w.mean, w.quat, w.scale, w.opacity, S, gD, None, gN)
        for a, b in zip(ref, g):
            a += b
        frames.append(dict(tl=tl, fo=fo, gD=gD, gN=gN))
    return ref, frames


def _check_images(B, frames, max_fragile):
    for f, fr in enumerate(frames):
        fo = fr["fo"]
        ok = ~fo.fragile
        assert fo.stats["n_fragile"] < max_fragile * ok.size
        for name, a, b in (("range", B.range[f], fo.range), ("alpha", B.alpha[f], fo.alpha)):
            a = a.cpu().numpy().astype(np.float64)
            tol = 1e-4 * np.abs(b) + 1e-6
            bad = (np.abs(a - b) > tol) & ok
            assert not bad.any(), "frame %d %s: %d pixels out of tolerance" % (f, name, bad.sum())
        n = B.normal[f].cpu().numpy().astype(np.float64)
        tol = 1e-4 * np.maximum(np.linalg.norm(fo.normal, axis=0), fo.alpha) + 1e-6
        bad = (np.linalg.norm(n - fo.normal, axis=0) > tol) & ok
        assert not bad.any(), "frame %d normal: %d pixels out of tolerance" % (f, bad.sum())


def _check_grads(B, ref, N):
    for name, a, b in (("g_mean", B.g_mean, ref[0]), ("g_quat", B.g_quat, ref[1]), ("g_scale", B.g_scale, ref[2]),
                       ("g_opacity", B.g_opacity[:, None], ref[3][:, None])):
        a = a.cpu().numpy().astype(np.float64)
        assert np.isfinite(a).all()
        err = np.linalg.norm(a - b, axis=1)
        tol = 1e-3 * np.linalg.norm(b, axis=1) + 1e-6
        assert (err <= tol).all(), "%s: %d surfels out of tolerance (worst %.3g tol-units)" % (
            name, (err > tol).sum(), float((err / tol).max()))


def test_batch_miniature_against_oracle_and_serial_calls():
    """3 keyframes, 40k surfels, 32x256: lists, images, summed gradients; equality with serial single-frame calls;
    accumulate = 1 on top of an existing buffer; overflow protocol."""
    lgs = _lgs()
    w = make_mapping_batch(n_surfels=40_000, H=32, W=256, n_frames=3)
    F = len(w.sensors)
    p = [_dev(x) for x in (w.mean, w.quat, w.scale, w.opacity)]
    ref, frames = _oracle_batch(w, check_lists=True)
    K = sum(len(fr["tl"].keys) for fr in frames)
    B = lgs.BatchRasterizer(w.N, w.sensors, K + 4096)
    B.forward(*p)
    torch.cuda.synchronize()
    nv, nk, nc, ovf = B.query()
    assert not ovf and nk == K
    assert nv == sum(int((fr["tl"].rects[:, 1] > 0).sum()) for fr in frames)
    # lists: frame f owns tile ids [f n_tiles, (f+1) n_tiles) and the key range that follows the earlier frames'
    keys, vals, ranges, rects = B.tile_lists()
    nt = len(frames[0]["tl"].tile_ranges)
    k0 = 0
    for f, fr in enumerate(frames):
        tl = fr["tl"]
        Kf = len(tl.keys)
        assert np.array_equal(rects[f * w.N:(f + 1) * w.N], tl.rects)
        assert np.array_equal(ranges[f * nt:(f + 1) * nt], tl.tile_ranges + np.uint32(k0))
        assert np.array_equal(keys[k0:k0 + Kf], tl.keys + (np.uint64(f * nt) << np.uint64(32)))
        assert np.array_equal(vals[k0:k0 + Kf], tl.vals)
        k0 += Kf
    # (the 50-layer slabs put alpha G near 1/255 on every layer, and in this 32x256 miniature a slab fills a large part
    # of the image: up to 3.6 % of a frame's pixels are fragile, against 1.25 % at full size)
    _check_images(B, frames, 0.05)
    # the batch equals F single-frame calls: images bit for bit
    R = lgs.Rasterizer(w.N, w.sensors[0], K + 4096)
    for f, S in enumerate(w.sensors):
        R.set_pose(S.T_ws)
        R.forward(*p)
        torch.cuda.synchronize()
        assert torch.equal(R.range, B.range[f]) and torch.equal(R.alpha, B.alpha[f]) and torch.equal(R.normal, B.normal[f])
    # backward with the oracle's upstream images of every frame, summed over the frames
    gD = _dev(np.stack([fr["gD"] for fr in frames]))
    gN = _dev(np.stack([fr["gN"] for fr in frames]))
    B.backward(*p, gD, None, gN)
    torch.cuda.synchronize()
    _check_grads(B, ref, w.N)
    culled = np.all([fr["tl"].rects[:, 1] == 0 for fr in frames], axis=0)
    assert not B.g_mean.cpu().numpy()[culled].any()
    # accumulate = 1 adds to what the buffers hold
    g1 = [t.clone() for t in (B.g_mean, B.g_quat, B.g_scale, B.g_opacity)]
    B.backward(*p, gD, None, gN, accumulate=True)
    torch.cuda.synchronize()
    for a, b in zip((B.g_mean, B.g_quat, B.g_scale, B.g_opacity), g1):
        a2, b2 = a.reshape(w.N, -1).double(), 2 * b.reshape(w.N, -1).double()
        err = (a2 - b2).norm(dim=1)
        assert bool((err <= 1e-3 * b2.norm(dim=1) + 1e-5 * float(b2.norm(dim=1).max())).all())
    # overflow: the batch renders as zeros and the query reports the capacity all frames need together
    B2 = lgs.BatchRasterizer(w.N, w.sensors, K // 2)
    B2.forward(*p)
    torch.cuda.synchronize()
    nv, nk2, nc, ovf = B2.query()
    assert ovf and nk2 == K and not B2.range.any() and not B2.alpha.any()
    B2.backward(*p, gD, None, gN)
    torch.cuda.synchronize()
    assert not B2.g_mean.any() and not B2.g_opacity.any()
    # bad arguments: frames whose grids differ, too many frames
    import dataclasses
    with pytest.raises(lgs.LgsError):
        bad = [B.sensors[0], dataclasses.replace(B.sensors[1], r_max=50.0)]
        lgs.lgs_render_forward_batch(*p, bad, B.workspace, B.max_keys, B.range[:2], B.alpha[:2], B.normal[:2])
    assert lgs.lgs_workspace_bytes_batch(w.N, 32, 256, K, lgs.LGS_MAX_FRAMES + 1) == 0


def test_batch_own_chain_with_loss_per_frame():
    """forward_batch -> lgs_loss_mapping per frame (its own keep mask and 1/|Omega|) -> backward_batch with nothing
    injected, against the same chain run as F single-frame calls with accumulate = 1."""
    lgs = _lgs()
    w = make_mapping_batch(n_surfels=40_000, H=32, W=256, n_frames=4)
    F = len(w.sensors)
    p = [_dev(x) for x in (w.mean, w.quat, w.scale, w.opacity)]
    scans = [simulate_scan(w.scene, S, w.scan_seed + f) for f, S in enumerate(w.sensors)]
    tgt = _dev(np.stack([s[0] for s in scans]))
    tn = _dev(np.stack([s[1] for s in scans]))
    keep = _dev(np.stack(w.keep_masks).astype(np.uint8))
    B = lgs.BatchRasterizer(w.N, w.sensors, 100_000)
    B.forward(*p)
    nk = B.query()[1]               # (overflow -> the capacity all frames need together -> retry)
    B = lgs.BatchRasterizer(w.N, w.sensors, nk + 1024)
    B.forward(*p)
    B.loss_mapping(tgt, tn, keep, 0.1, 1e-6, **w.lambdas)
    B.backward(*p)
    torch.cuda.synchronize()
    assert not B.query()[3]
    R = lgs.Rasterizer(w.N, w.sensors[0], nk + 1024)
    for f, S in enumerate(w.sensors):
        R.set_pose(S.T_ws)
        R.forward(*p)
        R.loss_mapping(tgt[f], tn[f], keep[f], 0.1, 1e-6, **w.lambdas)
        R.backward(*p, accumulate=(f > 0))
        torch.cuda.synchronize()
        assert torch.equal(R.loss5, B.loss5[f, :5])
        # (the N_surf term adds into the four neighbours' dL/dD with float atomics: last-bit order noise)
        assert torch.allclose(R.dL_drange, B.dL_drange[f], rtol=1e-5, atol=1e-9) and torch.equal(R.dL_dnormal, B.dL_dnormal[f])
    for a, b in zip((B.g_mean, B.g_quat, B.g_scale, B.g_opacity), (R.g_mean, R.g_quat, R.g_scale, R.g_opacity)):
        a2, b2 = a.reshape(w.N, -1).double(), b.reshape(w.N, -1).double()
        err = (a2 - b2).norm(dim=1)
        # (float atomics inside a frame: order-of-summation noise only)
        assert bool((err <= 2e-4 * b2.norm(dim=1) + 1e-6 * float(b2.norm(dim=1).max()) + 1e-9).all()), float(err.max())


def test_batch_full_size_config5():
    """BASELINE.json configs[4] at full size: 8 keyframes of 64x1024 against the shared 2M-surfel map with the dense
    slabs, keep masks, gradients of all 8 frames summed -- ONE forward and ONE backward call."""
    lgs = _lgs()
    w = make_mapping_batch()
    p = [_dev(x) for x in (w.mean, w.quat, w.scale, w.opacity)]
    ref, frames = _oracle_batch(w, check_lists=False)
    # size the key buffer with the documented protocol (overflow -> query -> retry)
    B = lgs.BatchRasterizer(w.N, w.sensors, 1 << 20)
    B.forward(*p)
    nv, nk, nc, ovf = B.query()
    assert ovf
    del B
    torch.cuda.empty_cache()
    B = lgs.BatchRasterizer(w.N, w.sensors, int(nk * 1.02) + 4096)
    B.forward(*p)
    torch.cuda.synchronize()
    nv, nk, nc, ovf = B.query()
    assert not ovf
    _check_images(B, frames, 0.02)
    assert abs(nc - sum(fr["fo"].stats["I_c"] for fr in frames)) <= 4 * sum(fr["fo"].stats["n_fragile"] for fr in frames)
    gD = _dev(np.stack([fr["gD"] for fr in frames]))
    gN = _dev(np.stack([fr["gN"] for fr in frames]))
    B.backward(*p, gD, None, gN)
    torch.cuda.synchronize()
    _check_grads(B, ref, w.N)


def test_kitti_ten_poses_full_size_serial_and_batched():
    """BASELINE.json configs[2] at full size: 64x2048, 1M surfels, ALL ten poses.  The gradients of the ten frames
    summed (accumulate = 1) against the summed oracle gradients -- once as ten single-frame calls, once as ONE batched
    call of ten frames; images of every pose element by element."""
    lgs = _lgs()
    w = make_kitti()
    assert len(w.sensors) == 10
    p = [_dev(x) for x in (w.mean, w.quat, w.scale, w.opacity)]
    ref, frames = _oracle_batch(w, check_lists=False)
    B = lgs.BatchRasterizer(w.N, w.sensors, 1 << 20)
    B.forward(*p)
    nk = B.query()[1]
    del B
    torch.cuda.empty_cache()
    B = lgs.BatchRasterizer(w.N, w.sensors, int(nk * 1.02) + 4096)
    B.forward(*p)
    torch.cuda.synchronize()
    assert not B.query()[3]
    _check_images(B, frames, 0.005)
    gD = _dev(np.stack([fr["gD"] for fr in frames]))
    gN = _dev(np.stack([fr["gN"] for fr in frames]))
    B.backward(*p, gD, None, gN)
    torch.cuda.synchronize()
    _check_grads(B, ref, w.N)
    # the same as ten single-frame calls with accumulate = 1
    R = lgs.Rasterizer(w.N, w.sensors[0], int(nk * 0.2) + 4096)
    for f, S in enumerate(w.sensors):
        R.set_pose(S.T_ws)
        R.forward(*p)
        R.backward(*p, gD[f], None, gN[f], accumulate=(f > 0))
        torch.cuda.synchronize()
        assert not R.query()[3]
        assert torch.equal(R.range, B.range[f]) and torch.equal(R.alpha, B.alpha[f])
    _check_grads(R, ref, w.N)
