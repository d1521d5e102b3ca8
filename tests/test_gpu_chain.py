"""The GPU's OWN chain forward -> lgs_loss_mapping -> backward, nothing injected between the calls and no
synchronisation, against the oracle's chain render_forward -> loss -> render_backward (one mapping
iteration renders, compares and optimises in one chain).  This is the test that notices a cross-kernel ordering
error (programmatic dependent launches): a consumer that starts on half-written images or
upstream gradients produces gradients that differ from the oracle's.

Both sides get ONE keep_mask that drops the oracle's fragile pixels (a cut-off decided within rounding distance,
DESIGN.md section 6) and the pixels whose L1 sign is decided within the image tolerance (|D^ - D| < 2e-4 max(D, 1):
the GPU's D^ may differ from the oracle's by 1e-4 relative, so a smaller margin could flip the sign on one side).
Dropping a pixel from Omega_M also removes its 4-neighbours from Omega_S (Eq. 11's N_surf needs all four), so no
value computed from a dropped pixel's D^ reaches a gradient.  Tolerance: north_star's, per surfel and parameter
group, |dg| <= 1e-3 |g| + 1e-6."""
import numpy as np
import pytest

import oracle
from oracle import mapping_step as ms
from workloads import make_large_map, make_newer_college, simulate_scan

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

LAM_A, EPS_A = 0.1, 1e-6       # lambda_alpha, epsilon of Eq. 10 (R20)


def _lgs():
    import paper_2607_04127_b200 as lgs
    return lgs


def _dev(x):
    return torch.from_numpy(np.ascontiguousarray(x)).to("cuda:0")


def _oracle_chain(w, S):
    fo = oracle.render_forward(w.mean, w.quat, w.scale, w.opacity, S)
    tgt, tn = simulate_scan(w.scene, S, w.scan_seed)
    sign_fragile = np.abs(fo.range - tgt) < 2e-4 * np.maximum(tgt, 1.0)
    keep = (~(fo.fragile | sign_fragile)).astype(np.uint8)
    lr = oracle.loss_range_normal(S, fo.range, fo.alpha, fo.normal, tgt, tn, keep, **w.lambdas)
    La, gA = ms.loss_alpha(fo.alpha, tgt, keep, LAM_A, EPS_A)
    g = oracle.render_backward(w.mean, w.quat, w.scale, w.opacity, S, lr.gD, gA, lr.gN)
    loss = np.array([lr.loss + LAM_A * La, lr.L_depth, lr.L_ng, lr.L_ns, La])
    return tgt, tn, keep, loss, g


def _check(R, loss_ref, g_ref, what):
    got = R.loss5.cpu().numpy().astype(np.float64)
    assert np.allclose(got, loss_ref, rtol=2e-5, atol=1e-7), (what, got, loss_ref)
    for name, a, b in (("g_mean", R.g_mean, g_ref[0]), ("g_quat", R.g_quat, g_ref[1]), ("g_scale", R.g_scale, g_ref[2]),
                       ("g_opacity", R.g_opacity[:, None], g_ref[3][:, None])):
        a = a.cpu().numpy().astype(np.float64)
        assert np.isfinite(a).all()
        err = np.linalg.norm(a - b, axis=1)
        tol = 1e-3 * np.linalg.norm(b, axis=1) + 1e-6
        bad = err > tol
        assert not bad.any(), "%s %s: %d surfels out of tolerance (worst %.3g tol-units)" % (
            what, name, bad.sum(), (err / tol).max())


@pytest.mark.parametrize("maker", [make_newer_college, make_large_map])
def test_own_chain_eager_and_graph(maker):
    """configs[1] (the graded 64x1024 / 300k frame) and configs[3] (128x2048 / 4M) at full size."""
    lgs = _lgs()
    w = maker()
    S = w.sensors[0]
    tgt, tn, keep, loss_ref, g_ref = _oracle_chain(w, S)
    p = [_dev(x) for x in (w.mean, w.quat, w.scale, w.opacity)]
    tgt_d, tn_d, keep_d = _dev(tgt), _dev(tn), _dev(keep)
    K = len(oracle.tile_lists(w.mean, w.quat, w.scale, w.opacity, S).keys)
    R = lgs.Rasterizer(w.N, S, int(1.1 * K) + 1024)
    lam = w.lambdas
    stream = torch.cuda.Stream()

    def step():
        R.forward(*p, stream=stream)
        R.loss_mapping(tgt_d, tn_d, keep_d, LAM_A, EPS_A, lam["lambda_n"], lam["lambda_ng"], lam["lambda_ns"], False,
                       stream=stream)
        R.backward(*p, stream=stream)

    def poison():
        # whatever a consumer would read too early is garbage, not last step's (identical) values
        for t in (R.range, R.alpha, R.normal, R.dL_drange, R.dL_dalpha, R.dL_dnormal, R.g_mean, R.g_quat, R.g_scale,
                  R.g_opacity):
            t.fill_(float("nan"))

    stream.wait_stream(torch.cuda.current_stream())
    for rep in range(3):                       # eager: the three calls back to back on one stream, no sync between them
        with torch.cuda.stream(stream):
            poison()
            step()
        stream.synchronize()
        assert not R.query(stream)[3]
        _check(R, loss_ref, g_ref, "eager[%d]" % rep)
    eager = [t.clone() for t in (R.dL_drange, R.dL_dalpha, R.dL_dnormal, R.g_mean, R.g_quat, R.g_scale, R.g_opacity)]
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=stream):
        step()
    for rep in range(5):                       # replayed graph: launch gaps are at their smallest here
        with torch.cuda.stream(stream):
            poison()
            graph.replay()
        stream.synchronize()
        _check(R, loss_ref, g_ref, "graph[%d]" % rep)
        # replay against eager: only the order of float atomics may differ
        now = (R.dL_drange, R.dL_dalpha, R.dL_dnormal, R.g_mean, R.g_quat, R.g_scale, R.g_opacity)
        for k, (a, b) in enumerate(zip(now, eager)):
            if k < 3:
                assert torch.allclose(a, b, rtol=1e-4, atol=1e-10), ("upstream image", k, rep)
            else:
                a2, b2 = a.reshape(w.N, -1).double(), b.reshape(w.N, -1).double()
                err = (a2 - b2).norm(dim=1)
                assert bool((err <= 2e-4 * b2.norm(dim=1) + 2e-7).all()), ("gradient", k, rep, float(err.max()))


def test_results_do_not_depend_on_programmatic_dependent_launch():
    """The same chain with every kernel in plain stream order (lgs_debug_set_pdl(0)) and with the overlapped launches:
    a large image so that the loss and composite kernels take several waves."""
    lgs = _lgs()
    w = make_newer_college(n_surfels=400_000, H=128, W=2048)
    S = w.sensors[0]
    tgt, tn = simulate_scan(w.scene, S, w.scan_seed)
    p = [_dev(x) for x in (w.mean, w.quat, w.scale, w.opacity)]
    tgt_d, tn_d = _dev(tgt), _dev(tn)
    R = lgs.Rasterizer(w.N, S, 3_000_000)
    outs = {}
    try:
        for pdl in (False, True):
            lgs.lgs_debug_set_pdl(pdl)
            for rep in range(3):
                for t in (R.range, R.dL_drange, R.dL_dnormal, R.g_mean):
                    t.fill_(float("nan"))
                R.forward(*p)
                R.loss_mapping(tgt_d, tn_d, None, LAM_A, EPS_A)
                R.backward(*p)
                torch.cuda.synchronize()
                assert not R.query()[3]
                cur = [t.clone() for t in (R.range, R.alpha, R.normal, R.loss5, R.dL_drange, R.dL_dalpha, R.dL_dnormal,
                                           R.g_mean, R.g_quat, R.g_scale, R.g_opacity)]
                if pdl not in outs:
                    outs[pdl] = cur
                ref = outs[False]
                for k, (a, b) in enumerate(zip(cur, ref)):
                    if k < 3:
                        assert torch.equal(a, b), ("image", k, pdl, rep)       # the forward has no atomics on its images
                    elif k < 7:
                        assert torch.allclose(a, b, rtol=1e-4, atol=1e-10), ("loss / upstream", k, pdl, rep)
                    else:
                        a2, b2 = a.reshape(w.N, -1).double(), b.reshape(w.N, -1).double()
                        err = (a2 - b2).norm(dim=1)
                        assert bool((err <= 2e-4 * b2.norm(dim=1) + 2e-7).all()), ("gradient", k, pdl, rep)
    finally:
        lgs.lgs_debug_set_pdl(True)


def test_scan_to_range_image_then_loss_back_to_back():
    """lgs_scan_to_range_image writes the loss stage's targets; the loss call follows it immediately on the same stream
    (its first kernel is launched with programmatic stream serialisation and reads only the targets)."""
    lgs = _lgs()
    w = make_newer_college(n_surfels=100_000, H=128, W=2048)
    S = w.sensors[0]
    tgt, tn = simulate_scan(w.scene, S, w.scan_seed)
    H, W = S.H, S.W
    jj, ii = np.meshgrid(np.arange(H), np.arange(W), indexing="ij")
    phi = -np.pi + (ii + 0.5) * (2 * np.pi / W)
    eM, em = float(np.float32(S.elev_max)), float(np.float32(S.elev_min))
    th = eM - (jj + 0.5) * ((eM - em) / H)
    dirs = np.stack([np.cos(th) * np.cos(phi), np.cos(th) * np.sin(phi), np.sin(th)], -1)
    pts = _dev((dirs * tgt[..., None]).reshape(-1, 3).astype(np.float32))
    nrm = _dev(np.ascontiguousarray(tn.reshape(3, -1).T))
    p = [_dev(x) for x in (w.mean, w.quat, w.scale, w.opacity)]
    R = lgs.Rasterizer(w.N, S, 1_500_000)
    R.forward(*p)
    torch.cuda.synchronize()
    zbuf = torch.empty(8 * H * W, dtype=torch.uint8, device="cuda:0")
    img, img_n = torch.empty((H, W), device="cuda:0"), torch.empty((3, H, W), device="cuda:0")
    # reference: the two calls separated by a synchronisation
    lgs.lgs_scan_to_range_image(pts, nrm, R.sensor, zbuf, img, img_n)
    torch.cuda.synchronize()
    R.loss_mapping(img, img_n, None, LAM_A, EPS_A)
    torch.cuda.synchronize()
    ref = [t.clone() for t in (R.loss5, R.dL_drange, R.dL_dalpha, R.dL_dnormal)]
    assert float(ref[0][0]) > 0
    for rep in range(5):
        img.fill_(float("nan")); img_n.fill_(float("nan"))
        for t in (R.dL_drange, R.dL_dalpha, R.dL_dnormal):
            t.fill_(float("nan"))
        lgs.lgs_scan_to_range_image(pts, nrm, R.sensor, zbuf, img, img_n)
        R.loss_mapping(img, img_n, None, LAM_A, EPS_A)
        torch.cuda.synchronize()
        for a, b in zip((R.loss5, R.dL_drange, R.dL_dalpha, R.dL_dnormal), ref):
            assert torch.allclose(a, b, rtol=1e-5, atol=1e-10), rep


def test_two_loss_calls_back_to_back_on_one_workspace():
    """include/lgs.h promises plain stream order for lgs_loss_*: two calls in a row that share the loss workspace and
    the gradient images need nothing between them.  The first kernel of a loss call is launched with programmatic
    stream serialisation and can become resident while the previous call's gradient kernel still runs; it therefore
    may only read the caller's inputs before its griddepcontrol.wait (it used to clear dL/dD and the loss counters
    there, under the feet of the previous call).  Both losses and the gradient images left by the second call are
    compared with the same sequence in plain stream order (lgs_debug_set_pdl(0)); 256x4096 pixels = 4,096 CTAs
    (three and a half waves), so the last CTAs of the first call's gradient kernel are still busy when the second
    call's first kernel arrives.  The loss outputs are poisoned before every round: a loss that is never written (the
    last-block counter reset under the first call's feet) shows up as NaN."""
    lgs = _lgs()
    from helpers import make_sensor
    S = make_sensor(256, 4096)
    sensor = lgs.Sensor.of(S)
    H, W = S.H, S.W
    rng = np.random.default_rng(77)

    def images(seed_shift):
        r = rng.uniform(2.0, 60.0, (H, W)).astype(np.float32)
        t = (r + rng.normal(0, 0.3, (H, W))).astype(np.float32)
        t[rng.uniform(size=(H, W)) < 0.2] = 0.0
        n = rng.normal(size=(3, H, W)); n /= np.linalg.norm(n, axis=0, keepdims=True)
        tn = rng.normal(size=(3, H, W)); tn /= np.linalg.norm(tn, axis=0, keepdims=True)
        tn[:, rng.uniform(size=(H, W)) < 0.3] = 0.0
        a = rng.uniform(0.1, 1.0, (H, W)).astype(np.float32)
        return [_dev(x) for x in (r, a, n.astype(np.float32), t, tn.astype(np.float32))]

    A, B = images(0), images(1)
    lws = torch.empty(lgs.lgs_loss_workspace_bytes(H, W), dtype=torch.uint8, device="cuda:0")
    gD = torch.empty((H, W), device="cuda:0"); gA = torch.empty((H, W), device="cuda:0")
    gN = torch.empty((3, H, W), device="cuda:0")
    lossA = torch.zeros(4, device="cuda:0"); lossB = torch.zeros(4, device="cuda:0")

    def run():
        lossA.fill_(float("nan")); lossB.fill_(float("nan"))
        for (r, a, n, t, tn), out in ((A, lossA), (B, lossB)):
            lgs.lgs_loss_range_normal(sensor, r, a, n, t, tn, None, 1.0, 0.05, 0.01, False, lws, out, gD, gA, gN)
        torch.cuda.synchronize()
        return lossA.cpu().numpy().copy(), lossB.cpu().numpy().copy(), gD.cpu().numpy().copy(), gN.cpu().numpy().copy()

    lgs.lgs_debug_set_pdl(0)
    try:
        refA, refB, ref_gD, ref_gN = run()
    finally:
        lgs.lgs_debug_set_pdl(1)
    assert refA[0] > 0 and refB[0] > 0 and abs(refA[0] - refB[0]) > 1e-6
    for it in range(25):
        gotA, gotB, got_gD, got_gN = run()
        assert np.allclose(gotA, refA, rtol=1e-6, atol=0), (it, gotA, refA)
        assert np.allclose(gotB, refB, rtol=1e-6, atol=0), (it, gotB, refB)
        # dL/dD is a sum of a handful of float atomics per pixel (order varies); dL/dN has one writer per pixel
        assert np.allclose(got_gD, ref_gD, rtol=1e-5, atol=1e-9 + 1e-6 * np.abs(ref_gD).max())
        assert np.array_equal(got_gN, ref_gN)
