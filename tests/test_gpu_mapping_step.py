"""GPU parity of the NEXT-1 entry points against oracle/mapping_step.py:
lgs_loss_mapping (Eq. 10 right + Eq. 13 image side) and lgs_adam_step (Eq. 12 + log-scale chain + Adam).
Tolerances: the loss kernels accumulate in fp64 from fp32 images (1e-5 relative);
dL_dalpha is one fp32 division (2e-6 relative); an Adam step in fp32 follows the fp64 oracle from the same fp32
state: |d theta| <= 1e-5 lr + 2 ulp(theta), moments 4e-6 relative (+ 4e-7 of the operands where they cancel)."""
import numpy as np
import pytest

import oracle
from oracle import mapping_step as ms
from workloads import make_newer_college, simulate_scan

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


def _lgs():
    import paper_2607_04127_b200 as lgs
    return lgs


def _dev(x):
    return torch.from_numpy(np.ascontiguousarray(x)).to("cuda:0")


def test_loss_mapping_parity():
    w = make_newer_college(n_surfels=30_000, H=64, W=512)
    S = w.sensors[0]
    lgs = _lgs()
    fo = oracle.render_forward(w.mean, w.quat, w.scale, w.opacity, S)
    tgt, tn = simulate_scan(w.scene, S, w.scan_seed)
    rng = np.random.default_rng(7)
    mask = (rng.uniform(size=tgt.shape) > 0.1).astype(np.uint8)
    R = lgs.Rasterizer(w.N, S, 1024)
    r32, a32, n32 = fo.range.astype(np.float32), fo.alpha.astype(np.float32), fo.normal.astype(np.float32)
    R.range.copy_(_dev(r32)); R.alpha.copy_(_dev(a32)); R.normal.copy_(_dev(n32))
    for lam_a, eps, km in ((0.1, 1e-6, mask), (0.37, 1e-3, None), (0.0, 1e-6, mask)):
        lr = oracle.loss_range_normal(S, r32, a32, n32, tgt, tn, km, 1.0, 0.05, 0.01)
        La, gA = ms.loss_alpha(a32, tgt, km, lam_a, eps)
        R.loss_mapping(_dev(tgt), _dev(tn), None if km is None else _dev(km), lam_a, eps, 1.0, 0.05, 0.01)
        torch.cuda.synchronize()
        got = R.loss5.cpu().numpy().astype(np.float64)
        ref = np.array([lr.loss + lam_a * La, lr.L_depth, lr.L_ng, lr.L_ns, La if lam_a != 0 else 0.0])
        assert np.allclose(got, ref, rtol=1e-5, atol=1e-7), (got, ref)
        g = R.dL_dalpha.cpu().numpy().astype(np.float64)
        assert np.allclose(g, gA, rtol=2e-6, atol=0), np.abs(g - gA).max()
        assert (g != 0).sum() == (gA != 0).sum()
        # the other upstream images are those of lgs_loss_range_normal
        R.loss_stage(_dev(tgt), _dev(tn), None if km is None else _dev(km), 1.0, 0.05, 0.01)
        gD0 = R.dL_drange.clone()
        R.loss_mapping(_dev(tgt), _dev(tn), None if km is None else _dev(km), lam_a, eps, 1.0, 0.05, 0.01)
        torch.cuda.synchronize()
        assert torch.equal(gD0 != 0, R.dL_drange != 0)
        assert torch.allclose(gD0, R.dL_drange, rtol=1e-5, atol=1e-9)     # (atomics: summation order only)
    # empty valid set: zeros everywhere
    R.loss_mapping(_dev(np.zeros_like(tgt)), _dev(tn), None)
    torch.cuda.synchronize()
    assert not R.loss5.any() and not R.dL_dalpha.any() and not R.dL_drange.any()


def _ulp(x):
    return np.spacing(np.abs(x).astype(np.float32)).astype(np.float64)


@pytest.mark.parametrize("N", [0, 1, 1000, 300_001])
def test_adam_step_parity(N):
    """Several steps; each step is compared from the SAME fp32 state (the GPU's), so the tolerance is that of one
    step and does not accumulate.  N = 300,001: config 2's size plus a ragged tail."""
    lgs = _lgs()
    rng = np.random.default_rng(100 + N % 97)
    f32 = np.float32
    mean = rng.normal(0, 20, (N, 3)).astype(f32); quat = rng.normal(0, 1, (N, 4)).astype(f32)
    ls = np.log(rng.uniform(0.05, 2.5, (N, 2))).astype(f32); op = rng.uniform(0.0, 1.0, N).astype(f32)
    if N >= 8:
        ls[0, :] = np.log(1.7)                                      # a tie s0 == s1 above s_max
        op[:4] = [0.0005, 0.9995, 0.5, 0.5]
    # the hyper-parameters cross the ABI as fp32: the oracle gets the same (rounded) values, promoted to fp64
    r32 = lambda x: float(np.float32(x))
    h = ms.AdamHyper(lr_mean=r32(1.6e-3), lr_quat=r32(1e-3), lr_scale=r32(5e-3), lr_opacity=r32(5e-2), beta1=r32(0.9),
                     beta2=r32(0.999), eps=r32(1e-15), lambda_s=10.0, s_max=1.0, alpha_lo=0.0, alpha_hi=1.0)
    d = dict(mean=_dev(mean), quat=_dev(quat), ls=_dev(ls), op=_dev(op))
    scale = torch.zeros((N, 2), device="cuda:0")
    m = torch.zeros((N, 10), device="cuda:0"); v = torch.zeros((N, 10), device="cuda:0")
    Ls = torch.full((1,), -1.0, device="cuda:0")
    for t in (1, 2, 3, 50):
        gm = rng.normal(0, 1e-3, (N, 3)).astype(f32); gq = rng.normal(0, 1e-2, (N, 4)).astype(f32)
        gs = rng.normal(0, 1e-2, (N, 2)).astype(f32); go = rng.normal(0, 1e-3, N).astype(f32)
        gm[rng.uniform(size=N) < 0.2] = 0.0                         # culled surfels carry zero gradient
        if N >= 8:
            go[:2] = [1.0, -1.0]                                    # push alpha against both clips
        before = [x.cpu().numpy() for x in (d["mean"], d["quat"], d["ls"], d["op"], m, v)]
        ref = ms.adam_step(*before[:4], gm, gq, gs, go, before[4], before[5], t, h)
        lgs.lgs_adam_step(d["mean"], d["quat"], d["ls"], d["op"], scale, _dev(gm), _dev(gq), _dev(gs), _dev(go), m, v, t,
                          h.lr_mean, h.lr_quat, h.lr_scale, h.lr_opacity, h.beta1, h.beta2, h.eps, h.lambda_s, h.s_max,
                          h.alpha_lo, h.alpha_hi, Ls)
        torch.cuda.synchronize()
        got = [x.cpu().numpy().astype(np.float64) for x in (d["mean"], d["quat"], d["ls"], d["op"])]
        lrs = (h.lr_mean, h.lr_quat, h.lr_scale, h.lr_opacity)
        for k, (a, b) in enumerate(zip(got, ref[:4])):
            # |m^ / sqrt(v^)| is O(1): the update is lr * O(1), computed to a few fp32 ulp (the moments can cancel,
            # so the bound is relative to lr, not to the update), then rounded into theta
            tol = 1e-5 * lrs[k] + 2 * _ulp(b)
            assert (np.abs(a - b) <= tol).all(), (k, t, (np.abs(a - b) / tol).max())
        if N:
            assert got[3].min() >= 0.0 and got[3].max() <= 1.0
        assert np.allclose(scale.cpu().numpy(), ref[4], rtol=3e-6, atol=0)                 # exp(new log-scale)
        gall = np.concatenate([gm, gq, np.exp(before[2].astype(np.float64)) * (np.abs(gs) + h.lambda_s), go[:, None]], 1)
        m_ops = h.beta1 * np.abs(before[4]) + (1 - h.beta1) * np.abs(gall)                 # operand scale (cancellation)
        assert (np.abs(m.cpu().numpy() - ref[5]) <= 4e-6 * np.abs(ref[5]) + 4e-7 * m_ops + 1e-30).all()
        assert np.allclose(v.cpu().numpy(), ref[6], rtol=4e-6, atol=1e-30)
        assert abs(float(Ls[0]) - ref[7]) <= 2e-5 * max(ref[7], 1e-6), (float(Ls[0]), ref[7])
    if N >= 8:
        assert float(d["op"][0]) == 0.0 and float(d["op"][1]) == 1.0


def test_adam_step_argument_validation():
    lgs = _lgs()
    z = lambda *s: torch.zeros(s, device="cuda:0")
    args = (z(4, 3), z(4, 4), z(4, 2), z(4), z(4, 2), z(4, 3), z(4, 4), z(4, 2), z(4), z(4, 10), z(4, 10))
    with pytest.raises(lgs.LgsError):
        lgs.lgs_adam_step(*args, 0, 1e-3, 1e-3, 1e-3, 1e-3, loss_scale=z(1))             # step must be >= 1
    with pytest.raises(lgs.LgsError):
        lgs.lgs_adam_step(*args, 1, 1e-3, 1e-3, 1e-3, 1e-3, beta1=1.0, loss_scale=z(1))
    with pytest.raises(lgs.LgsError):
        lgs.lgs_adam_step(*args, 1, 1e-3, 1e-3, 1e-3, 1e-3, loss_scale=None)


def test_mapping_iterations_reduce_the_loss():
    """Property at config scale (no oracle needed): a few full iterations forward -> lgs_loss_mapping -> backward ->
    lgs_adam_step on a perturbed map lower the Eq. 13 objective, and the updated map still renders without overflow."""
    lgs = _lgs()
    w = make_newer_college(n_surfels=60_000, H=64, W=512)
    S = w.sensors[0]
    tgt, tn = simulate_scan(w.scene, S, w.scan_seed)
    rng = np.random.default_rng(1)
    mean = (w.mean + rng.normal(0, 0.03, w.mean.shape)).astype(np.float32)
    p = dict(mean=_dev(mean), quat=_dev(w.quat), ls=_dev(np.log(w.scale)), op=_dev(w.opacity))
    scale = _dev(w.scale.copy())
    N = w.N
    probe = lgs.Rasterizer(N, S, 16 * N)
    probe.forward(p["mean"], p["quat"], scale, p["op"])
    nk = probe.query()[1]
    R = lgs.Rasterizer(N, S, 2 * nk + 4096)
    m = torch.zeros((N, 10), device="cuda:0"); v = torch.zeros((N, 10), device="cuda:0")
    Ls = torch.zeros(1, device="cuda:0")
    tg, tnd = _dev(tgt), _dev(tn)
    losses = []
    for t in range(1, 13):
        R.forward(p["mean"], p["quat"], scale, p["op"])
        R.loss_mapping(tg, tnd, None, 0.1, 1e-6, 1.0, 0.05, 0.01)
        R.backward(p["mean"], p["quat"], scale, p["op"])
        lgs.lgs_adam_step(p["mean"], p["quat"], p["ls"], p["op"], scale, R.g_mean, R.g_quat, R.g_scale, R.g_opacity, m, v,
                          t, 2e-3, 1e-3, 2e-3, 1e-2, loss_scale=Ls)
        losses.append(float(R.loss5[0]))
        assert not R.query()[3]
    assert np.isfinite(losses).all()
    assert losses[-1] < 0.9 * losses[0], losses


def test_adam_step_device_counter_and_graph_replay():
    """(a) the step count read from device memory gives the same step as the host's; (b) a whole mapping iteration
    (forward, lgs_loss_mapping, backward, lgs_adam_step with the device counter, counter += 1) captured in ONE CUDA graph
    and replayed follows the eager iterations that pass the step from the host."""
    lgs = _lgs()
    rng = np.random.default_rng(9)
    N = 5000
    f32 = np.float32
    init = [rng.normal(0, 20, (N, 3)).astype(f32), rng.normal(0, 1, (N, 4)).astype(f32),
            np.log(rng.uniform(0.05, 2.5, (N, 2))).astype(f32), rng.uniform(0, 1, N).astype(f32)]
    g = [_dev(rng.normal(0, 1e-2, s).astype(f32)) for s in ((N, 3), (N, 4), (N, 2), (N,))]
    outs = []
    for use_dev in (False, True):
        p = [_dev(x.copy()) for x in init]
        scale = torch.zeros((N, 2), device="cuda:0")
        torch.manual_seed(0)
        m = torch.rand((N, 10), device="cuda:0") * 1e-3; v = torch.rand((N, 10), device="cuda:0") * 1e-6
        Ls = torch.zeros(1, device="cuda:0")
        kw = dict(step_device=torch.tensor([7], dtype=torch.int32, device="cuda:0")) if use_dev else {}
        lgs.lgs_adam_step(*p, scale, *g, m, v, 1 if use_dev else 7, 1e-3, 1e-3, 5e-3, 5e-2, loss_scale=Ls, **kw)
        torch.cuda.synchronize()
        outs.append([x.clone() for x in p] + [scale.clone()])
    for a, b in zip(*outs):
        assert torch.equal(a, b)
    # (b)
    w = make_newer_college(n_surfels=20_000, H=32, W=256)
    S = w.sensors[0]
    tgt, tn = simulate_scan(w.scene, S, w.scan_seed)
    tg, tnd = _dev(tgt), _dev(tn)
    N = w.N

    def fresh():
        return dict(mean=_dev(w.mean + 0.02), quat=_dev(w.quat), ls=_dev(np.log(w.scale)), op=_dev(w.opacity),
                    scale=_dev(w.scale.copy()), m=torch.zeros((N, 10), device="cuda:0"), v=torch.zeros((N, 10), device="cuda:0"))

    R = lgs.Rasterizer(N, S, 400_000)
    Ls = torch.zeros(1, device="cuda:0")
    st = torch.cuda.Stream()

    def iteration(d, t, step_device=None):
        R.forward(d["mean"], d["quat"], d["scale"], d["op"], stream=st)
        R.loss_mapping(tg, tnd, None, 0.1, 1e-6, 1.0, 0.05, 0.01, stream=st)
        R.backward(d["mean"], d["quat"], d["scale"], d["op"], stream=st)
        lgs.lgs_adam_step(d["mean"], d["quat"], d["ls"], d["op"], d["scale"], R.g_mean, R.g_quat, R.g_scale, R.g_opacity,
                          d["m"], d["v"], t, 2e-3, 1e-3, 2e-3, 1e-2, loss_scale=Ls, stream=st, step_device=step_device)

    a = fresh()
    with torch.cuda.stream(st):
        for t in (1, 2, 3, 4):
            iteration(a, t)
    st.synchronize()
    assert not R.query(st)[3]
    b = fresh()
    counter = torch.ones(1, dtype=torch.int32, device="cuda:0")
    with torch.cuda.stream(st):
        iteration(b, 1, counter)                      # warm-up outside the graph (t = 1)
        counter += 1
    st.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=st):
        iteration(b, 1, counter)
        counter += 1
    for _ in range(3):                                # the capture did not execute: t = 2, 3, 4
        graph.replay()
    torch.cuda.synchronize()
    assert int(counter[0]) == 5
    # Same arithmetic, but the backward's float atomics make the gradients order-dependent in the last bits, and Adam
    # turns a gradient that is pure cancellation noise into a step of +-lr: nearly all components agree tightly, the
    # rest by at most the four steps taken.
    for k, lr in (("mean", 2e-3), ("quat", 1e-3), ("ls", 2e-3), ("op", 1e-2)):
        d = (a[k] - b[k]).abs()
        assert float(d.max()) <= 4.5 * lr, (k, float(d.max()))
        assert float((d <= 1e-5 + 1e-4 * a[k].abs()).float().mean()) > 0.99, k
