"""Pins for the oracle's loss stage and backward pass.

The backward is pinned by fp64 central finite differences of scalars computed with
the oracle's *forward* only (north_star's named check), plus identities that any
correct gradient must satisfy (q . dL/dq = 0, Euler homogeneity of L_depth).
"""
import numpy as np
import pytest

import oracle
from helpers import beam, frame_quat, make_sensor, _rot_zyx


def small_scene(seed, n=16, H=8, W=32):
    rng = np.random.default_rng(seed)
    S = make_sensor(H, W, T_ws=np.concatenate([_rot_zyx(0.4, 0.05, -0.03), [[0.3], [-0.2], [0.1]]], 1), f64_pose=True)
    el = rng.uniform(np.deg2rad(-20), np.deg2rad(20), n)
    az = rng.uniform(-np.pi, np.pi, n)
    r = rng.uniform(4.0, 9.0, n)
    d = np.stack([np.cos(el) * np.cos(az), np.cos(el) * np.sin(az), np.sin(el)], 1)
    R, t = S.T_ws[:, :3], S.T_ws[:, 3]
    mean = (d * r[:, None]) @ R.T + t
    nrm = -d + 0.5 * rng.normal(size=(n, 3))
    quat = np.stack([frame_quat(R @ v, tu_hint=rng.normal(size=3))[0] for v in nrm]) * rng.uniform(0.5, 2.0, (n, 1))
    scale = rng.uniform(0.5, 1.2, (n, 2))
    opa = rng.uniform(0.3, 0.9, n)
    return S, mean, quat, scale, opa


def fd_grad(f, params, idx_list, h_rel=1e-6):
    """Central differences of scalar f(params) w.r.t. selected (array index, flat position)."""
    out = []
    for (ai, pos) in idx_list:
        p = [a.copy() for a in params]
        x0 = p[ai].flat[pos]
        h = h_rel * max(1.0, abs(x0))
        p[ai].flat[pos] = x0 + h
        fp = f(*p)
        p[ai].flat[pos] = x0 - h
        fm = f(*p)
        out.append((fp - fm) / (2 * h))
    return np.array(out)


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_backward_matches_finite_differences_of_linear_functional(seed):
    """F = sum_p gD D^ + gA A^ + gN . N^ with fixed random upstream images."""
    S, mean, quat, scale, opa = small_scene(seed)
    H, W = S.H, S.W
    rng = np.random.default_rng(100 + seed)
    base = oracle.render_forward(mean, quat, scale, opa, S, oracle.BRUTE)
    assert base.stats["I_c"] > 40
    keep = ~base.fragile
    gD = rng.normal(size=(H, W)) * keep
    gA = rng.normal(size=(H, W)) * keep
    gN = rng.normal(size=(3, H, W)) * keep

    def F(m, q, s, o):
        r = oracle.render_forward(m, q, s, o, S, oracle.BRUTE)
        assert np.array_equal(r.ncontrib, base.ncontrib), "a cut-off decision flipped inside the FD step"
        return float((gD * r.range).sum() + (gA * r.alpha).sum() + (gN * r.normal).sum())

    gm, gq, gs, go = oracle.render_backward(mean, quat, scale, opa, S, gD, gA, gN, oracle.BRUTE)
    params = [mean, quat, scale, opa]
    grads = [gm, gq, gs, go]
    idx = [(ai, pos) for ai in range(4) for pos in range(params[ai].size)]
    num = fd_grad(F, params, idx)
    ana = np.array([grads[ai].flat[pos] for ai, pos in idx])
    scale_ref = np.abs(ana).max()
    assert scale_ref > 1e-2
    assert np.allclose(num, ana, rtol=2e-6, atol=2e-7 * scale_ref), np.abs(num - ana).max()
    # normalisation of q: the gradient has no component along q
    assert np.abs((gq * quat).sum(1)).max() < 1e-12 * max(1.0, np.abs(gq).max())


def test_backward_bounded_equals_brute():
    S, mean, quat, scale, opa = small_scene(5, n=40, H=16, W=64)
    rng = np.random.default_rng(3)
    gD = rng.normal(size=(S.H, S.W)); gA = rng.normal(size=(S.H, S.W)); gN = rng.normal(size=(3, S.H, S.W))
    a = oracle.render_backward(mean, quat, scale, opa, S, gD, gA, gN, oracle.BRUTE)
    b = oracle.render_backward(mean, quat, scale, opa, S, gD, gA, gN, oracle.BOUNDED)
    for x, y in zip(a, b):
        assert np.allclose(x, y, rtol=1e-12, atol=1e-13)


def test_clamped_alpha_has_zero_opacity_gradient():
    S = make_sensor(8, 32)
    d0 = beam(S, 4, 10)
    q, _ = frame_quat(-d0)
    gD = np.zeros((8, 32)); gD[4, 10] = 1.0
    gm, gq, gs, go = oracle.render_backward((6 * d0)[None], q[None], [[0.8, 0.8]], [1.0], S, gD, None, None)
    assert go[0] == 0.0                      # min(0.99, alpha G) is flat above the clamp (reading R17)
    gm2, _, _, go2 = oracle.render_backward((6 * d0)[None], q[None], [[0.8, 0.8]], [0.5], S, gD, None, None)
    assert abs(go2[0] - 6.0) < 1e-9          # dD^/dalpha = G tau = 1 * 6 at the centre pixel
    assert abs(gm2[0] @ d0 - 0.5) < 1e-9     # dD^/dr = a for a fronto-parallel surfel moved along its beam


def _total_loss(S, target, tnormal, mask, lam):
    def L(m, q, s, o):
        r = oracle.render_forward(m, q, s, o, S, oracle.BRUTE)
        return oracle.loss_range_normal(S, r.range, r.alpha, r.normal, target, tnormal, mask, *lam).loss
    return L


@pytest.mark.parametrize("seed", [0, 3])
def test_full_chain_loss_gradient_matches_finite_differences(seed):
    """L = L_depth + lambda_n (lambda_ng L_ng + lambda_ns L_ns) end to end (Eq. 10, 11, 13)."""
    S, mean, quat, scale, opa = small_scene(seed, n=24, H=10, W=32)
    H, W = S.H, S.W
    rng = np.random.default_rng(7 + seed)
    base = oracle.render_forward(mean, quat, scale, opa, S, oracle.BRUTE)
    assert not base.fragile.any()
    target = base.range + np.where(rng.uniform(size=(H, W)) < 0.5, -0.3, 0.4)
    target = np.where(rng.uniform(size=(H, W)) < 0.1, 0.0, np.abs(target) + 0.05)   # some invalid pixels
    tn = rng.normal(size=(3, H, W))
    tn /= np.linalg.norm(tn, axis=0, keepdims=True)
    tn[:, rng.uniform(size=(H, W)) < 0.2] = 0.0                                      # some without N_g-icp
    mask = (rng.uniform(size=(H, W)) > 0.1).astype(np.uint8)
    lam = (1.0, 0.5, 0.3)
    lr = oracle.loss_range_normal(S, base.range, base.alpha, base.normal, target, tn, mask, *lam)
    assert lr.n_M > 100 and lr.n_N > 50 and lr.n_S > 20 and not lr.sign_fragile.any()
    assert abs(lr.loss - (lr.L_depth + lam[0] * (lam[1] * lr.L_ng + lam[2] * lr.L_ns))) < 1e-14
    grads = oracle.render_backward(mean, quat, scale, opa, S, lr.gD, lr.gA, lr.gN, oracle.BRUTE)
    L = _total_loss(S, target, tn, mask, lam)
    params = [mean, quat, scale, opa]
    rs = np.random.default_rng(1)
    idx = [(ai, int(pos)) for ai in range(4) for pos in rs.choice(params[ai].size, size=min(24, params[ai].size), replace=False)]
    num = fd_grad(L, params, idx)
    ana = np.array([grads[ai].flat[pos] for ai, pos in idx])
    assert np.abs(ana).max() > 1e-4
    assert np.allclose(num, ana, rtol=5e-6, atol=5e-8 * np.abs(ana).max()), np.abs(num - ana).max()
    # detaching N_surf changes the range gradient only
    lr2 = oracle.loss_range_normal(S, base.range, base.alpha, base.normal, target, tn, mask, *lam, detach_surf=True)
    assert np.array_equal(lr2.gN, lr.gN) and not np.array_equal(lr2.gD, lr.gD) and lr2.loss == lr.loss


def test_loss_stage_gradients_match_finite_differences_of_images():
    rng = np.random.default_rng(11)
    S = make_sensor(9, 24)
    H, W = S.H, S.W
    rngimg = rng.uniform(3, 8, (H, W))
    alpha = rng.uniform(0.2, 1, (H, W))
    nrm = rng.normal(size=(3, H, W)) * 0.5
    target = rngimg + rng.choice([-0.5, 0.5], size=(H, W))
    target[rng.uniform(size=(H, W)) < 0.15] = 0
    tn = rng.normal(size=(3, H, W)); tn /= np.linalg.norm(tn, axis=0)
    mask = (rng.uniform(size=(H, W)) > 0.1).astype(np.uint8)
    lam = (0.7, 0.4, 0.9)
    lr = oracle.loss_range_normal(S, rngimg, alpha, nrm, target, tn, mask, *lam)

    def L(r, n):
        return oracle.loss_range_normal(S, r, alpha, n, target, tn, mask, *lam).loss

    num = fd_grad(L, [rngimg, nrm], [(0, p) for p in range(H * W)] + [(1, p) for p in range(0, 3 * H * W, 5)])
    ana = np.concatenate([lr.gD.ravel(), lr.gN.ravel()[::5]])
    assert np.allclose(num, ana, rtol=1e-6, atol=1e-9)
    assert np.all(lr.gA == 0)
    # masks: invalid / dropped pixels carry no gradient and do not count
    bad = (target <= 0) | (mask == 0)
    assert lr.n_M == int((~bad).sum())
    assert np.all(lr.gN[:, bad] == 0)
    # empty valid set: everything is zero (reading R14)
    z = oracle.loss_range_normal(S, rngimg, alpha, nrm, np.zeros((H, W)), tn, mask, *lam)
    assert z.loss == 0 and not z.gD.any() and not z.gN.any()


def test_loss_depth_value_and_sign_convention():
    S = make_sensor(4, 8)
    r = np.full((4, 8), 5.0); t = np.full((4, 8), 5.0)
    t[0, 0] = 4.0; t[1, 1] = 7.0; t[2, 2] = 0.0
    lr = oracle.loss_range_normal(S, r, np.ones((4, 8)), np.zeros((3, 4, 8)), t, None, None, 1.0, 0.05, 0.0)
    assert lr.n_M == 31 and abs(lr.L_depth - 3.0 / 31) < 1e-15 and lr.L_ng == 0
    assert lr.gD[0, 0] == 1 / 31 and lr.gD[1, 1] == -1 / 31 and lr.gD[2, 2] == 0 and lr.gD[3, 3] == 0  # sign(0) = 0


def test_surface_normal_of_a_rendered_plane_is_the_plane_normal():
    """Finite differences of points on a plane lie in the plane, so N_surf is exactly the plane
    normal facing the sensor: L_ns = 0 when N^ is that unit normal; likewise L_ng."""
    S = make_sensor(12, 48, fov_deg=(-20, 25))
    jj, ii = np.meshgrid(np.arange(S.H), np.arange(S.W), indexing="ij")
    d = beam(S, jj, ii)
    n = np.array([0.2, -0.1, 1.0]); n /= np.linalg.norm(n)
    k = -3.0                                  # plane n.x = k below the sensor
    den = d @ n
    rng_img = np.where(den < -0.05, k / np.where(den < -0.05, den, 1), 0.0)
    nf = np.broadcast_to(n[:, None, None], (3, S.H, S.W)).copy()   # n.c = k < 0 -> n faces the sensor
    lr = oracle.loss_range_normal(S, rng_img, np.ones_like(rng_img), nf, rng_img, nf * (rng_img > 0), None, 1.0, 1.0, 1.0)
    assert lr.n_S > 50 and abs(lr.L_ns) < 1e-12 and abs(lr.L_ng) < 1e-12 and lr.L_depth == 0
    # flipping N^ gives a cosine loss of 2 on every pixel of Omega_S, normalised by |Omega_M| (Eq. 11)
    lr2 = oracle.loss_range_normal(S, rng_img, np.ones_like(rng_img), -nf, rng_img, None, None, 1.0, 1.0, 1.0)
    assert abs(lr2.L_ns - 2.0 * lr2.n_S / lr2.n_M) < 1e-12


def test_euler_homogeneity_of_depth_loss():
    """With t_ws = 0 and the gates off, L_depth is homogeneous of degree 1 in (mu, s, D):
    sum_i mu_i.g_mu_i + s_i.g_s_i + sum_p D_p dL/dD_p = L_depth, with dL/dD_p = -gD_p."""
    S, mean, quat, scale, opa = small_scene(2, n=30, H=12, W=48)
    S = make_sensor(S.H, S.W, T_ws=np.concatenate([_rot_zyx(0.4, 0.05, -0.03), np.zeros((3, 1))], 1), f64_pose=True)
    rng = np.random.default_rng(0)
    base = oracle.render_forward(mean, quat, scale, opa, S)
    target = np.abs(base.range + rng.normal(0, 0.3, base.range.shape)) + 0.1
    lr = oracle.loss_range_normal(S, base.range, base.alpha, base.normal, target, None, None, 1.0, 0.0, 0.0)
    gm, gq, gs, go = oracle.render_backward(mean, quat, scale, opa, S, lr.gD, None, None)
    lhs = (mean * gm).sum() + (scale * gs).sum() - (target * lr.gD).sum()
    assert lr.L_depth > 0.05 and abs(lhs - lr.L_depth) < 1e-10 * max(1, lr.L_depth)
