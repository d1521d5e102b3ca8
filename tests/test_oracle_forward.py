"""Pins for the oracle's forward pass: closed forms, invariants, special cases.

Nothing here re-types the oracle's ray/plane code: expected values come from the angle
between beams (closed form), from algebraic compositing identities, or from symmetries.
"""
import numpy as np
import pytest

import oracle
from helpers import beam, frame_quat, make_sensor, quat_mul, quat_to_mat, _rot_zyx
from workloads import make_newer_college, make_random_shell, make_tiny


def _render(mean, quat, scale, opa, sensor, mode=oracle.BOUNDED):
    return oracle.render_forward(np.atleast_2d(mean), np.atleast_2d(quat), np.atleast_2d(scale), np.atleast_1d(opa),
                                 sensor, mode)


@pytest.mark.parametrize("mode", [oracle.BRUTE, oracle.BOUNDED])
@pytest.mark.parametrize("alpha0", [0.7, 1.0])
def test_single_fronto_parallel_surfel_closed_form(mode, alpha0):
    """north_star's named check.  c = r0 d0, n = -d0, s0 = s1 = s.  At any pixel with
    cos(gamma) = d.d0 > 0: tau = r0/cos(gamma), rho^2 = (r0 tan(gamma)/s)^2,
    a = min(.99, alpha0 exp(-rho^2/2)) if rho^2 <= 9 and a >= 1/255 else 0;
    D^ = a tau, A^ = a, N^ = -a d0."""
    S = make_sensor(32, 128)
    j0, i0, r0, s = 10, 37, 7.5, 0.4
    d0 = beam(S, j0, i0)
    q, _ = frame_quat(-d0)
    out = _render(r0 * d0, q, [s, s], alpha0, S, mode)
    jj, ii = np.meshgrid(np.arange(S.H), np.arange(S.W), indexing="ij")
    d = beam(S, jj, ii)
    cg = d @ d0
    tg2 = (1 - cg ** 2) / cg ** 2
    rho2 = r0 ** 2 * tg2 / s ** 2
    a = np.minimum(0.99, alpha0 * np.exp(-0.5 * rho2))
    a = np.where((cg > 0) & (rho2 <= 9) & (a >= 1 / 255), a, 0.0)
    safe = np.abs(rho2 - 9) > 1e-6
    assert np.allclose(out.alpha[safe], a[safe], rtol=1e-12, atol=1e-14)
    assert np.allclose(out.range[safe], (a * r0 / cg)[safe], rtol=1e-12, atol=1e-13)
    for k in range(3):
        assert np.allclose(out.normal[k][safe], (-a * d0[k])[safe], rtol=1e-12, atol=1e-14)
    # the centre pixel renders exactly the known range and opacity
    assert abs(out.alpha[j0, i0] - min(0.99, alpha0)) < 1e-14
    assert abs(out.range[j0, i0] - min(0.99, alpha0) * r0) < 1e-12
    assert (a > 0).sum() > 20 and out.stats["I_c"] == int((a > 0).sum())


def test_anisotropic_axes_assignment():
    """s0 scales the first column of R(q) (e_0 = in-plane major axis).
    With s0 >> s1 the footprint is elongated along t_u: closed form along each axis."""
    S = make_sensor(64, 256)
    j0, i0, r0 = 31, 128, 10.0
    d0 = beam(S, j0, i0)
    # t_u along +azimuth (horizontal), t_v vertical
    hint = np.cross([0, 0, 1.0], d0)
    q, R = frame_quat(-d0, tu_hint=hint)
    s0, s1 = 0.9, 0.15
    out = _render(r0 * d0, q, [s0, s1], 0.8, S)
    jj, ii = np.meshgrid(np.arange(S.H), np.arange(S.W), indexing="ij")
    d = beam(S, jj, ii)
    cg = d @ d0
    hit = (r0 / cg)[..., None] * d - r0 * d0
    u = hit @ R[:, 0] / s0
    v = hit @ R[:, 1] / s1
    rho2 = u * u + v * v
    a = np.where((cg > 0) & (rho2 <= 9) & (0.8 * np.exp(-0.5 * rho2) >= 1 / 255), 0.8 * np.exp(-0.5 * rho2), 0)
    safe = np.abs(rho2 - 9) > 1e-6
    assert np.allclose(out.alpha[safe], a[safe], atol=1e-12)
    cols = np.where(out.alpha[j0] > 0)[0]
    rows = np.where(out.alpha[:, i0] > 0)[0]
    dphi, dth = 2 * np.pi / S.W, np.deg2rad(45) / S.H
    assert len(cols) * dphi > 3 * len(rows) * dth  # wide in azimuth, thin in elevation


def test_two_coaxial_surfels_compositing_and_order():
    S = make_sensor(16, 64)
    j0, i0 = 8, 20
    d0 = beam(S, j0, i0)
    q, _ = frame_quat(-d0)
    r1, r2, a1, a2 = 5.0, 9.0, 0.6, 0.5
    for (ra, rb, aa, ab) in [(r1, r2, a1, a2), (r2, r1, a1, a2)]:
        out = _render(np.stack([ra * d0, rb * d0]), np.stack([q, q]), [[0.3, 0.3], [0.3, 0.3]], [aa, ab], S)
        # the nearer surfel composites first whatever its index
        (rn, an), (rf, af) = sorted([(ra, aa), (rb, ab)])
        assert abs(out.alpha[j0, i0] - (an + (1 - an) * af)) < 1e-14
        assert abs(out.range[j0, i0] - (an * rn + (1 - an) * af * rf)) < 1e-13
    # equal keys: ties break by ascending surfel index (reading R5)
    out = _render(np.stack([r1 * d0, r1 * d0]), np.stack([q, q]), [[0.3, 0.3], [0.3, 0.3]], [a1, a2], S)
    assert abs(out.alpha[j0, i0] - (a1 + (1 - a1) * a2)) < 1e-14


def test_early_stop_is_stop_before_apply():
    """Stack of coaxial surfels with a = 0.8: T_m * 0.2 < 1e-4 first holds at m = 5
    (0.2^5*... = 6.4e-5), so 5 are applied, the 6th is not: A^ = 1 - 0.2^5."""
    S = make_sensor(16, 64)
    j0, i0 = 5, 11
    d0 = beam(S, j0, i0)
    q, _ = frame_quat(-d0)
    n = 8
    mean = np.stack([(4.0 + k) * d0 for k in range(n)])
    out = _render(mean, np.tile(q, (n, 1)), np.full((n, 2), 0.2), np.full(n, 0.8), S)
    assert out.ncontrib[j0, i0] == 5
    assert abs(out.alpha[j0, i0] - (1 - 0.2 ** 5)) < 1e-14
    expected_D = sum(0.2 ** k * 0.8 * (4.0 + k) for k in range(5))
    assert abs(out.range[j0, i0] - expected_D) < 1e-12
    assert out.stats["n_stopped"] >= 1


def test_cutoffs_alpha_and_3sigma():
    S = make_sensor(16, 64)
    j0, i0 = 8, 30
    d0 = beam(S, j0, i0)
    q, _ = frame_quat(-d0)
    # opacity below 1/255: culled entirely
    out = _render(5 * d0, q, [0.3, 0.3], 0.0039, S)
    assert out.alpha.max() == 0 and out.stats["n_alive"] == 0
    # sensor inside the 3 sigma ball: culled
    out = _render(1.0 * d0, q, [0.4, 0.2], 0.9, S)
    assert out.stats["n_alive"] == 0
    # range gates act on the centre key
    Sg = make_sensor(16, 64, r_min=2.0, r_max=6.0)
    assert _render(7 * d0, q, [0.3, 0.3], 0.9, Sg).stats["n_alive"] == 0
    assert _render(1.5 * d0, q, [0.1, 0.1], 0.9, Sg).stats["n_alive"] == 0
    assert _render(5 * d0, q, [0.3, 0.3], 0.9, Sg).stats["n_alive"] == 1
    # back side of the surfel still renders; the normal faces the sensor
    qb, _ = frame_quat(d0)
    out = _render(5 * d0, qb, [0.3, 0.3], 0.9, S)
    assert abs(out.alpha[j0, i0] - 0.9) < 1e-14
    assert np.allclose(out.normal[:, j0, i0], -0.9 * d0, atol=1e-13)


def test_invariants_on_tiny():
    w = make_tiny()
    S = w.sensors[0]
    out = oracle.render_forward(w.mean, w.quat, w.scale, w.opacity, S, oracle.BOUNDED)
    A = out.alpha
    assert A.min() >= 0 and A.max() <= 1
    nn = np.linalg.norm(out.normal, axis=0)
    assert (nn <= A + 1e-12).all()
    has = A > 0
    rbar = out.range[has] / A[has]
    r = np.linalg.norm(w.mean.astype(np.float64), axis=1)
    smax = w.scale.max(1).astype(np.float64)
    assert rbar.min() >= (r - 3 * smax).min() - 1e-9 and rbar.max() <= (r + 3 * smax).max() + 1e-9
    assert out.stats["I_c"] == int(out.ncontrib.sum()) and out.stats["I_c"] <= out.stats["I_3sigma"]
    assert out.stats["n_fragile"] < 0.005 * A.size


@pytest.mark.parametrize("k", [1, 7, 100])
def test_seam_shift_invariance(k):
    """Yawing the pose by k*2pi/W shifts the images circularly by k columns (north_star's named check)."""
    w = make_random_shell(5, 600, 32, 128, s_lo=0.1, s_hi=0.6)
    S0 = make_sensor(32, 128, f64_pose=True)
    psi = k * 2 * np.pi / S0.W
    T = np.concatenate([_rot_zyx(psi, 0, 0), np.zeros((3, 1))], 1)
    S1 = make_sensor(32, 128, T_ws=T, f64_pose=True)
    a = oracle.render_forward(w.mean, w.quat, w.scale, w.opacity, S0)
    b = oracle.render_forward(w.mean, w.quat, w.scale, w.opacity, S1)
    # a world point at azimuth phi is seen at phi - psi: image moves by -k columns
    ok = ~(np.roll(a.fragile, -k, axis=1) | b.fragile)
    assert ok.mean() > 0.99
    for x, y in [(a.range, b.range), (a.alpha, b.alpha), (a.normal[2], b.normal[2])]:
        assert np.allclose(np.roll(x, -k, axis=1)[ok], y[ok], rtol=1e-9, atol=1e-10)
    # N^ is in the sensor frame: its horizontal part rotates with the pose
    nx = np.cos(psi) * a.normal[0] + np.sin(psi) * a.normal[1]
    assert np.allclose(np.roll(nx, -k, axis=1)[ok], b.normal[0][ok], rtol=1e-9, atol=1e-10)


def test_surfel_on_the_seam_is_mirror_symmetric():
    S = make_sensor(32, 128)
    c = np.array([-6.0, 0.0, 0.3])   # azimuth exactly pi: straddles columns W-1 | 0
    q, _ = frame_quat(-c)
    out = _render(c, q, [0.5, 0.5], 0.9, S)
    assert out.alpha[:, 0].max() > 0.5 and out.alpha[:, -1].max() > 0.5
    assert np.allclose(out.alpha, out.alpha[:, ::-1], atol=1e-12)
    assert np.allclose(out.range, out.range[:, ::-1], atol=1e-11)
    assert out.alpha[:, 40:90].max() == 0


def test_rigid_frame_independence():
    w = make_random_shell(9, 400, 24, 96)
    g = _rot_zyx(0.7, -0.3, 1.1)
    t = np.array([3.0, -2.0, 0.5])
    qg = np.array([np.sqrt(max(0, 1 + np.trace(g))) / 2, 0, 0, 0])
    qg[1:] = np.array([g[2, 1] - g[1, 2], g[0, 2] - g[2, 0], g[1, 0] - g[0, 1]]) / (4 * qg[0])
    assert np.allclose(quat_to_mat(qg), g)
    S0 = make_sensor(24, 96, f64_pose=True)
    S1 = make_sensor(24, 96, T_ws=np.concatenate([g, t[:, None]], 1), f64_pose=True)
    mean = w.mean.astype(np.float64)
    quat = w.quat.astype(np.float64)
    mean1 = mean @ g.T + t
    quat1 = np.stack([quat_mul(qg, q) for q in quat])
    a = oracle.render_forward(mean, quat, w.scale, w.opacity, S0)
    b = oracle.render_forward(mean1, quat1, w.scale, w.opacity, S1)
    ok = ~(a.fragile | b.fragile)
    for x, y in [(a.range, b.range), (a.alpha, b.alpha), (a.normal, b.normal)]:
        assert np.allclose(x[..., ok], y[..., ok], rtol=1e-9, atol=1e-10)


def test_reparametrisations_leave_the_image_unchanged():
    w = make_random_shell(11, 300, 24, 96)
    S = w.sensors[0]
    quat = w.quat.astype(np.float64)
    a = oracle.render_forward(w.mean, quat, w.scale, w.opacity, S)
    for q2 in (-quat, 3.7 * quat):
        b = oracle.render_forward(w.mean, q2, w.scale, w.opacity, S)
        assert np.allclose(a.range, b.range, atol=1e-10) and np.allclose(a.normal, b.normal, atol=1e-11)
    # swap (s0, s1) together with a quarter turn about the normal e_2
    qz = np.array([np.cos(np.pi / 4), 0, 0, np.sin(np.pi / 4)])
    q3 = np.stack([quat_mul(q, qz) for q in quat])
    b = oracle.render_forward(w.mean, q3, w.scale[:, ::-1], w.opacity, S)
    ok = ~(a.fragile | b.fragile)
    assert np.allclose(a.range[ok], b.range[ok], atol=1e-9) and np.allclose(a.alpha[ok], b.alpha[ok], atol=1e-10)


def test_bounded_equals_brute_bit_for_bit():
    w = make_tiny()
    S = w.sensors[0]
    a = oracle.render_forward(w.mean, w.quat, w.scale, w.opacity, S, oracle.BRUTE)
    b = oracle.render_forward(w.mean, w.quat, w.scale, w.opacity, S, oracle.BOUNDED)
    for x, y in [(a.range, b.range), (a.alpha, b.alpha), (a.normal, b.normal), (a.ncontrib, b.ncontrib),
                 (a.fragile, b.fragile)]:
        assert np.array_equal(x, y)
    # a 20k-surfel sub-sample of the graded scene, on a quarter-width image
    w = make_newer_college(n_surfels=20_000, H=32, W=256)
    S = w.sensors[0]
    a = oracle.render_forward(w.mean, w.quat, w.scale, w.opacity, S, oracle.BRUTE)
    b = oracle.render_forward(w.mean, w.quat, w.scale, w.opacity, S, oracle.BOUNDED)
    assert a.stats["I_c"] > 20_000
    for x, y in [(a.range, b.range), (a.alpha, b.alpha), (a.normal, b.normal), (a.ncontrib, b.ncontrib)]:
        assert np.array_equal(x, y)


def test_golden_paper_constants():
    """The only numbers the paper prints for this path: the loss weights."""
    import inspect
    import os
    vals = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "paper_constants.txt")) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if line:
                k, v = line.split("=")
                vals[k.strip()] = float(v)
    sig = inspect.signature(oracle.loss_range_normal)
    assert sig.parameters["lambda_n"].default == vals["lambda_n"]
    assert sig.parameters["lambda_ng"].default == vals["lambda_n_g"]
    assert sig.parameters["lambda_ns"].default == vals["lambda_n_s"]
