"""Pins of oracle/map_manage.py (control score Eq. 9, adaptive split, planar cover-and-prune;
PAPER.md:115-123, 158-166) against what the paper and the mathematics fix: closed cases worked by hand, numpy's own
sort / quantile / indexing as independent definitions, and invariants chosen so that a dropped term, a swapped axis, a
wrong tie rule or an off-by-one rank fails one of them."""
import numpy as np
import pytest

from oracle import map_manage as mm
from helpers import quat_to_mat

W_L, W_C, W_R = 0.55, 0.30, 0.15          # PAPER.md:123 (also tests/golden/paper_constants.txt)
UNIT = ((0.0, 1.0), (0.0, 1.0), (0.0, 1.0))


def test_paper_weights_are_the_golden_ones():
    txt = open(__import__("os").path.join(__import__("os").path.dirname(__file__), "golden", "paper_constants.txt")).read()
    for name, val in (("w_l", W_L), ("w_c", W_C), ("w_r", W_R)):
        assert "%s = %g" % (name, val) in txt


def test_control_score_closed_cases():
    # a line (sigma_1 = sigma_2 = 0): linear = 1, curv = 0; a plane (sigma_0 = sigma_1, sigma_2 = 0): both 0;
    # a ball (all equal): linear = 0, curv = 1/3
    sig = np.array([[2.0, 0.0, 0.0], [1.5, 1.5, 0.0], [0.7, 0.7, 0.7]])
    res = np.array([0.0, 0.4, 1.0])
    c = mm.control_score(sig, res, UNIT, eps=0.0)
    assert np.allclose(c, [W_L * 1.0, W_R * 0.4, W_C / 3.0 + W_R * 1.0], atol=1e-15)
    # eigenvalues are the SQUARES of the standard deviations: sigma = (2, 1, 0) -> linear = 3/4, not 1/2
    assert np.isclose(mm.control_score([[2.0, 1.0, 0.0]], [0.0], UNIT, eps=0.0)[0], W_L * 0.75)
    # min-max normalisation and both clips
    b = ((0.5, 1.0), (0.0, 0.1), (1.0, 3.0))
    c = mm.control_score([[2.0, 1.0, 0.0], [1.0, 1.0, 1.0]], [2.0, 10.0], b, eps=0.0)
    assert np.isclose(c[0], W_L * 0.5 + W_R * 0.5)                       # linear~ = (.75 - .5) / .5, res~ = 1/2
    assert np.isclose(c[1], W_C * 1.0 + W_R * 1.0)                       # curv~ and res~ saturate, linear~ clips at 0
    assert mm.control_score([[1.0, 0.0, 0.0]], [1.0], UNIT, weights=(0.8, 0.3, 0.5), eps=0.0)[0] == 1.0   # outer clip


def test_control_score_against_a_vectorised_rederivation():
    rng = np.random.default_rng(3)
    sig = np.sort(rng.uniform(0.01, 1.0, (500, 3)), axis=1)[:, ::-1]
    res = rng.uniform(0, 0.3, 500)
    b = ((0.1, 0.9), (0.0, 0.2), (0.02, 0.25))
    lam = sig ** 2
    lin = (lam[:, 0] - lam[:, 1]) / (lam[:, 0] + 1e-12)
    cur = lam[:, 2] / (lam.sum(1) + 1e-12)
    t = [np.clip((x - lo) / (hi - lo), 0, 1) for x, (lo, hi) in zip((lin, cur, res), b)]
    ref = np.clip(W_L * t[0] + W_C * t[1] + W_R * t[2], 0, 1)
    assert np.allclose(mm.control_score(sig, res, b), ref, atol=1e-14)


@pytest.mark.parametrize("q", [0.0, 0.01, 0.25, 0.5, 0.731, 0.99, 1.0])
def test_quantile_is_the_inverted_cdf_order_statistic(q):
    rng = np.random.default_rng(5)
    x = rng.uniform(0, 1, 1001).astype(np.float32)
    x[::7] = x[3]                                                         # duplicates
    ref = np.quantile(x, q, method="inverted_cdf") if q > 0 else x.min()
    assert mm.quantile(x, q) == np.float32(ref)
    assert mm.quantile_rank(0.5, 10) == 5 and mm.quantile_rank(0.51, 10) == 6 and mm.quantile_rank(1.0, 10) == 10


def test_split_select_rules():
    c = np.array([0.9, 0.2, 0.9, 0.95, 0.5, 0.9, 0.7], dtype=np.float32)
    op = np.array([0.8, 0.8, 0.8, 0.01, 0.8, 0.8, 0.8], dtype=np.float32)
    # threshold is strict, alpha_min inclusive: 3 fails on opacity, 4 fails c > 0.5
    assert list(mm.split_select(c, op, 0.5, 0.05, 10)) == [0, 2, 5, 6]
    # cap: largest scores first, ties by lower index; the result is reported in index order
    assert list(mm.split_select(c, op, 0.5, 0.05, 2)) == [0, 2]
    assert list(mm.split_select(c, op, 0.5, 0.05, 3)) == [0, 2, 5]
    assert list(mm.split_select(c, op, 0.5, 0.05, 0)) == []
    rng = np.random.default_rng(1)
    c = np.round(rng.uniform(0, 1, 400), 2).astype(np.float32)           # many ties
    op = rng.uniform(0, 1, 400).astype(np.float32)
    cand = np.nonzero((c > np.float32(0.6)) & (op >= np.float32(0.3)))[0]
    order = cand[np.lexsort((cand, -c[cand].astype(np.float64)))][:37]   # numpy's own (score desc, index asc)
    assert list(mm.split_select(c, op, 0.6, 0.3, 37)) == sorted(order.tolist())


def test_split_apply_children():
    rng = np.random.default_rng(2)
    N = 12
    mean = rng.normal(0, 5, (N, 3)).astype(np.float32); quat = rng.normal(size=(N, 4)).astype(np.float32)
    ls = np.log(rng.uniform(0.1, 1.0, (N, 2))).astype(np.float32); op = rng.uniform(0.2, 1, N).astype(np.float32)
    m = rng.normal(size=(N, 10)).astype(np.float32); v = rng.uniform(size=(N, 10)).astype(np.float32)
    sel = np.array([1, 4, 9])
    o_mean, o_quat, o_ls, o_op, o_scale, o_m, o_v = mm.split_apply(mean, quat, ls, op, m, v, sel, 0.5, 1.6)
    assert o_mean.shape[0] == N + 3
    keep = np.setdiff1d(np.arange(N), sel)
    for a, b in ((o_mean, mean), (o_quat, quat), (o_ls, ls), (o_op, op), (o_m, m), (o_v, v)):
        assert np.array_equal(a[keep], b[keep])                          # everything else untouched
    for r, i in enumerate(sel):
        a_i = quat_to_mat(quat[i].astype(np.float64))[:, 0]              # in-plane major axis R(q) e_0
        s0 = np.exp(float(ls[i, 0]))
        plus, minus = o_mean[i].astype(np.float64), o_mean[N + r].astype(np.float64)
        assert np.allclose((plus + minus) / 2, mean[i], atol=1e-6)       # shifted in OPPOSITE directions
        assert np.allclose(plus - minus, 2 * 0.5 * s0 * a_i, atol=2e-6)  # ... along a_i, by shift * s_0 each
        for dst in (i, N + r):
            assert np.array_equal(o_quat[dst], quat[i]) and o_op[dst] == op[i]
            assert np.allclose(np.exp(o_ls[dst].astype(np.float64)), np.exp(ls[i].astype(np.float64)) / 1.6, rtol=1e-6)
            assert not o_m[dst].any() and not o_v[dst].any()
    assert np.allclose(o_scale, np.exp(o_ls.astype(np.float64)), rtol=1e-6)


def _plane_case():
    """Nine coplanar surfels (z = 2) in one 4 m cell around the representative at the origin of the cell."""
    ident = np.array([1.0, 0, 0, 0], dtype=np.float32)
    xy = np.array([[1.0, 1.0], [1.1, 1.0], [1.0, 1.3], [1.6, 1.0], [1.0, 2.2], [2.5, 2.5], [0.4, 1.0], [1.0, 0.1], [3.0, 1.0]])
    mean = np.concatenate([xy, np.full((9, 1), 2.0)], 1).astype(np.float32)
    quat = np.tile(ident, (9, 1))
    scale = np.full((9, 2), 0.2, dtype=np.float32); scale[:, 1] = 0.1     # u along x (s0 = .2), v along y (s1 = .1)
    op = np.full(9, 0.5, dtype=np.float32); op[0] = 0.9                   # surfel 0 is the representative
    c = np.full(9, 0.1, dtype=np.float32)
    return mean, quat, scale, op, c


def test_cover_prune_closed_case():
    mean, quat, scale, op, c = _plane_case()
    kw = dict(axes=(0, 1), origin=(0.0, 0.0), cell=4.0, dims=(2, 2), thr=0.2, alpha_min=0.05, s_max=10.0)
    # rho^2 of the 8 members w.r.t. surfel 0: (dx/.2)^2 + (dy/.1)^2
    rho2 = np.array([0.25, 9.0, 9.0, 144.0, 56.25 + 225.0, 9.0, 81.0, 100.0])
    keep, ns, d = mm.cover_prune_pass(mean, quat, scale, op, c, kappa=3.0, q_cover=0.0, cap=100, **kw)
    assert d["reps"] == {0: 0} and np.allclose(d["rho2"][1:], rho2, rtol=1e-5)
    # q_cover = 0 -> R = kappa: members inside the representative's 3-sigma ellipse go (rho^2 <= 9, boundary included)
    assert list(np.nonzero(~keep)[0]) == [1, 2, 3, 6] and np.array_equal(ns, scale)
    # q_cover = 0.75 -> rank ceil(.75 * 8) = 6 -> R^2 = 6th smallest = 100: six members go, the scale grows by 10/3
    keep, ns, _ = mm.cover_prune_pass(mean, quat, scale, op, c, kappa=3.0, q_cover=0.75, cap=100, **kw)
    assert list(np.nonzero(~keep)[0]) == [1, 2, 3, 6, 7, 8]
    assert np.allclose(ns[0], scale[0] * (10.0 / 3.0), rtol=1e-6) and np.array_equal(ns[1:], scale[1:])
    # s_max caps the expansion, the cap keeps the removals of lowest index
    keep, ns, _ = mm.cover_prune_pass(mean, quat, scale, op, c, kappa=3.0, q_cover=0.75, cap=2, **{**kw, "s_max": 0.3})
    assert list(np.nonzero(~keep)[0]) == [1, 2] and np.allclose(ns[0], [0.3, 0.3])


def test_frame_uv_against_scipy_rotation():
    """Both columns the cover radius uses, t_u = R(q^) e_0 and t_v = R(q^) e_1, against scipy's rotation matrix of the
    same (unnormalised) quaternion -- a library routine, not a retyped formula.  A wrong sign or a swapped product in
    any of the six entries is an O(1) error for a generic q; fp32 rounding is ~1e-7."""
    from scipy.spatial.transform import Rotation
    rng = np.random.default_rng(3)
    for q in np.concatenate([rng.normal(size=(50, 4)), [[1, 0, 0, 0], [0, 1, 0, 0], [0, 0, 1, 0], [0, 0, 0, 1]]]):
        q = (q * rng.uniform(0.2, 3.0)).astype(np.float32)
        R = Rotation.from_quat([q[1], q[2], q[3], q[0]]).as_matrix()      # scipy takes (x, y, z, w)
        tu, tv = mm._frame_uv(q)
        assert np.allclose(np.array(tu, dtype=np.float64), R[:, 0], atol=2e-6)
        assert np.allclose(np.array(tv, dtype=np.float64), R[:, 1], atol=2e-6)


def test_cover_prune_rotated_representative():
    """The tangent-plane offsets of the members are taken in the REPRESENTATIVE's frame (u along R(q) e_0 over s_0,
    v along R(q) e_1 over s_1).  (i) _plane_case with the representative turned 90 degrees about its normal: u and v
    swap roles and the hand-computed list becomes (dy/.2)^2 + (dx/.1)^2.  (ii) A generic, tilted representative and
    members placed at mu + a t_u + b t_v + c n with (t_u, t_v, n) from scipy: rho^2 must come out as (a/s0)^2 + (b/s1)^2
    whatever c is -- a wrong entry of t_v (say 2(yz - wx)) changes every v."""
    from scipy.spatial.transform import Rotation
    mean, quat, scale, op, c = _plane_case()
    kw = dict(axes=(0, 1), origin=(0.0, 0.0), cell=4.0, dims=(2, 2), thr=0.2, alpha_min=0.05, s_max=10.0, kappa=3.0,
              q_cover=0.0, cap=100)
    quat = quat.copy(); quat[0] = [np.sqrt(0.5), 0.0, 0.0, np.sqrt(0.5)]      # +90 deg about z: t_u = +y, t_v = -x
    keep, _, d = mm.cover_prune_pass(mean, quat, scale, op, c, **kw)
    rho2 = np.array([1.0, 2.25, 36.0, 36.0, 56.25 + 225.0, 36.0, 20.25, 400.0])
    assert d["reps"] == {0: 0} and np.allclose(d["rho2"][1:], rho2, rtol=1e-5)
    assert list(np.nonzero(~keep)[0]) == [1, 2]
    # (ii)
    rng = np.random.default_rng(8)
    q0 = np.array([0.61, -0.37, 0.52, 0.29]) * 1.7
    R = Rotation.from_quat([q0[1], q0[2], q0[3], q0[0]]).as_matrix()
    ab = rng.uniform(-0.6, 0.6, (8, 2)); cn = rng.uniform(-0.3, 0.3, 8)
    mu0 = np.array([2.0, 2.0, 1.0])
    pts = mu0 + ab[:, :1] * R[:, 0] + ab[:, 1:] * R[:, 1] + cn[:, None] * R[:, 2]
    mean2 = np.concatenate([[mu0], pts]).astype(np.float32)
    quat2 = np.tile(np.array([1.0, 0, 0, 0], dtype=np.float32), (9, 1)); quat2[0] = q0.astype(np.float32)
    _, _, d = mm.cover_prune_pass(mean2, quat2, scale, op, c, **kw)
    assert d["reps"] == {0: 0}
    assert np.allclose(d["rho2"][1:], (ab[:, 0] / 0.2) ** 2 + (ab[:, 1] / 0.1) ** 2, rtol=1e-4, atol=1e-4)


def test_cover_prune_candidates_cells_and_planes():
    mean, quat, scale, op, c = _plane_case()
    kw = dict(origin=(0.0, 0.0), cell=4.0, dims=(2, 2), thr=0.2, alpha_min=0.05, kappa=3.0, q_cover=0.0, s_max=10.0,
              cap=100)
    c2 = c.copy(); c2[1] = 0.5                               # not planar: neither removed nor counted
    op2 = op.copy(); op2[2] = 0.01                           # too transparent: same
    keep, _, d = mm.cover_prune_pass(mean, quat, scale, op2, c2, axes=(0, 1), **kw)
    assert keep[1] and keep[2] and list(np.nonzero(~keep)[0]) == [3, 6]
    # a tie in alpha picks the lower index as representative
    op3 = op.copy(); op3[4] = 0.9
    assert mm.cover_prune_pass(mean, quat, scale, op3, c, axes=(0, 1), **kw)[2]["reps"] == {0: 0}
    # cell size 1 m: members fall into other cells and are no longer grouped with surfel 0
    keep, _, d = mm.cover_prune_pass(mean, quat, scale, op, c, axes=(0, 1), **{**kw, "cell": 1.0, "dims": (8, 8)})
    assert d["n_groups"] > 1 and d["reps"][mm.cell_of((1.0, 1.0), (0, 0), 1.0, (8, 8))] == 0
    # outside the grid / NaN: takes no part
    far = mean.copy(); far[3, 0] = 100.0; far[6, 1] = np.nan
    keep, _, _ = mm.cover_prune_pass(far, quat, scale, op, c, axes=(0, 1), **kw)
    assert keep[3] and keep[6]
    # the pass projects onto the axes it is given: in the (x, z) plane all nine share z = 2 -> same cell row
    keep_xz, _, d = mm.cover_prune_pass(mean, quat, scale, op, c, axes=(0, 2), **kw)
    assert d["reps"] == {0: 0} and np.array_equal(keep_xz, mm.cover_prune_pass(mean, quat, scale, op, c, axes=(0, 1), **kw)[0])


def test_cover_prune_invariants_on_a_random_map():
    rng = np.random.default_rng(11)
    N = 3000
    mean = np.concatenate([rng.uniform(-20, 20, (N, 2)), rng.normal(0, 0.02, (N, 1))], 1).astype(np.float32)
    quat = (np.array([1, 0, 0, 0]) + rng.normal(0, 0.05, (N, 4))).astype(np.float32)
    scale = rng.uniform(0.05, 0.4, (N, 2)).astype(np.float32); op = rng.uniform(0, 1, N).astype(np.float32)
    c = rng.uniform(0, 1, N).astype(np.float32)
    thr = mm.quantile(c, 0.6)
    cap = N // 10
    keep, ns, d = mm.cover_prune_pass(mean, quat, scale, op, c, (0, 1), (-20.0, -20.0), 1.0, (40, 40), thr, 0.1, 3.0, 0.5,
                                      1.0, cap)
    cand = (c <= thr) & (op >= np.float32(0.1))
    assert (~keep).sum() == cap                                           # the cap binds on this map
    assert not (~keep & ~cand).any()                                      # only planar candidates are removed
    reps = np.array(sorted(d["reps"].values()))
    assert keep[reps].all()                                               # a representative is never removed
    changed = np.nonzero((ns != scale).any(1))[0]
    assert set(changed) <= set(reps) and (ns >= scale).all() and (ns <= 1.0).all()
    kept, (m2,) = mm.compact(keep, mean)
    assert np.array_equal(m2, mean[keep]) and np.array_equal(kept, np.nonzero(keep)[0])
