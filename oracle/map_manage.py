"""ORACLE -- test infrastructure only (see oracle/__init__.py).

Plain numpy definition of the rest of the paper's map management (section 3.3
"Control Score" and section 3.5 "Real-time Map Budget Control"):

  control_score      Eq. 9: linearity / curvature of the tracking covariance + normalised residual
  quantile           Q_q(.) of PAPER.md:160, 166
  split_select       "Structure-aware Adaptive Splitting": which surfels split
  split_apply        the two children of a split surfel, shifted along a_i = R(q_i) e_0
  cover_prune_pass   one pass of "Multi-pass Planar Cover and Prune", PAPER.md:158-164
  compact            keep-flag compaction (what follows a pass: order-preserving, every row moves with its surfel)

Everything the paper leaves open is a caller input, listed as readings R29-R36 in DESIGN.md section 3:
 R29  the "~" of Eq. 9 is min-max normalisation x~ = clip((x - lo) / (hi - lo), 0, 1) with (lo, hi) per term supplied by
      the caller (Fig. 3's caption says "robustly normalized": robust bounds, e.g. quantiles, are the caller's);
      Eq. 9 is printed garbled ("w_l linear" under one tilde): read as w_l linear~ + w_c curv~ + w_r res~.
 R30  Q_q(x) = the k-th smallest value, k = clip(ceil(q N), 1, N) (no interpolation: the result is an element of x).
 R31  split candidates: c_i > Q_{q_split}(c) and alpha_i >= alpha_min; at most cap = floor(ratio N) of them split --
      those with the largest c_i, ties by lower index.
 R32  children: means mu_i +- shift * s_{i,0} * a_i (a_i = first column of R(q_i / |q_i|)), both scales divided by
      `shrink`, q and alpha copied, optimiser moments zero; child "+" takes the parent's row, child "-" is appended
      in index order of the parents, so the map grows from N to N + n_split.
 R33  a cover-and-prune pass projects the means onto two world axes (the caller runs one pass per orthogonal plane) and
      groups them in a dense grid of square cells (origin, cell size, dims from the caller); surfels outside the grid or
      with non-finite means take no part.
 R34  planar candidates: c_i <= Q_{q_plane}(c) and alpha_i >= alpha_min; the representative g_r of a cell is its
      candidate of largest alpha (ties: lower index); the other candidates of the cell are its members.
 R35  cover region, in g_r's tangent-plane coordinates u = t_u.(mu_m - mu_r) / s_r0, v = t_v.(mu_m - mu_r) / s_r1:
      rho^2 = u^2 + v^2 <= R^2 with R^2 = max(kappa^2, Q_{q_cover}(rho^2 over the members)), i.e. the representative's
      kappa-sigma ellipse, expanded isotropically (both scales times R / kappa, capped at s_max) until it holds the
      q_cover-quantile of the members.  Members inside are redundant and removed.
 R36  per-pass cap: at most floor(ratio N) removals, taken in ascending index order.
Decisions (cell, candidate, representative, inside / outside, ranks) are integer work and are taken in fp32 with the
operation order written here, so that the CUDA path can be compared bit for bit; float outputs carry a tolerance.

Parity with the authors' map management is unpinned (the paper prints none of these constants or rules); the
functions are pinned by closed cases, invariants and numpy's own sort / quantile (tests/test_oracle_map_manage.py).
Nothing here is imported by the CUDA path.
"""
from __future__ import annotations

import math

import numpy as np

F = np.float32


def control_score(sigma, res, bounds, weights=(0.55, 0.30, 0.15), eps=1e-12):
    """Eq. 9.  sigma [N,3] standard deviations sorted descending, res [N] G-ICP residuals,
    bounds = ((lo_l, hi_l), (lo_c, hi_c), (lo_r, hi_r)).  Returns c [N] in [0, 1] (fp64)."""
    sigma = np.asarray(sigma, dtype=np.float64)
    res = np.asarray(res, dtype=np.float64)
    out = np.zeros(sigma.shape[0])
    for i in range(sigma.shape[0]):
        l0, l1, l2 = sigma[i, 0] ** 2, sigma[i, 1] ** 2, sigma[i, 2] ** 2      # lambda_{i,j} = sigma_{i,j}^2
        linear = (l0 - l1) / (l0 + eps)
        curv = l2 / (l0 + l1 + l2 + eps)
        terms = []
        for x, (lo, hi) in zip((linear, curv, res[i]), bounds):
            terms.append(min(max((x - lo) / (hi - lo), 0.0), 1.0))
        c = weights[0] * terms[0] + weights[1] * terms[1] + weights[2] * terms[2]
        out[i] = min(max(c, 0.0), 1.0)
    return out


def quantile_rank(q, n):
    """k of R30 (1-based)."""
    return min(max(int(math.ceil(float(q) * n)), 1), n)


def quantile(x, q):
    """Q_q(x), R30: the k-th smallest element."""
    x = np.asarray(x, dtype=np.float32)
    if x.shape[0] == 0:
        return F(0.0)
    return np.sort(x, kind="stable")[quantile_rank(q, x.shape[0]) - 1]


def split_select(c, opacity, thr, alpha_min, cap):
    """R31.  thr = Q_{q_split}(c) (passed in so that both sides use the same threshold).  Returns the ascending
    indices of the surfels that split."""
    c = np.asarray(c, dtype=np.float32)
    op = np.asarray(opacity, dtype=np.float32)
    cand = [i for i in range(c.shape[0]) if c[i] > F(thr) and op[i] >= F(alpha_min)]
    if len(cand) > cap:
        cand.sort(key=lambda i: (-float(c[i]), i))          # largest score first, ties by lower index
        cand = cand[:cap]
    return np.asarray(sorted(cand), dtype=np.int64)


def _frame_uv(q):
    """First two columns (t_u = R e_0, t_v = R e_1) of R(q / |q|), fp32, every operation rounded on its own in the
    order written (the CUDA path writes the same sequence with __fmul_rn / __fadd_rn / __fdiv_rn / __fsqrt_rn)."""
    w, x, y, z = (F(q[0]), F(q[1]), F(q[2]), F(q[3]))
    n = np.sqrt(F(F(F(w * w) + F(x * x)) + F(y * y)) + F(z * z))
    w, x, y, z = F(w / n), F(x / n), F(y / n), F(z / n)
    two, one = F(2.0), F(1.0)
    xx, yy, zz = F(x * x), F(y * y), F(z * z)
    xy, xz, yz = F(x * y), F(x * z), F(y * z)
    wx, wy, wz = F(w * x), F(w * y), F(w * z)
    tu = (F(one - F(two * F(yy + zz))), F(two * F(xy + wz)), F(two * F(xz - wy)))
    tv = (F(two * F(xy - wz)), F(one - F(two * F(xx + zz))), F(two * F(yz + wx)))
    return tu, tv


def split_apply(mean, quat, log_scale, opacity, m, v, sel, shift, shrink):
    """R32.  Returns the grown arrays (mean, quat, log_scale, opacity, scale, m, v) with N + len(sel) rows."""
    mean = np.asarray(mean, dtype=np.float32); quat = np.asarray(quat, dtype=np.float32)
    ls = np.asarray(log_scale, dtype=np.float32); op = np.asarray(opacity, dtype=np.float32)
    m = np.asarray(m, dtype=np.float32); v = np.asarray(v, dtype=np.float32)
    N, ns = mean.shape[0], len(sel)
    out = [np.concatenate([a, np.zeros((ns,) + a.shape[1:], dtype=np.float32)]) for a in (mean, quat, ls, op, m, v)]
    o_mean, o_quat, o_ls, o_op, o_m, o_v = out
    dls = np.log(np.float64(shrink))
    for r, i in enumerate(sel):
        tu, _ = _frame_uv(quat[i])
        s0 = np.exp(np.float64(ls[i, 0]))                       # the activated major scale s_{i,0}
        delta = np.array([float(tu[0]), float(tu[1]), float(tu[2])]) * (float(shift) * s0)
        child_ls = (ls[i].astype(np.float64) - dls).astype(np.float32)
        for dst, sign in ((i, +1.0), (N + r, -1.0)):
            o_mean[dst] = (mean[i].astype(np.float64) + sign * delta).astype(np.float32)
            o_quat[dst] = quat[i]
            o_ls[dst] = child_ls
            o_op[dst] = op[i]
            o_m[dst] = 0.0
            o_v[dst] = 0.0
    scale = np.exp(o_ls.astype(np.float64)).astype(np.float32)
    return o_mean, o_quat, o_ls, o_op, scale, o_m, o_v


def cell_of(mean_ab, origin, cell, dims):
    """R33: dense-grid cell of a projected mean (fp32 subtract, divide, floor), or -1 outside / not finite."""
    ia = np.floor(F(F(F(mean_ab[0]) - F(origin[0])) / F(cell)))
    ib = np.floor(F(F(F(mean_ab[1]) - F(origin[1])) / F(cell)))
    if not (ia >= 0 and ia < dims[0] and ib >= 0 and ib < dims[1]):      # (False for NaN)
        return -1
    return int(ia) * int(dims[1]) + int(ib)


def cover_prune_pass(mean, quat, scale, opacity, c, axes, origin, cell, dims, thr, alpha_min, kappa, q_cover, s_max,
                     cap):
    """One pass of planar cover-and-prune, R33-R36.  axes = (a, b) world axes of the projection plane;
    thr = Q_{q_plane}(c).  Returns (keep [N] bool, new scale [N,2] fp32, diagnostics dict)."""
    mean = np.asarray(mean, dtype=np.float32); quat = np.asarray(quat, dtype=np.float32)
    scale = np.asarray(scale, dtype=np.float32); op = np.asarray(opacity, dtype=np.float32)
    c = np.asarray(c, dtype=np.float32)
    N = mean.shape[0]
    groups = {}
    for i in range(N):
        if c[i] <= F(thr) and op[i] >= F(alpha_min):                     # planar candidate, R34
            g = cell_of((mean[i, axes[0]], mean[i, axes[1]]), origin, cell, dims)
            if g >= 0:
                groups.setdefault(g, []).append(i)
    new_scale = scale.copy()
    removed = np.zeros(N, dtype=bool)
    rho2_all = np.full(N, np.nan, dtype=np.float32)
    reps = {}
    for g, idx in groups.items():
        r = idx[0]
        for i in idx[1:]:
            if op[i] > op[r]:                                            # largest alpha, ties: lower index
                r = i
        reps[g] = r
        members = [i for i in idx if i != r]
        if not members:
            continue
        tu, tv = _frame_uv(quat[r])
        rho2 = []
        for i in members:
            d0, d1, d2 = F(mean[i, 0] - mean[r, 0]), F(mean[i, 1] - mean[r, 1]), F(mean[i, 2] - mean[r, 2])
            u = F(F(F(F(tu[0] * d0) + F(tu[1] * d1)) + F(tu[2] * d2)) / scale[r, 0])
            w_ = F(F(F(F(tv[0] * d0) + F(tv[1] * d1)) + F(tv[2] * d2)) / scale[r, 1])
            rho2.append(F(F(u * u) + F(w_ * w_)))
            rho2_all[i] = rho2[-1]
        n = len(members)
        k = min(max(int(np.ceil(F(F(q_cover) * F(n)))), 1), n)            # rank of the q_cover-quantile (fp32 product)
        Q = sorted(rho2)[k - 1]
        R2 = max(F(F(kappa) * F(kappa)), Q)
        f = F(np.sqrt(R2) / F(kappa))
        new_scale[r, 0] = min(F(f * scale[r, 0]), F(s_max))
        new_scale[r, 1] = min(F(f * scale[r, 1]), F(s_max))
        for i, x in zip(members, rho2):
            if x <= R2:
                removed[i] = True
    # R36: the cap keeps the removals of lowest index
    order = np.nonzero(removed)[0]
    if len(order) > cap:
        removed[order[cap:]] = False
    return ~removed, new_scale, dict(reps=reps, rho2=rho2_all, n_groups=len(groups))


def compact(keep, *rows):
    """Order-preserving compaction by keep flags: (kept indices, [rows restricted to them])."""
    kept = np.asarray([i for i in range(len(keep)) if keep[i]], dtype=np.int64)
    return kept, [np.asarray(a)[kept] for a in rows]
