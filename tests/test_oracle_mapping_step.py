"""Pins of oracle/mapping_step.py: closed forms, finite differences, and torch's own
BCE / autograd / torch.optim.Adam as independent library routines.  All CPU (-m "not gpu")."""
from __future__ import annotations

import os

import numpy as np
import torch

from oracle import mapping_step as ms

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "paper_constants.txt")


def _paper_constants():
    out = {}
    for ln in open(GOLDEN):
        ln = ln.strip()
        if ln and not ln.startswith("#") and "=" in ln:
            k, v = ln.split("=")
            out[k.strip()] = float(v)
    return out


def test_defaults_are_the_papers_weights():
    c = _paper_constants()
    assert ms.AdamHyper().lambda_s == c["lambda_s"] == 10
    assert ms.loss_alpha.__defaults__[1] == c["lambda_alpha"] == 0.1


def test_loss_alpha_closed_forms():
    H, W = 4, 6
    tgt = np.ones((H, W)); tgt[0, :] = 0.0                       # one row invalid: |Omega_D| = 18
    for a0 in (1.0, 0.5, 0.01):
        A = np.full((H, W), a0)
        L, g = ms.loss_alpha(A, tgt, None, lambda_alpha=0.1, eps=1e-6)
        assert abs(L - (-np.log(a0 + 1e-6))) < 1e-14              # mean of a constant
        assert np.all(g[0] == 0.0)
        np.testing.assert_allclose(g[1:], -0.1 / (18 * (a0 + 1e-6)), rtol=1e-14)
    # A^ = 0 is finite thanks to eps; empty Omega_D gives zeros
    L, g = ms.loss_alpha(np.zeros((H, W)), tgt, None, eps=1e-6)
    assert abs(L - (-np.log(1e-6))) < 1e-12
    L, g = ms.loss_alpha(np.ones((H, W)), np.zeros((H, W)))
    assert L == 0.0 and not g.any()
    # the keep mask removes pixels from Omega_D
    keep = np.ones((H, W), dtype=np.uint8); keep[1, :3] = 0
    L, g = ms.loss_alpha(np.full((H, W), 0.5), tgt, keep)
    assert np.all(g[1, :3] == 0.0) and np.all(g[1, 3:] != 0.0)
    np.testing.assert_allclose(g[1, 3:], -0.1 / (15 * (0.5 + 1e-6)), rtol=1e-14)


def test_loss_alpha_is_positive_only_bce_of_torch():
    rng = np.random.default_rng(3)
    H, W = 8, 16
    A = rng.uniform(0.05, 0.999, (H, W))
    tgt = rng.uniform(-1, 5, (H, W))                              # ~17 % invalid
    keep = (rng.uniform(size=(H, W)) > 0.1).astype(np.uint8)
    eps, lam = 1e-6, 0.1
    L, g = ms.loss_alpha(A, tgt, keep, lam, eps)
    At = torch.tensor(A, dtype=torch.float64, requires_grad=True)
    M = torch.tensor((tgt > 0) & (keep != 0))
    bce = torch.nn.functional.binary_cross_entropy((At + eps)[M], torch.ones(int(M.sum()), dtype=torch.float64),
                                                   reduction="mean")   # BCE(A^, 1)
    assert abs(L - float(bce.detach())) < 1e-13
    (lam * bce).backward()
    np.testing.assert_allclose(g, At.grad.numpy(), rtol=1e-12, atol=0)
    # central differences of lambda_alpha * L_alpha
    for (j, i) in ((1, 2), (5, 9), (7, 15)):
        h = 1e-6
        Ap, Am = A.copy(), A.copy(); Ap[j, i] += h; Am[j, i] -= h
        fd = lam * (ms.loss_alpha(Ap, tgt, keep, lam, eps)[0] - ms.loss_alpha(Am, tgt, keep, lam, eps)[0]) / (2 * h)
        assert abs(fd - g[j, i]) <= 1e-7 * max(1.0, abs(g[j, i]))


def test_loss_scale_closed_form_and_autograd():
    s = np.array([[0.2, 0.1], [1.5, 0.3], [0.4, 2.0], [1.0, 1.0], [3.0, 2.5]])
    L, g = ms.loss_scale(s, s_max=1.0)
    assert abs(L - (0.5 + 1.0 + 2.0)) < 1e-15                     # rows 1, 2, 4; row 3 sits on the threshold
    np.testing.assert_array_equal(g, [[0, 0], [1, 0], [0, 1], [0, 0], [1, 0]])
    L, g = ms.loss_scale(np.array([[2.0, 2.0]]), 1.0)             # tie: even split
    assert L == 1.0 and g.tolist() == [[0.5, 0.5]]
    rng = np.random.default_rng(5)
    s = rng.uniform(0.05, 2.0, (200, 2))
    L, g = ms.loss_scale(s, 0.8)
    st = torch.tensor(s, requires_grad=True)
    Lt = torch.clamp(torch.amax(st, dim=1) - 0.8, min=0).sum()    # Eq. 12 with torch's own ops
    Lt.backward()
    assert abs(L - float(Lt)) < 1e-12
    np.testing.assert_array_equal(g, st.grad.numpy())


def _random_problem(rng, N):
    mean = rng.normal(0, 10, (N, 3)); quat = rng.normal(0, 1, (N, 4))
    log_scale = np.log(rng.uniform(0.05, 2.5, (N, 2))); opacity = rng.uniform(0.02, 0.98, N)
    return mean, quat, log_scale, opacity


def test_adam_step_matches_torch_optim_adam():
    """Five steps with changing gradients: torch.optim.Adam on fp64 leaf tensors, the log-scale chain rule and
    L_scale coming from torch autograd through exp (nothing of oracle/mapping_step.py is re-typed here)."""
    rng = np.random.default_rng(11)
    N = 64
    mean, quat, ls, op = _random_problem(rng, N)
    h = ms.AdamHyper(lr_mean=1e-2, lr_quat=2e-3, lr_scale=5e-3, lr_opacity=3e-2, eps=1e-15, lambda_s=10.0, s_max=1.0,
                     alpha_lo=-10.0, alpha_hi=10.0)                # clip inactive in this test
    tm, tq, tl, to = (torch.tensor(x, requires_grad=True) for x in (mean, quat, ls, op))
    opt = torch.optim.Adam([{"params": [tm], "lr": h.lr_mean}, {"params": [tq], "lr": h.lr_quat},
                            {"params": [tl], "lr": h.lr_scale}, {"params": [to], "lr": h.lr_opacity}],
                           betas=(h.beta1, h.beta2), eps=h.eps)
    m = np.zeros((N, 10)); v = np.zeros((N, 10))
    for t in range(1, 6):
        gm, gq, gs, go = rng.normal(0, 1, (N, 3)), rng.normal(0, 1, (N, 4)), rng.normal(0, 1, (N, 2)), rng.normal(0, 1, N)
        mean, quat, ls, op, s_new, m, v, Ls = ms.adam_step(mean, quat, ls, op, gm, gq, gs, go, m, v, t, h)
        opt.zero_grad()
        s = torch.exp(tl)
        # image-side gradients enter as a linear probe <g, theta>; L_scale (Eq. 12) and exp() go through autograd
        loss = (tm * torch.tensor(gm)).sum() + (tq * torch.tensor(gq)).sum() + (s * torch.tensor(gs)).sum() + \
               (to * torch.tensor(go)).sum() + h.lambda_s * torch.clamp(torch.amax(s, dim=1) - h.s_max, min=0).sum()
        Ls_t = float(torch.clamp(torch.amax(s, dim=1) - h.s_max, min=0).sum())
        loss.backward()
        opt.step()
        assert abs(Ls - Ls_t) <= 1e-12 * max(1.0, Ls_t)
        for a, b in ((mean, tm), (quat, tq), (ls, tl), (op, to)):
            np.testing.assert_allclose(a, b.detach().numpy(), rtol=1e-10, atol=1e-12)
        np.testing.assert_allclose(s_new, np.exp(ls), rtol=0, atol=0)


def test_adam_first_step_closed_form_and_clip():
    """t = 1: m^ = g, v^ = g^2 -> every component moves by lr * sign(g) (up to eps); alpha is clipped."""
    rng = np.random.default_rng(2)
    N = 16
    mean, quat, ls, op = _random_problem(rng, N)
    ls[:] = np.log(0.5)                                            # below s_max: no L_scale gradient
    op[:4] = 0.999; op[4:8] = 0.001
    gm, gq, gs, go = rng.normal(0, 1, (N, 3)), rng.normal(0, 1, (N, 4)), rng.normal(0, 1, (N, 2)), rng.normal(0, 1, N)
    go[:4] = -1.0; go[4:8] = 1.0                                   # push alpha out of [0, 1]
    h = ms.AdamHyper(lr_mean=1e-2, lr_quat=2e-3, lr_scale=5e-3, lr_opacity=3e-2, eps=1e-15, s_max=1.0)
    m0 = np.zeros((N, 10))
    mean2, quat2, ls2, op2, s2, m, v, Ls = ms.adam_step(mean, quat, ls, op, gm, gq, gs, go, m0, m0, 1, h)
    assert Ls == 0.0
    np.testing.assert_allclose(mean2, mean - 1e-2 * np.sign(gm), rtol=0, atol=1e-12)
    np.testing.assert_allclose(quat2, quat - 2e-3 * np.sign(gq), rtol=0, atol=1e-12)
    np.testing.assert_allclose(ls2, ls - 5e-3 * np.sign(gs), rtol=0, atol=1e-12)     # sign(s g) = sign(g), s > 0
    assert np.all(op2[:4] == 1.0) and np.all(op2[4:8] == 0.0)
    np.testing.assert_allclose(op2[8:], op[8:] - 3e-2 * np.sign(go[8:]), rtol=0, atol=1e-12)
    np.testing.assert_allclose(m[:, :3], 0.1 * gm, rtol=1e-14); np.testing.assert_allclose(v[:, :3], 1e-3 * gm * gm, rtol=1e-12)


def test_scale_regulariser_pulls_oversized_surfels_back():
    """With zero image-side gradients only surfels with max(s) > s_max move, and only in their larger component."""
    ls = np.log(np.array([[0.5, 0.2], [2.0, 0.3], [0.4, 3.0]]))
    N = 3
    z3, z4, z2, z1 = np.zeros((N, 3)), np.zeros((N, 4)), np.zeros((N, 2)), np.zeros(N)
    h = ms.AdamHyper(lr_scale=1e-2, s_max=1.0)
    out = ms.adam_step(z3, z4 + [1, 0, 0, 0], ls, z1 + 0.5, z3, z4, z2, z1, np.zeros((N, 10)), np.zeros((N, 10)), 1, h)
    ls2, Ls = out[2], out[7]
    assert abs(Ls - (1.0 + 2.0)) < 1e-14
    np.testing.assert_allclose(ls2[0], ls[0], atol=0)
    np.testing.assert_allclose(ls2[1], ls[1] - [1e-2, 0], atol=1e-12)
    np.testing.assert_allclose(ls2[2], ls[2] - [0, 1e-2], atol=1e-12)
