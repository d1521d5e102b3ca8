"""ORACLE -- test infrastructure only (see oracle/__init__.py).

Plain fp64 numpy definition of the steps that close the paper's mapping iteration after the
rasteriser's backward (section 3.4):

  loss_alpha       L_alpha of Eq. 10 (right): positive-only BCE(A^, 1) over the valid pixels
  loss_scale       L_scale of Eq. 12
  adam_step        one optimiser step on Theta = {mu, q, s~, alpha} with s~ = log s
                    and the Eq. 13 weight lambda_s of L_scale

Readings (R20-R24): epsilon of Eq. 10 is a caller input (default 1e-6); the paper
names no optimiser -> Adam (Kingma & Ba, as in the 3DGS / 2DGS lineage [13], [16]) with bias correction,
per-group learning rates supplied by the caller; alpha is optimised directly (Theta lists alpha, not a
logit) and clipped to [alpha_lo, alpha_hi] after the step; q is not re-normalised (the renderer normalises
inside, S1); at s0 == s1 the subgradient of max(s0, s1) is split evenly.

Parity with the authors' optimiser is unpinned (the paper prints no value for it); the functions are
pinned against closed forms, finite differences and torch's own BCE / autograd / torch.optim.Adam
(tests/test_oracle_mapping_step.py).  Nothing here is imported by the CUDA path.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np


def valid_mask(target_range, keep_mask=None):
    """Omega_M = {D > 0 and keep}: M_D of PAPER.md:127 AND-ed with the reliability mask (R13)."""
    m = np.asarray(target_range, dtype=np.float64) > 0.0
    if keep_mask is not None:
        m &= np.asarray(keep_mask) != 0
    return m


def loss_alpha(alpha_hat, target_range, keep_mask=None, lambda_alpha=0.1, eps=1e-6):
    """Eq. 10 (right): L_alpha = -(1/|Omega_D|) sum_{Omega_D} log(A^_i + eps).

    Returns (L_alpha, gA) with gA = d(lambda_alpha * L_alpha)/dA^ (zero outside Omega_D; all zero if Omega_D is
    empty, R14)."""
    A = np.asarray(alpha_hat, dtype=np.float64)
    m = valid_mask(target_range, keep_mask)
    n = int(m.sum())
    gA = np.zeros_like(A)
    if n == 0:
        return 0.0, gA
    L = 0.0
    for idx in zip(*np.nonzero(m)):          # plain loop over the valid pixels, in the paper's notation
        L -= np.log(A[idx] + eps)
        gA[idx] = -lambda_alpha / (n * (A[idx] + eps))
    return L / n, gA


def loss_scale(scale, s_max):
    """Eq. 12: L_scale = sum_i max(0, max(s_ix, s_iy) - s_max).  Returns (L_scale, dL_scale/ds [N,2])."""
    s = np.asarray(scale, dtype=np.float64)
    L = 0.0
    g = np.zeros_like(s)
    for i in range(s.shape[0]):
        top = max(s[i, 0], s[i, 1])
        if top - s_max > 0.0:
            L += top - s_max
            if s[i, 0] > s[i, 1]:
                g[i, 0] = 1.0
            elif s[i, 1] > s[i, 0]:
                g[i, 1] = 1.0
            else:                              # tie: even split (reading R24)
                g[i, 0] = g[i, 1] = 0.5
    return L, g


@dataclass
class AdamHyper:
    lr_mean: float = 1.6e-4
    lr_quat: float = 1e-3
    lr_scale: float = 5e-3
    lr_opacity: float = 5e-2
    beta1: float = 0.9
    beta2: float = 0.999
    eps: float = 1e-15
    lambda_s: float = 10.0          # Eq. 13 weight of L_scale
    s_max: float = 1.0
    alpha_lo: float = 0.0
    alpha_hi: float = 1.0


def adam_step(mean, quat, log_scale, opacity, g_mean, g_quat, g_scale, g_opacity, m, v, step, h: AdamHyper):
    """One Adam step on Theta = {mu, q, s~, alpha}.

    g_* are the rasteriser's gradients of the image-side loss with respect to (mu, q, s, alpha) in ACTIVATED
    space (what lgs_render_backward returns).  The step adds lambda_s dL_scale/ds (Eq. 12-13), applies the
    chain rule of s = exp(s~) (g_s~ = s * g_s), and updates every component with Adam:
        m <- b1 m + (1 - b1) g;  v <- b2 v + (1 - b2) g^2;
        theta <- theta - lr (m / (1 - b1^t)) / (sqrt(v / (1 - b2^t)) + eps)
    m, v: [N,10] in the component order (mu 3, q 4, s~ 2, alpha 1); step = t >= 1.
    Returns (mean, quat, log_scale, opacity, scale = exp(new log_scale), m, v, L_scale before the step)."""
    mean = np.array(mean, dtype=np.float64); quat = np.array(quat, dtype=np.float64)
    log_scale = np.array(log_scale, dtype=np.float64); opacity = np.array(opacity, dtype=np.float64)
    m = np.array(m, dtype=np.float64); v = np.array(v, dtype=np.float64)
    s = np.exp(log_scale)
    L_scale, g_reg = loss_scale(s, h.s_max)
    g_ls = s * (np.asarray(g_scale, dtype=np.float64) + h.lambda_s * g_reg)
    g = np.concatenate([np.asarray(g_mean, dtype=np.float64), np.asarray(g_quat, dtype=np.float64), g_ls,
                        np.asarray(g_opacity, dtype=np.float64).reshape(-1, 1)], axis=1)
    theta = np.concatenate([mean, quat, log_scale, opacity.reshape(-1, 1)], axis=1)
    lr = np.array([h.lr_mean] * 3 + [h.lr_quat] * 4 + [h.lr_scale] * 2 + [h.lr_opacity])
    m = h.beta1 * m + (1.0 - h.beta1) * g
    v = h.beta2 * v + (1.0 - h.beta2) * g * g
    m_hat = m / (1.0 - h.beta1 ** step)
    v_hat = v / (1.0 - h.beta2 ** step)
    theta = theta - lr * m_hat / (np.sqrt(v_hat) + h.eps)
    mean, quat, log_scale, opacity = theta[:, 0:3], theta[:, 3:7], theta[:, 7:9], theta[:, 9]
    opacity = np.clip(opacity, h.alpha_lo, h.alpha_hi)
    return mean, quat, log_scale, opacity, np.exp(log_scale), m, v, L_scale
