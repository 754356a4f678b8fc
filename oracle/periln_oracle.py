"""ORACLE — TEST INFRASTRUCTURE, NOT THE PRODUCT.

Plain numpy (fp64) statement of the Peripheral-LayerNorm steps either side of the MoE block:

    x_{l+1} = x_l + alpha * LN_post(F(LN_pre(x_l)))          PAPER.md:571 Eq. 15; depth multiplier alpha: Fig. 12

"applies normalization exclusively to the residual branches — both immediately preceding (Pre-LN) and following (Post-LN)
the computational blocks — while preserving a linear, un-normalized main data path".  Readings (DESIGN.md
R14): LN is the standard LayerNorm over d_model with learnable gain and bias and eps = 1e-5 (the paper gives none); the
depth multiplier multiplies the post-LN output (before it, it would be erased by the normalisation).
Only tests/ may import this.  Pinned in tests/test_oracle_periln.py against torch.nn.functional.layer_norm + autograd.
"""
from __future__ import annotations

import numpy as np


def ln_fwd(x, gamma, beta, eps=1e-5):
    """Row-wise LayerNorm: returns (gamma * xhat + beta, mean [T], rstd [T])."""
    x = np.asarray(x, np.float64)
    mean = x.mean(axis=1)
    var = ((x - mean[:, None]) ** 2).mean(axis=1)          # biased variance, as LayerNorm defines it
    rstd = 1.0 / np.sqrt(var + eps)
    xhat = (x - mean[:, None]) * rstd[:, None]
    return np.asarray(gamma, np.float64) * xhat + np.asarray(beta, np.float64), mean, rstd


def ln_bwd(dout, x, mean, rstd, gamma):
    """Backward of ln_fwd for upstream dout: returns (dx, dgamma, dbeta)."""
    dout, x, gamma = np.asarray(dout, np.float64), np.asarray(x, np.float64), np.asarray(gamma, np.float64)
    xhat = (x - mean[:, None]) * rstd[:, None]
    dxhat = dout * gamma
    dx = rstd[:, None] * (dxhat - dxhat.mean(axis=1, keepdims=True) - xhat * (dxhat * xhat).mean(axis=1, keepdims=True))
    return dx, (dout * xhat).sum(axis=0), dout.sum(axis=0)


def periln_post_fwd(x, y, gamma, beta, alpha=1.0, eps=1e-5):
    """out = x + alpha * LN(y); returns (out, mean, rstd)."""
    ln, mean, rstd = ln_fwd(y, gamma, beta, eps)
    return np.asarray(x, np.float64) + alpha * ln, mean, rstd


def periln_post_bwd(dout, y, mean, rstd, gamma, alpha=1.0):
    """Gradients of periln_post_fwd w.r.t. y, gamma, beta (the residual path passes dout to x unchanged)."""
    dy, dg, db = ln_bwd(alpha * np.asarray(dout, np.float64), y, mean, rstd, gamma)
    return dy, dg, db


def periln_pre_bwd(dxn, x, mean, rstd, gamma, dout):
    """dx of the whole block input: the residual path's dout plus the pre-LN branch; also dgamma, dbeta of the pre-LN."""
    dx, dg, db = ln_bwd(dxn, x, mean, rstd, gamma)
    return dx + np.asarray(dout, np.float64), dg, db
