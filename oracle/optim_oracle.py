"""ORACLE — TEST INFRASTRUCTURE, NOT THE PRODUCT.

Plain numpy (fp64) statement of the two optimizer steps that sit on either side of the resident-delta pack at a round
boundary.  Only tests/ may import this.  Shares nothing with the CUDA path.

The paper names the optimizers and their hyper-parameters but prints no update formula ("Workers execute AdamW
(Loshchilov & Hutter, 2019) locally on their parameter subsets, while the server applies momentum"; Table 7:
"Local training uses AdamW with weight decay 0, betas (0.9, 0.95), and eps = 1e-8 ... DiLoCo/Nesterov uses server learning
rate 0.7 and momentum 0.9"; Alg. 2 l.19-20: Delta <- all-reduce, theta <- OuterOpt(Delta)).  The formulas
below are the cited methods' own (reading R13): decoupled-weight-decay Adam with bias correction, and SGD with
Nesterov momentum applied to the averaged outer gradient Delta = theta_round_start - theta_local (R10).
Pinned in tests/test_oracle_optim.py against torch.optim.AdamW and torch.optim.SGD(nesterov=True) (library routines) and
closed forms of the first step.
"""
from __future__ import annotations

import numpy as np


def adamw_step(w, g, m, v, step, lr, beta1=0.9, beta2=0.95, eps=1e-8, weight_decay=0.0):
    """One AdamW step (Loshchilov & Hutter 2019, Alg. 2) on fp64 copies; `step` counts from 1.  Returns (w, m, v)."""
    w, g, m, v = (np.asarray(a, dtype=np.float64) for a in (w, g, m, v))
    m = beta1 * m + (1.0 - beta1) * g
    v = beta2 * v + (1.0 - beta2) * g * g
    m_hat = m / (1.0 - beta1 ** step)
    v_hat = v / (1.0 - beta2 ** step)
    w = w - lr * weight_decay * w                      # decoupled weight decay
    w = w - lr * m_hat / (np.sqrt(v_hat) + eps)
    return w, m, v


def outer_nesterov_step(w_start, delta_avg, buf, lr=0.7, momentum=0.9):
    """Outer step on the replica-group average of delta = w_round_start - w_local (the payload of the pack kernel):
    buf <- momentum * buf + delta;  w <- w_start - lr * (delta + momentum * buf).   Returns (w_new, buf)."""
    w_start, delta_avg, buf = (np.asarray(a, dtype=np.float64) for a in (w_start, delta_avg, buf))
    buf = momentum * buf + delta_avg
    w_new = w_start - lr * (delta_avg + momentum * buf)
    return w_new, buf


def unpack_blocks(payload, elems, pack_slots, n_res):
    """payload [n_pack, sum(elems)] -> three [n_res, elems_i] arrays holding each packed slot's blocks (others zero) and the
    boolean mask of packed slots: the inverse of the pack layout (gate | up | down per slot)."""
    payload = np.asarray(payload)
    n_pack = payload.shape[0]
    slots = np.arange(n_pack) if pack_slots is None else np.asarray(pack_slots)
    outs = [np.zeros((n_res, e), payload.dtype) for e in elems]
    mask = np.zeros(n_res, bool)
    off = 0
    for i, e in enumerate(elems):
        outs[i][slots] = payload[:, off:off + e]
        off += e
    mask[slots] = True
    return outs, mask
