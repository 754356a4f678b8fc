"""Independent references used ONLY to pin the oracle (tests, -m "not gpu").

Two constructions that share nothing with oracle/fomoe_oracle.c:

* `brute_force_fwd`: pure-Python / numpy per-token loop that evaluates ALL E experts for every token and
  multiplies by an indicator (selected AND resident).  Tiny inputs only.
* `torch_dense_moe`: torch CPU float64 "standard top-k MoE over all E experts with W_down := 0 for experts
  outside S" (the zeroed-down-projection identity), evaluated densely with einsum; top-k from
  torch.topk; gradients from torch.autograd (no backward formula is typed here).
"""
from __future__ import annotations

import math

import numpy as np
import torch

GATE_SOFTMAX, GATE_SIGMOID = 0, 1
RULE_DROP_ONLY, RULE_RENORM_TOPK, RULE_RENORM_RESIDENT = 0, 1, 2
EXPERT_SWIGLU, EXPERT_SILU = 0, 1   # SILU: the paper's expert W_down silu(W_up x); W_gate is ignored


def tiny_problem(seed, T=6, d=5, E=4, k=2, F=3, n_res=2, n_sh=0, F_sh=0, wscale=0.5):
    """Random tiny problem in float64 with comfortable top-k margins (selection is piecewise constant)."""
    rng = np.random.default_rng(seed)
    while True:
        x = rng.standard_normal((T, d))
        w_r = rng.standard_normal((d, E)) * wscale
        z = x @ w_r
        srt = np.sort(z, axis=1)[:, ::-1]
        if E == 1 or np.min(srt[:, :min(k, E - 1)] - srt[:, 1:min(k, E - 1) + 1]) > 1e-2:
            break
    resident = np.sort(rng.permutation(E)[:n_res]).astype(np.int32)
    full = dict(  # weights for ALL E experts (the references need them; the oracle gets resident ones only)
        w_gate=rng.standard_normal((E, F, d)) * wscale, w_up=rng.standard_normal((E, F, d)) * wscale,
        w_down=rng.standard_normal((E, d, F)) * wscale)
    shared = None
    if n_sh:
        shared = (rng.standard_normal((n_sh, F_sh, d)) * wscale, rng.standard_normal((n_sh, F_sh, d)) * wscale,
                  rng.standard_normal((n_sh, d, F_sh)) * wscale)
    dy = rng.standard_normal((T, d))
    return dict(x=x, w_r=w_r, resident=resident, full=full, shared=shared, dy=dy, k=k, E=E)


def resident_stacks(prob):
    S = prob["resident"]
    f = prob["full"]
    return f["w_gate"][S].copy(), f["w_up"][S].copy(), f["w_down"][S].copy()


def _gate_probs(z, gate_fn):
    if gate_fn == GATE_SIGMOID:
        return [1.0 / (1.0 + math.exp(-v)) for v in z]
    m = max(z)
    ex = [math.exp(v - m) for v in z]
    s = sum(ex)
    return [v / s for v in ex]


def brute_force_fwd(prob, gate_fn=GATE_SOFTMAX, gate_rule=RULE_DROP_ONLY, tau=1.0, bias=None, expert_fn=EXPERT_SWIGLU):
    """All-experts-times-indicator evaluation with Python loops."""
    x, w_r, S, full, k, E = prob["x"], prob["w_r"], set(int(s) for s in prob["resident"]), prob["full"], prob["k"], prob["E"]
    T, d = x.shape
    y = np.zeros((T, d))
    for t in range(T):
        z = [sum(x[t, i] * w_r[i, e] for i in range(d)) / tau + (0.0 if bias is None else float(bias[e])) for e in range(E)]
        p = _gate_probs(z, gate_fn)
        order = sorted(range(E), key=lambda e: (-z[e], e))  # full stable sort, first k
        sel = order[:k]
        s_all = sum(p[e] for e in sel)
        s_kept = sum(p[e] for e in sel if e in S)
        for e in range(E):  # every expert is evaluated; the indicator zeroes the rest
            ind = 1.0 if (e in sel and e in S) else 0.0
            if expert_fn == EXPERT_SILU:
                v = full["w_up"][e] @ x[t]
                h = v / (1.0 + np.exp(-v))
            else:
                a = full["w_gate"][e] @ x[t]
                u = full["w_up"][e] @ x[t]
                h = a / (1.0 + np.exp(-a)) * u
            o = full["w_down"][e] @ h
            if gate_rule == RULE_DROP_ONLY:
                g = p[e]
            elif gate_rule == RULE_RENORM_TOPK:
                g = p[e] / s_all
            else:
                g = p[e] / s_kept if s_kept > 0 else 0.0
            y[t] += ind * g * o
        if prob["shared"] is not None:
            sg, su, sd = prob["shared"]
            for s in range(su.shape[0]):
                if expert_fn == EXPERT_SILU:
                    v = su[s] @ x[t]
                    y[t] += sd[s] @ (v / (1.0 + np.exp(-v)))
                    continue
                a = sg[s] @ x[t]
                u = su[s] @ x[t]
                y[t] += sd[s] @ (a / (1.0 + np.exp(-a)) * u)
    return y


def torch_dense_moe(prob, gate_fn=GATE_SOFTMAX, gate_rule=RULE_DROP_ONLY, tau=1.0, bias=None, expert_fn=EXPERT_SWIGLU):
    """Returns (y, grads dict) for L = sum(dy * y).  grads: dx, dw_router, dw_gate/up/down (resident slots), d_sh_*."""
    f64 = torch.float64
    x = torch.tensor(prob["x"], dtype=f64, requires_grad=True)
    w_r = torch.tensor(prob["w_r"], dtype=f64, requires_grad=True)
    S = torch.tensor(prob["resident"], dtype=torch.long)
    E, k = prob["E"], prob["k"]
    wg = torch.tensor(prob["full"]["w_gate"], dtype=f64, requires_grad=True)
    wu = torch.tensor(prob["full"]["w_up"], dtype=f64, requires_grad=True)
    wd_full = torch.tensor(prob["full"]["w_down"], dtype=f64, requires_grad=True)
    res_mask = torch.zeros(E, dtype=f64)
    res_mask[S] = 1.0
    wd = wd_full * res_mask[:, None, None]          # W_down := 0 outside S
    z = x @ w_r / tau
    if bias is not None:
        z = z + torch.tensor(bias, dtype=f64)
    p = torch.sigmoid(z) if gate_fn == GATE_SIGMOID else torch.softmax(z, dim=-1)
    idx = torch.topk(z, k, dim=-1).indices
    sel = torch.zeros_like(z).scatter(1, idx, 1.0)   # selected indicator [T,E]
    if gate_rule == RULE_DROP_ONLY:
        g = p * sel
    elif gate_rule == RULE_RENORM_TOPK:
        g = p * sel / (p * sel).sum(-1, keepdim=True)
    else:
        kept = sel * res_mask
        den = (p * kept).sum(-1, keepdim=True)
        g = torch.where(den > 0, p * kept / torch.where(den > 0, den, torch.ones_like(den)), torch.zeros_like(p))
    u = torch.einsum("td,efd->tef", x, wu)
    if expert_fn == EXPERT_SILU:
        h = torch.nn.functional.silu(u)
    else:
        a = torch.einsum("td,efd->tef", x, wg)
        h = torch.nn.functional.silu(a) * u
    o = torch.einsum("tef,edf->ted", h, wd)
    y = (g[:, :, None] * o).sum(1)
    sh = None
    if prob["shared"] is not None:
        sh = [torch.tensor(s, dtype=f64, requires_grad=True) for s in prob["shared"]]
        u2 = torch.einsum("td,sfd->tsf", x, sh[1])
        if expert_fn == EXPERT_SILU:
            h2 = torch.nn.functional.silu(u2)
        else:
            h2 = torch.nn.functional.silu(torch.einsum("td,sfd->tsf", x, sh[0])) * u2
        y = y + torch.einsum("tsf,sdf->td", h2, sh[2])
    L = (y * torch.tensor(prob["dy"], dtype=f64)).sum()
    L.backward()
    Sn = prob["resident"]
    silu_form = expert_fn == EXPERT_SILU
    wg_grad = np.zeros_like(prob["full"]["w_gate"]) if silu_form else wg.grad.numpy()
    grads = dict(dx=x.grad.numpy(), dw_router=w_r.grad.numpy(), dw_up=wu.grad.numpy()[Sn], dw_down=wd_full.grad.numpy()[Sn])
    if not silu_form:
        grads["dw_gate"] = wg_grad[Sn]
    ghost = np.setdiff1d(np.arange(E), Sn)
    grads["ghost_grad_max"] = max([float(np.abs(wg_grad[ghost]).max(initial=0.0)),
                                   float(np.abs(wu.grad.numpy()[ghost]).max(initial=0.0)),
                                   float(np.abs(wd_full.grad.numpy()[ghost]).max(initial=0.0))])
    if sh is not None:
        grads.update(d_sh_up=sh[1].grad.numpy(), d_sh_down=sh[2].grad.numpy())
        if not silu_form:
            grads["d_sh_gate"] = sh[0].grad.numpy()
    return y.detach().numpy(), grads
