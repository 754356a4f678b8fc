"""Test-side glue: build a seeded problem from a workload, margin-clean it with the oracle, run oracle and CUDA path."""
from __future__ import annotations

import numpy as np

from paper_2606_19025_b200 import workloads as W

MARGIN = 1e-4  # BASELINE.json: routing is bit-exact on inputs whose top-k logit margins exceed 1e-4


class Problem:
    def __init__(self, w: W.MoEWorkload, n_res=None):
        self.w = w
        self.resident = W.resident_set(w, n_res)
        self.x = W.make_x(w)
        self.dy = W.make_dy(w)
        self.w_router = W.make_router(w)
        self.bias = W.router_bias(w)
        self.wg, self.wu, self.wd = W.make_resident_experts(w, self.resident)
        self.shared = W.make_shared_experts(w)


def margins(logits: np.ndarray, k: int) -> np.ndarray:
    """Smallest adjacent gap among the top k+1 logits of every token (fp64)."""
    E = logits.shape[1]
    srt = -np.sort(-logits, axis=1)
    kk = min(k + 1, E)
    if kk < 2:
        return np.full(logits.shape[0], np.inf)
    return (srt[:, :kk - 1] - srt[:, 1:kk]).min(1)


def margin_clean(p: Problem, oracle64, max_attempts=20) -> int:
    """Redraw token rows whose top-(k+1) adjacent logit gaps are below MARGIN; returns #redrawn."""
    w = p.w
    total = 0
    for attempt in range(max_attempts):
        r = oracle64.route(p.x, p.w_router, p.resident, w.k, w.gate_fn, w.gate_rule, w.temperature, p.bias, w.route_mode)
        bad = np.nonzero(margins(r["logits"], w.k) <= MARGIN)[0]   # the bar itself: margins must EXCEED 1e-4, nothing wider
        if len(bad) == 0:
            return total
        p.x[bad] = W.redraw_x_rows(w, bad, attempt)
        total += len(bad)
    raise AssertionError("margin cleaning did not converge")


def oracle_all(p: Problem, o, bwd=True):
    w = p.w
    r = o.route(p.x, p.w_router, p.resident, w.k, w.gate_fn, w.gate_rule, w.temperature, p.bias, w.route_mode)
    y = o.moe_fwd(p.x, r, p.resident, p.wg, p.wu, p.wd, p.shared, expert_fn=w.expert_fn)
    b = None
    if bwd:
        b = o.moe_bwd(p.x, p.dy, p.w_router, r, p.resident, p.wg, p.wu, p.wd, p.shared, w.gate_fn, w.gate_rule, w.temperature,
                      expert_fn=w.expert_fn)
    return r, y, b


def make_layer(p: Problem):
    from paper_2606_19025_b200.layer import SkipTokenMoE
    return SkipTokenMoE(p.w, p.resident, p.w_router, p.wg, p.wu, p.wd, p.shared, p.bias)


def rel_err(got, ref) -> float:
    """max|err| / max|ref| (BASELINE.json's measure); 0/0 -> 0."""
    got = np.asarray(got, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    den = np.abs(ref).max() if ref.size else 0.0
    num = np.abs(got - ref).max() if ref.size else 0.0
    if den == 0.0:
        return 0.0 if num == 0.0 else np.inf
    return float(num / den)


def t2n(t):
    import torch
    return t.detach().to(torch.float32).cpu().numpy()
