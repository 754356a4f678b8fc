"""Seeded synthetic inputs for the skip-token MoE layer (BASELINE.json `configs`).

This module holds NONE of the method's arithmetic: it only draws random tensors, rounds them to the
storage dtype and draws the resident-expert set.  It is the one module both the CUDA path's tests /
bench and the oracle's tests may import; it imports neither of them.

Recipe:
  * independent streams keyed by (seed, tensor tag, index) so expert e's weights do not depend on which
    set is resident (`numpy.random.default_rng([seed, tag, index])`, PCG64);
  * x, dy ~ N(0,1): stands in for the unit-variance Peri-LN output that feeds router and experts
    (§B.1, 597 §B.3.2);  W_r and all expert weights ~ N(0, 0.02^2);
  * bf16 configs: x, dy and expert weights are rounded to bf16 (round-to-nearest-even) here and the SAME
    bits go to both sides; W_r stays fp32 (BASELINE.json config 2 "fp32 router");
  * resident set S (§3.3.1, N_le of N_e experts): C1 = {0,1,2,3}; otherwise the first n_res
    entries of ONE seeded permutation of [0,E), sorted, so the C4 sweep's sets are nested;
  * C4 skew: b_e = -alpha * ln(rank_e), rank = a seeded permutation of 1..E (BASELINE.json config 4).
"""
from __future__ import annotations

from dataclasses import dataclass, replace
from typing import Optional

import numpy as np

# tensor tags (stream keys)
_TAG = {
    "x": 1, "dy": 2, "w_router": 3, "w_gate": 4, "w_up": 5, "w_down": 6,
    "sh_gate": 7, "sh_up": 8, "sh_down": 9, "resident": 10, "zipf_rank": 11,
    "x_redraw": 12, "snapshot": 13,
}

GATE_SOFTMAX, GATE_SIGMOID = 0, 1
RULE_DROP_ONLY, RULE_RENORM_TOPK, RULE_RENORM_RESIDENT = 0, 1, 2


@dataclass(frozen=True)
class MoEWorkload:
    name: str
    T: int            # tokens (batch x seq flattened)
    d: int            # d_model
    E: int            # routed experts N_e
    k: int            # top-k
    F: int            # d_ff of a routed expert
    n_res: int        # resident experts N_le
    n_sh: int = 0     # always-resident shared experts
    F_sh: int = 0     # d_ff of a shared expert
    dtype: str = "bf16"      # "f32" | "bf16": x, expert weights, y, dy, dx, dW
    zipf_alpha: float = 0.0  # 0 = no router bias
    gate_fn: int = GATE_SOFTMAX       # BASELINE.json: softmax; paper Eq. 17: sigmoid
    gate_rule: int = RULE_DROP_ONLY   # paper: drop-only
    temperature: float = 1.0
    route_mode: int = 0               # 0 = skip-token, 1 = forced-local (partitioned router)
    expert_fn: int = 0                # 0 = SwiGLU (BASELINE.json), 1 = the paper's W_down silu(W_up x)
    seed: int = 0
    fixed_resident: Optional[tuple] = None

    def with_(self, **kw) -> "MoEWorkload":
        return replace(self, **kw)


# BASELINE.json `configs` 1..5 (C4 = C3 shapes, n_res swept, Zipf bias)
CONFIGS = {
    "C1": MoEWorkload("C1", T=256, d=64, E=8, k=2, F=128, n_res=4, dtype="f32", fixed_resident=(0, 1, 2, 3)),
    "C2": MoEWorkload("C2", T=8192, d=1024, E=16, k=2, F=2816, n_res=8),
    "C3": MoEWorkload("C3", T=16384, d=2048, E=64, k=6, F=1408, n_res=16, n_sh=2, F_sh=1408),
    "C4": MoEWorkload("C4", T=16384, d=2048, E=64, k=6, F=1408, n_res=16, n_sh=2, F_sh=1408, zipf_alpha=1.0),
    "C5": MoEWorkload("C5", T=32768, d=4096, E=128, k=8, F=1536, n_res=32),
}
C4_RESIDENT_SWEEP = (8, 16, 32, 64)
EXPERT_SWIGLU, EXPERT_SILU = 0, 1
ROUTE_SKIP_TOKEN, ROUTE_FORCED_LOCAL = 0, 1
# The paper's own sigma-MoE layer at its Table 1 shapes: sigmoid gate (Eq. 17), two-matrix SiLU expert of
# width d_expert = 128 (Eq. 16, §B.3.1), N_active of N_experts, sequence length 2048 x 8 sequences;
# half of the experts resident (overlap O_e / M = 1/2).  P0 is a small fp32 case for element-wise parity.
CONFIGS.update({
    "P0": MoEWorkload("P0", T=256, d=64, E=8, k=2, F=32, n_res=4, dtype="f32", gate_fn=GATE_SIGMOID, expert_fn=EXPERT_SILU),
    "P1": MoEWorkload("P1", T=16384, d=512, E=16, k=4, F=128, n_res=8, gate_fn=GATE_SIGMOID, expert_fn=EXPERT_SILU),    # Medium (150M)
    "P2": MoEWorkload("P2", T=16384, d=1024, E=32, k=8, F=128, n_res=16, gate_fn=GATE_SIGMOID, expert_fn=EXPERT_SILU),  # Large (2B)
    "P3": MoEWorkload("P3", T=16384, d=2048, E=64, k=16, F=128, n_res=32, gate_fn=GATE_SIGMOID, expert_fn=EXPERT_SILU), # XL (13B)
})


def config(name: str) -> MoEWorkload:
    return CONFIGS[name]


# ---------------------------------------------------------------------------------------------------
# dtype helpers (storage only)
# ---------------------------------------------------------------------------------------------------
def f32_to_bf16_bits(a: np.ndarray) -> np.ndarray:
    """fp32 -> bf16 bit pattern (uint16), round-to-nearest-even. Inputs are finite."""
    a = np.ascontiguousarray(a, dtype=np.float32)
    u = a.view(np.uint32)
    r = ((u >> np.uint32(16)) & np.uint32(1)) + np.uint32(0x7FFF)
    return ((u + r) >> np.uint32(16)).astype(np.uint16)


def bf16_bits_to_f32(b: np.ndarray) -> np.ndarray:
    return (np.ascontiguousarray(b, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32)


def bf16_round(a: np.ndarray) -> np.ndarray:
    """fp32 values rounded to the bf16 grid, still stored as fp32."""
    return bf16_bits_to_f32(f32_to_bf16_bits(a))


def _store(w: MoEWorkload, a: np.ndarray) -> np.ndarray:
    """Values as both sides see them: fp32 array holding storage-dtype-exact values."""
    a = np.ascontiguousarray(a, dtype=np.float32)
    return bf16_round(a) if w.dtype == "bf16" else a


def _rng(w: MoEWorkload, tag: str, index: int = 0, sub: int = 0) -> np.random.Generator:
    return np.random.default_rng([w.seed, _TAG[tag], index, sub])


def _normal(rng: np.random.Generator, shape, scale: float = 1.0) -> np.ndarray:
    a = rng.standard_normal(shape, dtype=np.float32)
    if scale != 1.0:
        a *= np.float32(scale)
    return a


# ---------------------------------------------------------------------------------------------------
# tensors
# ---------------------------------------------------------------------------------------------------
def make_x(w: MoEWorkload) -> np.ndarray:
    """Tokens x [T,d], N(0,1), storage-dtype-exact fp32."""
    return _store(w, _normal(_rng(w, "x"), (w.T, w.d)))


def redraw_x_rows(w: MoEWorkload, rows: np.ndarray, attempt: int) -> np.ndarray:
    """Fresh draws for the given token rows (used by the tests' margin cleaning)."""
    out = np.empty((len(rows), w.d), dtype=np.float32)
    for i, t in enumerate(np.asarray(rows, dtype=np.int64)):
        out[i] = _normal(_rng(w, "x_redraw", int(t), attempt), (w.d,))
    return _store(w, out)


def make_dy(w: MoEWorkload) -> np.ndarray:
    """Upstream gradient dy [T,d], N(0,1)."""
    return _store(w, _normal(_rng(w, "dy"), (w.T, w.d)))


def make_router(w: MoEWorkload) -> np.ndarray:
    """Router W_r [d,E] fp32, N(0,0.02^2): full, unpartitioned (§3.3.3)."""
    return _normal(_rng(w, "w_router"), (w.d, w.E), 0.02)


def make_expert_master(w: MoEWorkload, e: int):
    """fp32 master weights of routed expert e: (W_gate [F,d], W_up [F,d], W_down [d,F])."""
    return (_normal(_rng(w, "w_gate", e), (w.F, w.d), 0.02),
            _normal(_rng(w, "w_up", e), (w.F, w.d), 0.02),
            _normal(_rng(w, "w_down", e), (w.d, w.F), 0.02))


def make_expert(w: MoEWorkload, e: int):
    """Compute-dtype weights of routed expert e (storage-dtype-exact fp32)."""
    return tuple(_store(w, m) for m in make_expert_master(w, e))


def make_resident_experts(w: MoEWorkload, resident: np.ndarray):
    """Resident-compact stacks W_gate [n_res,F,d], W_up [n_res,F,d], W_down [n_res,d,F]; slot i <-> resident[i]
    (stored only for resident experts: the memory saving is the point)."""
    n = len(resident)
    silu = w.expert_fn == EXPERT_SILU   # the paper's expert has no W_gate: None in its place
    wg = None if silu else np.empty((n, w.F, w.d), dtype=np.float32)
    wu = np.empty((n, w.F, w.d), dtype=np.float32)
    wd = np.empty((n, w.d, w.F), dtype=np.float32)
    for i, e in enumerate(resident):
        g, wu[i], wd[i] = make_expert(w, int(e))
        if not silu:
            wg[i] = g
    return wg, wu, wd


def make_shared_experts(w: MoEWorkload):
    """Shared (always-resident, dense) experts: [n_sh,F_sh,d], [n_sh,F_sh,d], [n_sh,d,F_sh]; None if n_sh=0."""
    if w.n_sh == 0:
        return None
    sg = None if w.expert_fn == EXPERT_SILU else np.stack([_store(w, _normal(_rng(w, "sh_gate", s), (w.F_sh, w.d), 0.02)) for s in range(w.n_sh)])
    su = np.stack([_store(w, _normal(_rng(w, "sh_up", s), (w.F_sh, w.d), 0.02)) for s in range(w.n_sh)])
    sd = np.stack([_store(w, _normal(_rng(w, "sh_down", s), (w.d, w.F_sh), 0.02)) for s in range(w.n_sh)])
    return sg, su, sd


def resident_set(w: MoEWorkload, n_res: Optional[int] = None) -> np.ndarray:
    """Ascending global ids of the resident experts S (int32). Nested prefixes of one permutation."""
    n = w.n_res if n_res is None else n_res
    if w.fixed_resident is not None and n == len(w.fixed_resident):
        return np.asarray(w.fixed_resident, dtype=np.int32)
    perm = _rng(w, "resident").permutation(w.E)
    return np.sort(perm[:n]).astype(np.int32)


def router_bias(w: MoEWorkload) -> Optional[np.ndarray]:
    """Zipf load-skew device of BASELINE.json config 4: b_e = -alpha ln(rank_e), fp32 [E]; None if alpha=0."""
    if w.zipf_alpha == 0.0:
        return None
    rank = _rng(w, "zipf_rank").permutation(w.E) + 1
    return (-w.zipf_alpha * np.log(rank.astype(np.float64))).astype(np.float32)


def make_round_start_snapshot(w: MoEWorkload, e: int):
    """fp32 round-start copies of expert e's master weights for the delta pack (Alg. 2 l.19):
    master + N(0, 1e-3^2), i.e. what K local steps might have moved."""
    mg, mu, md = make_expert_master(w, e)
    r = _rng(w, "snapshot", e)
    return (mg + _normal(r, mg.shape, 1e-3), mu + _normal(r, mu.shape, 1e-3), md + _normal(r, md.shape, 1e-3))
