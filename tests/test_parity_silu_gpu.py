"""Parity of the paper-exact sigma-MoE layer — sigmoid gate (Eq. 17), two-matrix SiLU expert
W_down silu(W_up x) of width d_expert = 128 (§B.3.1, Eq. 16), drop-only skip-token rule
— against the fp64 oracle: element by element on small cases (fp32 SIMT and bf16 tcgen05 paths), and on sampled outputs at
the paper's Table 1 shapes in the CUDA-graph launch configuration bench.py times."""
import numpy as np
import pytest

import helpers as H
from paper_2606_19025_b200 import workloads as W
from test_parity_gpu import run_and_compare

pytestmark = pytest.mark.gpu
TOL = 2e-2


def test_p0_fp32_full(oracle64):
    errs, _ = run_and_compare(H.Problem(W.config("P0")), oracle64)
    print("P0", errs)


@pytest.mark.parametrize("rule", [W.RULE_DROP_ONLY, W.RULE_RENORM_RESIDENT])
@pytest.mark.parametrize("gate_fn", [W.GATE_SIGMOID, W.GATE_SOFTMAX])
def test_small_bf16_full(oracle64, gate_fn, rule):
    """Several row tiles per slot, a ragged tail, one shared expert, F = 128 (a half-width column tile)."""
    w = W.MoEWorkload("silu_small", T=1500, d=256, E=16, k=4, F=128, n_res=7, n_sh=1, F_sh=192, gate_fn=gate_fn, gate_rule=rule,
                      expert_fn=W.EXPERT_SILU, seed=3)
    errs, _ = run_and_compare(H.Problem(w), oracle64)
    print("silu_small", errs)


def test_small_bf16_wide_expert(oracle64):
    """d_ff wider than one 256-column tile pair, odd tile counts."""
    w = W.MoEWorkload("silu_wide", T=1100, d=320, E=8, k=2, F=448, n_res=5, gate_fn=W.GATE_SIGMOID, expert_fn=W.EXPERT_SILU, seed=4)
    errs, _ = run_and_compare(H.Problem(w), oracle64)
    print("silu_wide", errs)


@pytest.mark.parametrize("E,k,n_res", [(64, 16, 32), (128, 32, 48), (32, 8, 16)])
def test_table1_active_counts(oracle64, E, k, n_res):
    """N_active = 8, 16, 32 of N_experts = 32, 64, 128 (Table 1) on the tensor-core router: ordered top-k
    lists, counts and the permutation bit-exact; outputs and gradients element by element."""
    w = W.MoEWorkload("silu_k", T=700, d=192, E=E, k=k, F=128, n_res=n_res, gate_fn=W.GATE_SIGMOID, expert_fn=W.EXPERT_SILU, seed=6)
    errs, _ = run_and_compare(H.Problem(w), oracle64)
    print("silu_k", E, k, errs)


def test_edge_cases_silu(oracle64):
    for kw in (dict(n_res=0, n_sh=1, F_sh=128), dict(n_res=16), dict(T=1, n_res=8), dict(T=127, n_res=3)):
        base = dict(T=300, d=128, E=16, k=4, F=128, n_res=8, gate_fn=W.GATE_SIGMOID, expert_fn=W.EXPERT_SILU, seed=5)
        base.update(kw)
        run_and_compare(H.Problem(W.MoEWorkload("silu_edge", **base)), oracle64)


@pytest.mark.parametrize("name", ["P1", "P2", "P3"])
def test_paper_shapes_sampled(oracle64, name):
    import torch
    w = W.config(name)
    p = H.Problem(w)
    H.margin_clean(p, oracle64)
    r = oracle64.route(p.x, p.w_router, p.resident, w.k, w.gate_fn, w.gate_rule, w.temperature, p.bias)
    layer = H.make_layer(p)
    x, dy = layer.to_dev(p.x), layer.to_dev(p.dy)
    step = layer.capture_step(x, dy)
    step()
    torch.cuda.synchronize()
    g = layer.routing_numpy()
    for key in ("topk_idx", "counts", "offsets", "row_token", "pair_row"):
        assert np.array_equal(g[key], r[key]), key
    assert H.rel_err(g["probs"], r["probs"]) <= 1e-4 and H.rel_err(g["gate"], r["gate"]) <= 1e-4
    kept = np.isin(r["topk_idx"], p.resident)
    assert abs(g["P"] / (w.T * w.k) - len(p.resident) / w.E) < 0.03     # sigma_st = N_le / N_e (Eq. 2)
    y = H.t2n(layer.y)
    none = ~kept.any(1)
    assert np.all(y[none] == 0)
    rng = np.random.default_rng(12)
    idx = np.sort(rng.choice(np.nonzero(kept.any(1))[0], 48, replace=False)).astype(np.int64)
    rs = oracle64.route(p.x[idx], p.w_router, p.resident, w.k, w.gate_fn, w.gate_rule, w.temperature, p.bias)
    ys = oracle64.moe_fwd(p.x[idx], rs, p.resident, None, p.wu, p.wd, None, expert_fn=w.expert_fn)
    bs = oracle64.moe_bwd(p.x[idx], p.dy[idx], p.w_router, rs, p.resident, None, p.wu, p.wd, None, w.gate_fn, w.gate_rule,
                          w.temperature, expert_fn=w.expert_fn)
    errs = {"y": H.rel_err(y[idx], ys), "dx": H.rel_err(H.t2n(layer.dx)[idx], bs["dx"])}
    for slot in sorted({0, len(p.resident) - 1, int(np.argmax(r["counts"])), int(np.argmin(r["counts"]))}):
        f_idx = np.sort(rng.choice(w.F, 3, replace=False)).astype(np.int32)
        _, ou, od = oracle64.dw_sample(p.x, p.dy, r, p.resident, slot, f_idx, None, p.wu[slot], p.wd[slot], expert_fn=w.expert_fn)
        fi = torch.from_numpy(f_idx.astype(np.int64)).cuda()
        errs[f"dw_up[{slot}]"] = H.rel_err(H.t2n(layer.dw_up[slot][fi]), ou)
        errs[f"dw_down[{slot}]"] = H.rel_err(H.t2n(layer.dw_down[slot][:, fi]).T, od)
    dy2 = np.zeros_like(p.dy)
    dy2[idx] = p.dy[idx]
    layer.backward(layer.to_dev(dy2), x)
    torch.cuda.synchronize()
    for key, t in dict(dw_router=layer.dw_router, dw_up=layer.dw_up, dw_down=layer.dw_down).items():
        errs["sparse " + key] = H.rel_err(H.t2n(t), bs[key])
    print(name, "P", g["P"], {k: f"{v:.1e}" for k, v in errs.items()})
    bad = {k: v for k, v in errs.items() if not v <= TOL}
    assert not bad, bad


# ---- forced-local routing: partitioned router, every selected pair is kept ----
@pytest.mark.parametrize("expert_fn", [W.EXPERT_SWIGLU, W.EXPERT_SILU])
@pytest.mark.parametrize("gate_fn", [W.GATE_SIGMOID, W.GATE_SOFTMAX])
def test_forced_local_bf16_full(oracle64, gate_fn, expert_fn):
    w = W.MoEWorkload("forced_bf16", T=1300, d=256, E=16, k=4, F=192, n_res=6, n_sh=1, F_sh=128, gate_fn=gate_fn,
                      expert_fn=expert_fn, route_mode=W.ROUTE_FORCED_LOCAL, seed=7)
    p = H.Problem(w)
    errs, layer = run_and_compare(p, oracle64)
    g = layer.routing_numpy()
    assert g["P"] == w.T * w.k and np.isin(g["topk_idx"], p.resident).all()      # nothing is skipped
    ghost = np.setdiff1d(np.arange(w.E), p.resident)
    assert np.all(g["probs"][:, ghost] == 0) and np.all(H.t2n(layer.dw_router)[:, ghost] == 0)
    print("forced_bf16", errs)


def test_forced_local_fp32_full(oracle64):
    w = W.config("P0").with_(route_mode=W.ROUTE_FORCED_LOCAL, n_res=5)
    errs, layer = run_and_compare(H.Problem(w), oracle64)
    assert layer.routing_numpy()["P"] == w.T * w.k
    print("forced_f32", errs)


def test_forced_local_rejects_k_above_n_res():
    from paper_2606_19025_b200 import binding as B
    cfg = B.make_config(T=64, d_model=64, E=8, top_k=4, d_ff=64, route_mode=B.FOMOE_ROUTE_FORCED_LOCAL)
    with pytest.raises(B.FomoeError):
        B.fomoe_workspace_bytes(cfg, 3)
