"""Parity of the CUDA path (through the C ABI) against the fp64 oracle, element by element, on seeded inputs.

Bars (BASELINE.json north_star): routing indices / counts / offsets / permutation bit-exact on margin-cleaned inputs;
fp32 outputs and gradients max|err|/max|ref| <= 1e-4; bf16 <= 2e-2.
"""
import numpy as np
import pytest

import helpers as H
from paper_2606_19025_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL = {"f32": 1e-4, "bf16": 2e-2}
INT_KEYS = ("topk_idx", "counts", "offsets", "row_token", "pair_row")


def run_and_compare(p: H.Problem, oracle64, bwd=True, clean=True):
    import torch
    if clean:
        H.margin_clean(p, oracle64)
    r, y, b = H.oracle_all(p, oracle64, bwd)
    layer = H.make_layer(p)
    x, dy = layer.to_dev(p.x), layer.to_dev(p.dy)
    layer.route(x)
    g = layer.routing_numpy()
    for key in INT_KEYS:
        assert np.array_equal(g[key], r[key]), key
    assert H.rel_err(g["probs"], r["probs"]) <= 1e-5
    assert H.rel_err(g["gate"], r["gate"]) <= 1e-5
    assert np.all(g["gate"][r["pair_row"] < 0] == 0)
    tol = TOL[p.w.dtype]
    layer.forward(x)
    yg = H.t2n(layer.y)
    errs = {"y": H.rel_err(yg, y)}
    none_kept = (r["pair_row"] < 0).all(1)
    if p.shared is None and none_kept.any():
        assert np.all(yg[none_kept] == 0)  # exactly zero rows
    if bwd:
        layer.backward(dy, x)
        torch.cuda.synchronize()
        got = dict(dx=layer.dx, dw_router=layer.dw_router, dw_gate=layer.dw_gate, dw_up=layer.dw_up, dw_down=layer.dw_down)
        if p.shared is not None:
            got.update(d_sh_gate=layer.d_shared[0], d_sh_up=layer.d_shared[1], d_sh_down=layer.d_shared[2])
        for key, t in got.items():
            if t is not None and t.numel():   # (None: W_gate does not exist in the paper's two-matrix expert)
                errs[key] = H.rel_err(H.t2n(t), b[key])
    bad = {k: v for k, v in errs.items() if not v <= tol}
    assert not bad, (bad, errs)
    return errs, layer


def test_config1_fp32_full(oracle64):
    """BASELINE.json config 1: tiny fp32 layer, forward + backward vs oracle."""
    errs, _ = run_and_compare(H.Problem(W.config("C1")), oracle64)
    print("C1", errs)


@pytest.mark.parametrize("gate_fn", [W.GATE_SOFTMAX, W.GATE_SIGMOID])
@pytest.mark.parametrize("rule", [W.RULE_DROP_ONLY, W.RULE_RENORM_TOPK, W.RULE_RENORM_RESIDENT])
def test_config1_gate_variants(oracle64, gate_fn, rule):
    run_and_compare(H.Problem(W.config("C1").with_(gate_fn=gate_fn, gate_rule=rule, temperature=0.8)), oracle64)


@pytest.mark.parametrize("dtype", ["f32", "bf16"])
def test_midsize_ragged_with_shared(oracle64, dtype):
    """Several row tiles, ragged T (not a tile multiple), odd expert counts, shared experts, Zipf bias."""
    w = W.MoEWorkload("mid", T=777, d=192, E=12, k=3, F=320, n_res=5, n_sh=2, F_sh=256, dtype=dtype, zipf_alpha=1.0, seed=3)
    errs, _ = run_and_compare(H.Problem(w), oracle64)
    print("mid", dtype, errs)


@pytest.mark.parametrize("dtype", ["f32", "bf16"])
def test_odd_shapes_scalar_paths(oracle64, dtype):
    """d, F not multiples of the vector / tile sizes."""
    w = W.MoEWorkload("odd", T=130, d=50, E=5, k=2, F=70, n_res=3, n_sh=1, F_sh=33, dtype=dtype, seed=4)
    run_and_compare(H.Problem(w), oracle64)


@pytest.mark.parametrize("n_res", [0, 1, 8])
def test_resident_extremes(oracle64, n_res):
    """n_res = 0 (everything skipped), 1, and E (all resident == standard top-k MoE)."""
    w = W.MoEWorkload("ext", T=300, d=64, E=8, k=2, F=128, n_res=n_res, dtype="f32", seed=5)
    errs, layer = run_and_compare(H.Problem(w), oracle64)
    if n_res == 0:
        assert float(layer.y.abs().max()) == 0.0 and float(layer.dw_router.abs().max()) == 0.0


def test_empty_batch(oracle64):
    """T = 0: nothing to route; weight gradients are exact zeros."""
    import torch
    p = H.Problem(W.MoEWorkload("empty", T=0, d=64, E=8, k=2, F=64, n_res=4, dtype="f32", seed=6))
    layer = H.make_layer(p)
    x, dy = layer.to_dev(p.x), layer.to_dev(p.dy)
    layer.step(x, dy)
    torch.cuda.synchronize()
    g = layer.routing_numpy()
    assert g["P"] == 0 and np.all(g["counts"] == 0) and np.all(g["offsets"] == 0)
    for t in (layer.dw_router, layer.dw_gate, layer.dw_up, layer.dw_down):
        assert float(t.abs().max()) == 0.0


def test_single_token_and_k_equals_E(oracle64):
    run_and_compare(H.Problem(W.MoEWorkload("one", T=1, d=64, E=4, k=4, F=64, n_res=2, dtype="f32", seed=6)), oracle64)


def test_large_E_topk8(oracle64):
    w = W.MoEWorkload("bigE", T=257, d=128, E=128, k=8, F=64, n_res=32, dtype="bf16", seed=7)
    run_and_compare(H.Problem(w), oracle64)


def test_wide_router_feeds_tensor_core_gemms(oracle64):
    """E = 192 > 128: the fp32 SIMT router (any E <= 512) in front of the tcgen05 expert GEMMs and tensor-core router backward."""
    w = W.MoEWorkload("wideE", T=520, d=128, E=192, k=4, F=128, n_res=40, dtype="bf16", gate_fn=W.GATE_SIGMOID, seed=10)
    errs, _ = run_and_compare(H.Problem(w), oracle64)
    print("wideE", errs)


def test_empty_batch_bf16(oracle64):
    """T = 0 on the tensor-core path: counts / offsets zero, weight gradients exactly zero, nothing hangs."""
    import torch
    p = H.Problem(W.MoEWorkload("empty_bf16", T=0, d=128, E=8, k=2, F=128, n_res=4, n_sh=1, F_sh=64, dtype="bf16", seed=6))
    layer = H.make_layer(p)
    x = layer.to_dev(p.x)
    layer.step(x, x)
    torch.cuda.synchronize()
    g = layer.routing_numpy()
    assert g["P"] == 0 and not g["counts"].any()
    for t in (layer.dw_router, layer.dw_gate, layer.dw_up, layer.dw_down, *layer.d_shared):
        assert not t.float().abs().max().item() > 0


def test_long_K_shared_wgrad_tail_split(oracle64):
    """Few, long shared-expert wgrad tiles (K = T = 8192, one 256 x 256 tile per weight matrix): each launch cuts its only
    round into 4 K pieces that wgrad_tail_fixup_kernel adds in a fixed order."""
    w = W.MoEWorkload("tail", T=8192, d=256, E=8, k=2, F=128, n_res=2, n_sh=1, F_sh=256, dtype="bf16", seed=12)
    errs, layer = run_and_compare(H.Problem(w), oracle64)
    print("tail", errs)


def test_routing_is_deterministic(oracle64):
    import torch
    p = H.Problem(W.MoEWorkload("det", T=2048, d=128, E=16, k=2, F=64, n_res=8, dtype="bf16", seed=8))
    layer = H.make_layer(p)
    x, dy = layer.to_dev(p.x), layer.to_dev(p.dy)
    layer.step(x, dy)
    a = {k: v.copy() for k, v in layer.routing_numpy().items() if k != "P"}
    y1, dx1, dw1 = layer.y.clone(), layer.dx.clone(), layer.dw_gate.clone()
    layer.step(x, dy)
    b = layer.routing_numpy()
    for k in a:
        assert np.array_equal(a[k], b[k]), k
    assert torch.equal(y1, layer.y) and torch.equal(dx1, layer.dx) and torch.equal(dw1, layer.dw_gate)


def test_pack_bit_exact(oracle64):
    import torch
    from paper_2606_19025_b200.layer import pack_resident_deltas
    w = W.MoEWorkload("pack", T=1, d=96, E=8, k=2, F=200, n_res=5, seed=9)
    S = W.resident_set(w)
    now = [np.stack(t) for t in zip(*(W.make_expert_master(w, int(e)) for e in S))]
    start = [np.stack(t) for t in zip(*(W.make_round_start_snapshot(w, int(e)) for e in S))]
    want = oracle64.pack(now, start)
    dn = [torch.from_numpy(a).cuda() for a in now]
    ds = [torch.from_numpy(a).cuda() for a in start]
    got = pack_resident_deltas(dn, ds).cpu().numpy()
    assert np.array_equal(got.view(np.uint32), want.view(np.uint32))
    slots = np.array([4, 1, 2], np.int32)
    got2 = pack_resident_deltas(dn, ds, torch.from_numpy(slots).cuda()).cpu().numpy()
    assert np.array_equal(got2.view(np.uint32), oracle64.pack(now, start, slots).view(np.uint32))


def test_bad_arguments_fail_loudly():
    import torch
    from paper_2606_19025_b200 import binding as B
    with pytest.raises(B.FomoeError):
        B.fomoe_workspace_bytes(B.make_config(16, 64, 8, 9, 64), 4)   # k > E
    with pytest.raises(B.FomoeError):
        B.fomoe_workspace_bytes(B.make_config(16, 64, 8, 2, 64), 9)   # n_res > E
    cfg = B.make_config(16, 64, 8, 2, 64, dtype=B.FOMOE_F32)
    rs = B.alloc_route_state(cfg, 4)
    with pytest.raises(B.FomoeError):
        B.fomoe_route(cfg, None, torch.zeros(64, 8, device="cuda"), None, torch.arange(4, dtype=torch.int32, device="cuda"), 4, rs)


@pytest.mark.parametrize("dtype,E", [("f32", 8), ("bf16", 16), ("bf16", 128)])
def test_nan_row_and_minus_inf_bias_stay_contained(oracle64, dtype, E):
    """A diverging step (NaN activations in one token, a -inf router bias on most experts so that fewer than k logits are
    finite) must not fault or corrupt the workspace: ids stay in [0, E), the step completes, and the rows of the other
    tokens are what they are without the NaN token (token rows are independent: Eq. 13)."""
    import torch
    k = 4
    w = W.MoEWorkload("nan", T=300, d=128, E=E, k=k, F=128, n_res=E // 2, dtype=dtype, seed=13)
    p = H.Problem(w)
    bias = np.zeros(E, np.float32)
    bias[2:] = -np.inf                      # two finite logits < k = 4
    p.bias = bias
    layer = H.make_layer(p)
    x_clean = layer.to_dev(p.x)
    dy = layer.to_dev(p.dy)
    layer.step(x_clean, dy)
    torch.cuda.synchronize()
    y_clean, idx_clean = layer.y.clone(), layer.route_state.topk_idx.clone()
    xb = p.x.copy()
    xb[7] = np.nan
    xb[8, 3] = np.inf
    x_bad = layer.to_dev(xb)
    layer.step(x_bad, dy)
    torch.cuda.synchronize()                # an illegal address would surface here
    g = layer.routing_numpy()
    assert g["topk_idx"].min() >= 0 and g["topk_idx"].max() < E
    assert g["counts"].sum() == g["P"] <= w.T * k and (g["pair_row"] < g["P"]).all()
    ok = np.ones(w.T, bool)
    ok[[7, 8]] = False
    okt = torch.from_numpy(ok).cuda()
    assert torch.equal(layer.route_state.topk_idx[okt], idx_clean[okt])
    assert torch.isfinite(layer.y[okt].float()).all()
    assert H.rel_err(H.t2n(layer.y[okt]), H.t2n(y_clean[okt])) <= (2e-2 if dtype == "bf16" else 1e-5)
    # and the layer still works afterwards
    layer.step(x_clean, dy)
    torch.cuda.synchronize()
    assert torch.equal(layer.y, y_clean)


def test_routing_stats_match_definitions(oracle64):
    """fomoe_routing_stats against the numpy definitions, on a Zipf-skewed workload."""
    from oracle import stats_oracle as SO
    w = W.MoEWorkload("stats", T=3000, d=128, E=24, k=3, F=64, n_res=9, dtype="bf16", zipf_alpha=1.0, seed=14)
    p = H.Problem(w)
    H.margin_clean(p, oracle64)
    r = oracle64.route(p.x, p.w_router, p.resident, w.k, w.gate_fn, w.gate_rule, w.temperature, p.bias)
    want = SO.routing_stats(r["topk_idx"], p.resident, w.E)
    layer = H.make_layer(p)
    layer.route(layer.to_dev(p.x))
    got = layer.routing_stats()
    assert np.array_equal(got["load"], want["load"])
    for key in ("kept_fraction", "ghost_fraction", "zero_kept_tokens", "load_cv", "routing_entropy", "max_load", "min_load"):
        assert abs(got[key] - want[key]) <= 1e-5 * max(1.0, abs(want[key])), (key, got[key], want[key])
    assert abs(got["kept_fraction"] - r["P"] / (w.T * w.k)) < 1e-6


def test_debug_validate_resident():
    import torch
    from paper_2606_19025_b200 import binding as B
    ids = lambda *a: torch.tensor(a, dtype=torch.int32, device="cuda")
    B.fomoe_debug_validate_resident(ids(0, 3, 7), 8)
    B.fomoe_debug_validate_resident(ids(), 8)
    for bad, what in ((ids(0, 3, 8), "outside"), (ids(-1, 2), "outside"), (ids(1, 1, 2), "duplicate"), (ids(4, 2), "unsorted")):
        with pytest.raises(B.FomoeError, match=what):
            B.fomoe_debug_validate_resident(bad, 8)


@pytest.mark.parametrize("pipelined", [False, True])
def test_step_host_matches_oracle_twice_in_a_row(oracle64, pipelined):
    """The end-to-end entry point bench.py times (fomoe_moe_step_host: uploads, kernels and downloads on three streams) against
    the oracle, called back to back with different inputs and no synchronisation in between.  pipelined: alternating staging
    buffers and deferred join (the form bench.py times: consecutive steps overlap), four calls, then ONE join + stream sync."""
    import torch
    w = W.MoEWorkload("e2e", T=2048, d=256, E=16, k=2, F=256, n_res=8, n_sh=1, F_sh=128, dtype="bf16", seed=15)
    p = H.Problem(w)
    H.margin_clean(p, oracle64)
    layer = H.make_layer(p)
    cs = torch.cuda.Stream()
    td = layer.tdtype
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(td).pin_memory()
    x1, dy1 = pin(p.x), pin(p.dy)
    x2, dy2 = pin(p.x[::-1].copy()), pin((0.5 * p.dy[::-1]).astype(np.float32))   # token-reversed, scaled: also margin-clean
    outs = [(torch.empty_like(x1).pin_memory(), torch.empty_like(x1).pin_memory()) for _ in range(2)]
    xd, dyd = torch.empty((w.T, w.d), dtype=td, device="cuda"), torch.empty((w.T, w.d), dtype=td, device="cuda")
    if pipelined:
        stage = [(xd, dyd), (torch.empty_like(xd), torch.empty_like(dyd))]
        scratch_out = (torch.empty_like(x1).pin_memory(), torch.empty_like(x1).pin_memory())
        seq = [((x2, dy2), scratch_out), ((x1, dy1), outs[0]), ((x2, dy2), outs[1])]     # first call: results overwritten later
        seq.insert(1, ((x1, dy1), scratch_out))
        for i, ((xh, dyh), (yh, dxh)) in enumerate(seq):
            layer.step_host(xh, dyh, yh, dxh, *stage[i % 2], copy_stream=cs, defer_join=True)
        layer.host_join()
        torch.cuda.current_stream().synchronize()      # the join made the compute stream wait for the downloads
    else:
        for (xh, dyh), (yh, dxh) in zip(((x1, dy1), (x2, dy2)), outs):
            layer.step_host(xh, dyh, yh, dxh, xd, dyd, copy_stream=cs)     # no sync in between: the second call must order itself
        torch.cuda.current_stream().synchronize()      # defer_join = 0: results are complete when the stream is
    for i, ((xh, dyh), (yh, dxh)) in enumerate(zip(((x1, dy1), (x2, dy2)), outs)):
        q = H.Problem(w)
        q.x, q.dy = xh.float().numpy(), dyh.float().numpy()
        r, y, b = H.oracle_all(q, oracle64)
        assert H.rel_err(yh.float().numpy(), y) <= 2e-2, i
        assert H.rel_err(dxh.float().numpy(), b["dx"]) <= 2e-2, i
    # weight gradients left on the device are the second step's
    for key, t in (("dw_router", layer.dw_router), ("dw_gate", layer.dw_gate), ("dw_down", layer.dw_down), ("d_sh_up", layer.d_shared[1])):
        assert H.rel_err(H.t2n(t), b[key]) <= 2e-2, key
