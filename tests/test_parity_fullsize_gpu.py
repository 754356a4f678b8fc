"""Full-size parity (BASELINE.json configs 2-5, the launch configuration bench.py times).

C2, C3 and every residency of the C4 sweep at their REAL shapes: every output (routing, y, dx, dW_router, dW of every resident
expert, shared-expert gradients) element by element under the dense dy (test_fullsize_dense).  C5 (the oracle would need
minutes) on outputs the oracle can compute one by one (test_fullsize_sampled):
  * routing: every integer output bit-exact against the oracle's full route (margin-cleaned tokens); probs / gates;
  * y and dx on sampled tokens (per-token quantities: the oracle runs on the token subset with the same weights);
  * dW_gate / dW_up rows and dW_down columns of sampled (slot, f) over ALL rows of the slot (oracle_dw_sample);
  * a second backward with dy zero outside the sampled tokens: then EVERY weight gradient (router, experts, shared) equals
    the oracle's backward over the subset and dx is exactly zero elsewhere — whole tensors compared, same launch geometry;
  * properties that hold at any size (counts, zero rows).
"""
import numpy as np
import pytest

import helpers as H
from paper_2606_19025_b200 import workloads as W

pytestmark = pytest.mark.gpu
TOL = 2e-2
N_TOK = 32


def subset_route(oracle64, p, idx):
    w = p.w
    return oracle64.route(p.x[idx], p.w_router, p.resident, w.k, w.gate_fn, w.gate_rule, w.temperature, p.bias)


@pytest.mark.parametrize("name,n_res", [("C5", None)])
def test_fullsize_sampled(oracle64, name, n_res):
    import torch
    w = W.config(name)
    p = H.Problem(w, n_res)
    redrawn = H.margin_clean(p, oracle64)
    r = oracle64.route(p.x, p.w_router, p.resident, w.k, w.gate_fn, w.gate_rule, w.temperature, p.bias)
    layer = H.make_layer(p)
    x, dy = layer.to_dev(p.x), layer.to_dev(p.dy)
    step = layer.capture_step(x, dy)          # the launch configuration bench.py times: one CUDA graph per step
    step()
    torch.cuda.synchronize()

    # ---- routing: everything, bit-exact ----
    g = layer.routing_numpy()
    for key in ("topk_idx", "counts", "offsets", "row_token", "pair_row"):
        assert np.array_equal(g[key], r[key]), key
    assert H.rel_err(g["probs"], r["probs"]) <= 1e-4 and H.rel_err(g["gate"], r["gate"]) <= 1e-4
    kept = np.isin(r["topk_idx"], p.resident)
    assert g["P"] == int(kept.sum()) == int(g["counts"].sum())
    if w.zipf_alpha == 0:   # sigma_st = N_le / N_e under balanced routing (Eq. 2)
        assert abs(g["P"] / (w.T * w.k) - len(p.resident) / w.E) < 0.03
    y = H.t2n(layer.y)
    none = ~kept.any(1)
    if p.shared is None:
        assert none.any() and np.all(y[none] == 0)

    # ---- sampled tokens: y and dx ----
    rng = np.random.default_rng(11)
    with_kept = np.nonzero(kept.any(1))[0]
    n_none = min(4, int(none.sum()))
    idx = np.sort(np.concatenate([rng.choice(with_kept, N_TOK - n_none, replace=False),
                                  rng.choice(np.nonzero(none)[0], n_none, replace=False)])).astype(np.int64)
    rs = subset_route(oracle64, p, idx)
    assert np.array_equal(rs["topk_idx"], r["topk_idx"][idx])
    ys = oracle64.moe_fwd(p.x[idx], rs, p.resident, p.wg, p.wu, p.wd, p.shared)
    bs = oracle64.moe_bwd(p.x[idx], p.dy[idx], p.w_router, rs, p.resident, p.wg, p.wu, p.wd, p.shared, w.gate_fn, w.gate_rule,
                          w.temperature)
    errs = {"y": H.rel_err(y[idx], ys), "dx": H.rel_err(H.t2n(layer.dx)[idx], bs["dx"])}

    # ---- sampled (slot, f): weight gradients over all rows of the slot ----
    n_slots = len(p.resident)
    big = int(np.argmax(r["counts"]))
    small = int(np.argmin(r["counts"]))
    for slot in sorted({0, n_slots - 1, big, small}):
        f_idx = np.sort(rng.choice(w.F, 3, replace=False)).astype(np.int32)
        og, ou, od = oracle64.dw_sample(p.x, p.dy, r, p.resident, slot, f_idx, p.wg[slot], p.wu[slot], p.wd[slot])
        fi = torch.from_numpy(f_idx.astype(np.int64)).cuda()
        errs[f"dw_gate[{slot}]"] = H.rel_err(H.t2n(layer.dw_gate[slot][fi]), og)
        errs[f"dw_up[{slot}]"] = H.rel_err(H.t2n(layer.dw_up[slot][fi]), ou)
        errs[f"dw_down[{slot}]"] = H.rel_err(H.t2n(layer.dw_down[slot][:, fi]).T, od)

    # ---- sparse dy: whole weight-gradient tensors against the subset backward ----
    dy2 = np.zeros_like(p.dy)
    dy2[idx] = p.dy[idx]
    layer.backward(layer.to_dev(dy2), x)
    torch.cuda.synchronize()
    dx2 = H.t2n(layer.dx)
    mask = np.ones(w.T, bool)
    mask[idx] = False
    assert np.all(dx2[mask] == 0)
    errs["sparse dx"] = H.rel_err(dx2[idx], bs["dx"])
    got = dict(dw_router=layer.dw_router, dw_gate=layer.dw_gate, dw_up=layer.dw_up, dw_down=layer.dw_down)
    if p.shared is not None:
        got.update(d_sh_gate=layer.d_shared[0], d_sh_up=layer.d_shared[1], d_sh_down=layer.d_shared[2])
    for key, t in got.items():
        errs["sparse " + key] = H.rel_err(H.t2n(t), bs[key])
    print(name, "redrawn tokens", redrawn, "P", g["P"], "rows/slot min..max", int(r["counts"].min()), int(r["counts"].max()),
          {k: f"{v:.1e}" for k, v in errs.items()})
    bad = {k: v for k, v in errs.items() if not v <= TOL}
    assert not bad, bad


@pytest.mark.parametrize("n_res", W.C4_RESIDENT_SWEEP)
def test_c4_residency_sweep_reduced(oracle64, n_res):
    """BASELINE.json config 4 (residency / skew sweep) at T = 2048, all outputs element by element."""
    import torch
    w = W.config("C4").with_(T=2048, d=512, F=384, F_sh=384)
    p = H.Problem(w, n_res)
    H.margin_clean(p, oracle64)
    r, y, b = H.oracle_all(p, oracle64)
    layer = H.make_layer(p)
    x, dy = layer.to_dev(p.x), layer.to_dev(p.dy)
    layer.step(x, dy)
    torch.cuda.synchronize()
    g = layer.routing_numpy()
    for key in ("topk_idx", "counts", "offsets", "row_token", "pair_row"):
        assert np.array_equal(g[key], r[key]), key
    errs = dict(y=H.rel_err(H.t2n(layer.y), y), dx=H.rel_err(H.t2n(layer.dx), b["dx"]),
                dw_router=H.rel_err(H.t2n(layer.dw_router), b["dw_router"]), dw_gate=H.rel_err(H.t2n(layer.dw_gate), b["dw_gate"]),
                dw_up=H.rel_err(H.t2n(layer.dw_up), b["dw_up"]), dw_down=H.rel_err(H.t2n(layer.dw_down), b["dw_down"]),
                d_sh_gate=H.rel_err(H.t2n(layer.d_shared[0]), b["d_sh_gate"]), d_sh_down=H.rel_err(H.t2n(layer.d_shared[2]), b["d_sh_down"]))
    assert all(v <= TOL for v in errs.values()), errs
    # nested resident sets: the realised kept fraction grows with n_res (use the realised frequency under skew)
    print("C4 reduced n_res", n_res, "kept fraction", g["P"] / (w.T * w.k), "rows/slot", int(r["counts"].min()), int(r["counts"].max()))


# ------------------------------------------------------------------------------------------------------------------
# dense dy, every output, element by element, at the real shapes
# ------------------------------------------------------------------------------------------------------------------
_SHARED_PART = {}


def _shared_only(o, p):
    """Shared-expert part of the layer (applied to every token with gate 1, outside the router), computed once
    per workload: the oracle with NO resident expert.  y, dx and d_sh_* of the full layer are this plus the routed part
    (additivity pinned in tests/test_oracle_pins.py::test_shared_part_is_additive), which lets the C4 sweep pay for the
    16384-token shared FFN once instead of four times."""
    key = (p.w.name, p.w.T, p.w.d, p.w.F_sh, p.w.seed)
    if key not in _SHARED_PART:
        w = p.w
        none = np.zeros(0, np.int32)
        e0 = (np.zeros((0, w.F, w.d), np.float32), np.zeros((0, w.F, w.d), np.float32), np.zeros((0, w.d, w.F), np.float32))
        r0 = o.route(p.x, p.w_router, none, w.k, w.gate_fn, w.gate_rule, w.temperature, p.bias)
        y0 = o.moe_fwd(p.x, r0, none, *e0, p.shared)
        b0 = o.moe_bwd(p.x, p.dy, p.w_router, r0, none, *e0, p.shared, w.gate_fn, w.gate_rule, w.temperature)
        _SHARED_PART[key] = (y0, b0)
    return _SHARED_PART[key]


@pytest.mark.parametrize("name,n_res,real,split_shared", [
    ("C2", None, "f64", False), ("C3", None, "f32", False),
    ("C4", 8, "f32", True), ("C4", 16, "f32", True), ("C4", 32, "f32", True), ("C4", 64, "f32", True)])
def test_fullsize_dense(oracle64, oracle32, name, n_res, real, split_shared):
    """Reference: the f64 oracle where it finishes in well under a minute on the box, else the f32 build of the same source
    (its own rounding, ~1e-6 relative, is far below the 2e-2 bar).  Margin cleaning always uses f64 logits."""
    import time
    import torch
    o = oracle64 if real == "f64" else oracle32
    w = W.config(name)
    p = H.Problem(w, n_res)
    redrawn = H.margin_clean(p, oracle64)
    t0 = time.time()
    r = o.route(p.x, p.w_router, p.resident, w.k, w.gate_fn, w.gate_rule, w.temperature, p.bias)
    sh = None if split_shared else p.shared
    y = o.moe_fwd(p.x, r, p.resident, p.wg, p.wu, p.wd, sh)
    b = o.moe_bwd(p.x, p.dy, p.w_router, r, p.resident, p.wg, p.wu, p.wd, sh, w.gate_fn, w.gate_rule, w.temperature)
    if split_shared:
        y0, b0 = _shared_only(o, p)
        y = y + y0
        b = dict(b)
        b["dx"] = b["dx"] + b0["dx"]
        for key in ("d_sh_gate", "d_sh_up", "d_sh_down"):
            b[key] = b0[key]
    t_oracle = time.time() - t0

    layer = H.make_layer(p)
    x, dy = layer.to_dev(p.x), layer.to_dev(p.dy)
    step = layer.capture_step(x, dy)          # the launch configuration bench.py times: one CUDA graph per step
    step()
    torch.cuda.synchronize()
    g = layer.routing_numpy()
    for key in ("topk_idx", "counts", "offsets", "row_token", "pair_row"):
        assert np.array_equal(g[key], r[key]), key
    assert H.rel_err(g["probs"], r["probs"]) <= 1e-4 and H.rel_err(g["gate"], r["gate"]) <= 1e-4
    errs = {"y": H.rel_err(H.t2n(layer.y), y)}
    got = dict(dx=layer.dx, dw_router=layer.dw_router, dw_gate=layer.dw_gate, dw_up=layer.dw_up, dw_down=layer.dw_down)
    if p.shared is not None:
        got.update(d_sh_gate=layer.d_shared[0], d_sh_up=layer.d_shared[1], d_sh_down=layer.d_shared[2])
    for key, t in got.items():
        errs[key] = H.rel_err(H.t2n(t), b[key])
    # per-slot weight gradients: a dropped K block of a small group would hide under the tensor-wide max|ref|
    for slot in range(len(p.resident)):
        for key, t in (("dw_gate", layer.dw_gate), ("dw_up", layer.dw_up), ("dw_down", layer.dw_down)):
            if r["counts"][slot] > 0:
                errs[f"{key}[{slot}]"] = H.rel_err(H.t2n(t[slot]), b[key][slot])
            else:
                assert not H.t2n(t[slot]).any()
    worst = max(errs.items(), key=lambda kv: kv[1])
    print(name, "n_res", len(p.resident), "redrawn", redrawn, "P", g["P"], "kept", round(g["P"] / (w.T * w.k), 4),
          "rows/slot", int(r["counts"].min()), int(r["counts"].max()), f"oracle({real}) {t_oracle:.0f}s worst", worst)
    bad = {k: v for k, v in errs.items() if not v <= TOL}
    assert not bad, bad
