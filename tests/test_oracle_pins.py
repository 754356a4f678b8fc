"""Pins for the CPU oracle (oracle/fomoe_oracle.c) against things other than itself (-m "not gpu").

Each test names what it pins and the passage / mathematics that fixes the expected value:
golden closed forms, brute force on tiny inputs, torch autograd of an independent dense construction,
central finite differences, textbook special cases and structural invariants (SURVEY.md §8(c) pin table).
"""
import itertools
import json
from pathlib import Path

import numpy as np
import pytest

import refs
from refs import GATE_SIGMOID, GATE_SOFTMAX, RULE_DROP_ONLY, RULE_RENORM_RESIDENT, RULE_RENORM_TOPK

GOLDEN = json.loads((Path(__file__).parent / "golden" / "tiny_moe.json").read_text())


def run_oracle(o, prob, gate_fn=GATE_SOFTMAX, gate_rule=RULE_DROP_ONLY, tau=1.0, bias=None, bwd=True):
    wg, wu, wd = refs.resident_stacks(prob)
    r = o.route(prob["x"], prob["w_r"], prob["resident"], prob["k"], gate_fn, gate_rule, tau, bias)
    y = o.moe_fwd(prob["x"], r, prob["resident"], wg, wu, wd, prob["shared"])
    b = None
    if bwd:
        b = o.moe_bwd(prob["x"], prob["dy"], prob["w_r"], r, prob["resident"], wg, wu, wd, prob["shared"], gate_fn, gate_rule, tau)
    return r, y, b


# ----------------------------------------------------------------------------------------------------
# hand-derived worked example (closed forms of PAPER.md Eq. 13/14/17 + skip rule)
# ----------------------------------------------------------------------------------------------------
def _golden_prob():
    i = GOLDEN["inputs"]
    return dict(x=np.array(i["x"]), dy=np.array(i["dy"]), w_r=np.array(i["w_router"]), resident=np.array(i["resident"], np.int32),
                k=i["k"], E=3, shared=None,
                full=None, wg=np.array(i["w_gate"]), wu=np.array(i["w_up"]), wd=np.array(i["w_down"]))


@pytest.mark.parametrize("gate_fn,rule,key", [
    (GATE_SOFTMAX, RULE_DROP_ONLY, "softmax_drop"), (GATE_SIGMOID, RULE_DROP_ONLY, "sigmoid_drop"),
    (GATE_SOFTMAX, RULE_RENORM_TOPK, "softmax_renorm_topk"), (GATE_SOFTMAX, RULE_RENORM_RESIDENT, "softmax_renorm_resident")])
def test_golden_forward(oracle64, gate_fn, rule, key):
    p, e = _golden_prob(), GOLDEN["expected"]
    r = oracle64.route(p["x"], p["w_r"], p["resident"], p["k"], gate_fn, rule)
    assert r["topk_idx"].tolist() == e["topk_idx"]
    assert r["pair_row"].tolist() == e["pair_row"]
    assert r["counts"].tolist() == e["counts"] and r["offsets"].tolist() == e["offsets"]
    assert r["row_token"][: r["P"]].tolist() == e["row_token"]
    np.testing.assert_allclose(r["probs"], e["probs_sigmoid" if gate_fn == GATE_SIGMOID else "probs_softmax"], rtol=1e-14)
    np.testing.assert_allclose(r["gate"], e["gate_" + key], rtol=1e-14)
    y = oracle64.moe_fwd(p["x"], r, p["resident"], p["wg"], p["wu"], p["wd"])
    np.testing.assert_allclose(y, e["y_" + key], rtol=1e-13)


def test_golden_backward(oracle64):
    p, e = _golden_prob(), GOLDEN["expected"]["bwd_softmax_drop"]
    r = oracle64.route(p["x"], p["w_r"], p["resident"], p["k"])
    b = oracle64.moe_bwd(p["x"], p["dy"], p["w_r"], r, p["resident"], p["wg"], p["wu"], p["wd"])
    for key, want in e.items():
        np.testing.assert_allclose(b[key], np.array(want), rtol=1e-12, atol=1e-15, err_msg=key)


# ----------------------------------------------------------------------------------------------------
# brute force: all experts evaluated, times an indicator (tiny inputs)
# ----------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("seed", range(4))
@pytest.mark.parametrize("gate_fn", [GATE_SOFTMAX, GATE_SIGMOID])
@pytest.mark.parametrize("rule", [RULE_DROP_ONLY, RULE_RENORM_TOPK, RULE_RENORM_RESIDENT])
def test_forward_vs_brute_force(oracle64, seed, gate_fn, rule):
    prob = refs.tiny_problem(seed, T=7, d=5, E=5, k=3, F=4, n_res=[2, 3, 5, 0][seed], n_sh=seed % 2, F_sh=3)
    bias = np.linspace(-0.3, 0.3, 5) if seed == 1 else None
    tau = 1.0 if seed != 2 else 0.7
    _, y, _ = run_oracle(oracle64, prob, gate_fn, rule, tau, bias, bwd=False)
    np.testing.assert_allclose(y, refs.brute_force_fwd(prob, gate_fn, rule, tau, bias), rtol=1e-12, atol=1e-13)


# ----------------------------------------------------------------------------------------------------
# zeroed-down-projection identity + autograd: skip-token with set S == standard top-k MoE over all E with
# W_down := 0 outside S, forward AND backward; RENORM rules: autograd of their definition.
# ----------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("seed", range(3))
@pytest.mark.parametrize("gate_fn", [GATE_SOFTMAX, GATE_SIGMOID])
@pytest.mark.parametrize("rule", [RULE_DROP_ONLY, RULE_RENORM_TOPK, RULE_RENORM_RESIDENT])
def test_fwd_bwd_vs_torch_autograd(oracle64, seed, gate_fn, rule):
    prob = refs.tiny_problem(10 + seed, T=33, d=12, E=8, k=3, F=10, n_res=[3, 8, 5][seed], n_sh=[0, 2, 1][seed], F_sh=7)
    tau = [1.0, 1.0, 1.3][seed]
    _, y, b = run_oracle(oracle64, prob, gate_fn, rule, tau)
    y_ref, g = refs.torch_dense_moe(prob, gate_fn, rule, tau)
    np.testing.assert_allclose(y, y_ref, rtol=1e-11, atol=1e-12)
    assert g["ghost_grad_max"] == 0.0  # "missing experts are ignored by the local computational graph"
    for key in ("dx", "dw_router", "dw_gate", "dw_up", "dw_down", "d_sh_gate", "d_sh_up", "d_sh_down"):
        if key in g:
            np.testing.assert_allclose(b[key], g[key], rtol=1e-9, atol=1e-11, err_msg=key)


# ----------------------------------------------------------------------------------------------------
# central finite differences on L = sum(dy*y), f64 build, margins >> step
# ----------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("gate_fn,rule", list(itertools.product([GATE_SOFTMAX, GATE_SIGMOID],
                                                                 [RULE_DROP_ONLY, RULE_RENORM_TOPK, RULE_RENORM_RESIDENT])))
def test_finite_differences(oracle64, gate_fn, rule):
    prob = refs.tiny_problem(77, T=4, d=4, E=4, k=2, F=3, n_res=2, n_sh=1, F_sh=2)
    wg, wu, wd = refs.resident_stacks(prob)
    _, _, b = run_oracle(oracle64, prob, gate_fn, rule)

    def loss(x=None, w_r=None, wg_=None, wd_=None):
        x = prob["x"] if x is None else x
        w_r = prob["w_r"] if w_r is None else w_r
        r = oracle64.route(x, w_r, prob["resident"], prob["k"], gate_fn, rule)
        y = oracle64.moe_fwd(x, r, prob["resident"], wg if wg_ is None else wg_, wu, wd if wd_ is None else wd_, prob["shared"])
        return float((y * prob["dy"]).sum())

    eps = 1e-6
    rng = np.random.default_rng(0)
    for name, base, grad, kw in (("dx", prob["x"], b["dx"], "x"), ("dw_router", prob["w_r"], b["dw_router"], "w_r"),
                                 ("dw_gate", wg, b["dw_gate"], "wg_"), ("dw_down", wd, b["dw_down"], "wd_")):
        for _ in range(6):
            pos = tuple(rng.integers(0, s) for s in base.shape)
            hi, lo = base.copy(), base.copy()
            hi[pos] += eps
            lo[pos] -= eps
            fd = (loss(**{kw: hi}) - loss(**{kw: lo})) / (2 * eps)
            assert abs(fd - grad[pos]) <= 1e-6 * max(1.0, abs(fd)), (name, pos, fd, grad[pos])


# ----------------------------------------------------------------------------------------------------
# textbook special cases
# ----------------------------------------------------------------------------------------------------
def _ffn(x, wg, wu, wd):
    a, u = x @ wg.T, x @ wu.T
    return (a / (1 + np.exp(-a)) * u) @ wd.T


def test_single_expert_sigmoid_closed_form(oracle64):
    """E=1, k=1, sigmoid: y = sigmoid(w.x) * FFN(x) (Eq. 13 with one term)."""
    prob = refs.tiny_problem(3, T=9, d=6, E=1, k=1, F=5, n_res=1)
    _, y, _ = run_oracle(oracle64, prob, GATE_SIGMOID, bwd=False)
    f = prob["full"]
    want = (1 / (1 + np.exp(-(prob["x"] @ prob["w_r"])))) * _ffn(prob["x"], f["w_gate"][0], f["w_up"][0], f["w_down"][0])
    np.testing.assert_allclose(y, want, rtol=1e-12)


def test_k_equals_E_is_dense_softmax_mixture(oracle64):
    """k=E, all resident, softmax: y = sum_e softmax(z)_e FFN_e(x)."""
    prob = refs.tiny_problem(4, T=8, d=6, E=4, k=4, F=5, n_res=4)
    _, y, _ = run_oracle(oracle64, prob, GATE_SOFTMAX, bwd=False)
    z = prob["x"] @ prob["w_r"]
    p = np.exp(z - z.max(1, keepdims=True))
    p /= p.sum(1, keepdims=True)
    f = prob["full"]
    want = sum(p[:, [e]] * _ffn(prob["x"], f["w_gate"][e], f["w_up"][e], f["w_down"][e]) for e in range(4))
    np.testing.assert_allclose(y, want, rtol=1e-12)


def test_no_resident_expert_gives_shared_only_or_zero(oracle64):
    prob = refs.tiny_problem(5, T=6, d=5, E=4, k=2, F=3, n_res=0, n_sh=2, F_sh=4)
    r, y, b = run_oracle(oracle64, prob)
    sg, su, sd = prob["shared"]
    # shared experts == one dense FFN with concatenated hidden dimension
    want = _ffn(prob["x"], sg.reshape(-1, 5), su.reshape(-1, 5), np.concatenate(list(sd), axis=1))
    np.testing.assert_allclose(y, want, rtol=1e-12)
    assert r["P"] == 0 and np.all(r["gate"] == 0) and np.all(r["pair_row"] == -1)
    assert np.all(b["dw_router"] == 0)
    prob["shared"] = None
    _, y0, b0 = run_oracle(oracle64, prob)
    assert np.all(y0 == 0) and np.all(b0["dx"] == 0)


def test_shared_part_is_additive(oracle64):
    """Shared experts sit outside the router with gate 1: the layer is (routed part) + (shared part), so
    y, dx and the gradients split exactly.  tests/test_parity_fullsize_gpu.py uses this to pay for the shared FFN of the
    C4 sweep once; the routed-only and shared-only runs are pinned by the brute force / closed form above."""
    prob = refs.tiny_problem(15, T=9, d=6, E=5, k=2, F=4, n_res=3, n_sh=2, F_sh=3)
    r, y, b = run_oracle(oracle64, prob)
    routed = dict(prob, shared=None)
    _, y_r, b_r = run_oracle(oracle64, routed)
    only = dict(prob, resident=np.zeros(0, np.int32))
    wg, wu, wd = refs.resident_stacks(prob)
    r0 = oracle64.route(prob["x"], prob["w_r"], only["resident"], prob["k"])
    y_s = oracle64.moe_fwd(prob["x"], r0, only["resident"], wg[:0], wu[:0], wd[:0], prob["shared"])
    b_s = oracle64.moe_bwd(prob["x"], prob["dy"], prob["w_r"], r0, only["resident"], wg[:0], wu[:0], wd[:0], prob["shared"])
    np.testing.assert_allclose(y, y_r + y_s, rtol=1e-12, atol=1e-14)
    np.testing.assert_allclose(b["dx"], b_r["dx"] + b_s["dx"], rtol=1e-12, atol=1e-14)
    for key in ("d_sh_gate", "d_sh_up", "d_sh_down"):
        np.testing.assert_allclose(b[key], b_s[key], rtol=1e-12, atol=1e-14)
    for key in ("dw_router", "dw_gate", "dw_up", "dw_down"):
        np.testing.assert_allclose(b[key], b_r[key], rtol=1e-12, atol=1e-14)
    assert not b_s["dw_router"].any()


def test_all_resident_equals_standard_topk_moe(oracle64):
    """S = [0,E): the 'full overlap' limit is a plain top-k MoE; brute force has no residency term left."""
    prob = refs.tiny_problem(6, T=7, d=5, E=5, k=2, F=4, n_res=5)
    r, y, _ = run_oracle(oracle64, prob, bwd=False)
    assert r["P"] == 7 * 2 and np.all(r["pair_row"] >= 0)
    np.testing.assert_allclose(y, refs.brute_force_fwd(prob), rtol=1e-12, atol=1e-13)


# ----------------------------------------------------------------------------------------------------
# structural invariants of routing / permutation
# ----------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("gate_fn", [GATE_SOFTMAX, GATE_SIGMOID])
def test_routing_invariants(oracle64, gate_fn):
    rng = np.random.default_rng(1)
    T, d, E, k, n_res = 300, 16, 12, 4, 5
    x, w_r = rng.standard_normal((T, d)), rng.standard_normal((d, E))
    S = np.sort(rng.permutation(E)[:n_res]).astype(np.int32)
    r = oracle64.route(x, w_r, S, k, gate_fn)
    z = x @ w_r
    np.testing.assert_allclose(r["logits"], z, rtol=1e-12, atol=1e-13)
    # top-k == first k of a full stable sort by descending logit
    assert np.array_equal(r["topk_idx"], np.argsort(-r["logits"], axis=1, kind="stable")[:, :k])
    if gate_fn == GATE_SOFTMAX:
        np.testing.assert_allclose(r["probs"].sum(1), 1.0, rtol=1e-13)
        r2 = oracle64.route(x, w_r, S, k, gate_fn, bias=np.full(E, 3.0))  # shift invariance
        np.testing.assert_allclose(r2["probs"], r["probs"], rtol=1e-12)
    assert np.all((r["probs"] > 0) & (r["probs"] < 1))
    kept = np.isin(r["topk_idx"], S)
    P = int(kept.sum())
    assert r["P"] == P == r["counts"].sum() == r["offsets"][-1]
    assert np.array_equal(r["offsets"], np.concatenate([[0], np.cumsum(r["counts"])]))
    assert np.array_equal(r["counts"], [(r["topk_idx"] == e).sum() for e in S])
    assert np.all(r["pair_row"][~kept] == -1) and np.all(r["gate"][~kept] == 0)
    assert np.array_equal(np.sort(r["pair_row"][kept]), np.arange(P))          # each kept pair appears once
    tt, jj = np.nonzero(kept)
    assert np.array_equal(r["row_token"][r["pair_row"][tt, jj]], tt)           # mutually inverse
    assert np.all(r["row_token"][P:] == -1)
    np.testing.assert_array_equal(r["gate"][kept], np.take_along_axis(r["probs"], r["topk_idx"], 1)[kept])  # drop-only: unchanged
    for s in range(n_res):   # rows of a slot ascend in (t, j): tokens ascend (a token meets an expert once)
        rows = r["row_token"][r["offsets"][s]: r["offsets"][s + 1]]
        assert np.all(np.diff(rows) > 0)
        assert np.all(r["topk_idx"][rows] == S[s], axis=None) or np.all((r["topk_idx"][rows] == S[s]).any(1))


def test_topk_tie_break_prefers_lower_index(oracle64):
    x = np.ones((1, 2))
    w_r = np.array([[0.5, 1.0, 1.0, 0.5], [0.0, 0.0, 0.0, 0.0]])
    r = oracle64.route(x, w_r, np.arange(4, dtype=np.int32), 3)
    assert r["topk_idx"].tolist() == [[1, 2, 0]]


def test_renorm_resident_gates_sum_to_one(oracle64):
    prob = refs.tiny_problem(8, T=40, d=6, E=6, k=3, F=2, n_res=3)
    r = oracle64.route(prob["x"], prob["w_r"], prob["resident"], 3, GATE_SOFTMAX, RULE_RENORM_RESIDENT)
    has = (r["pair_row"] >= 0).any(1)
    np.testing.assert_allclose(r["gate"].sum(1)[has], 1.0, rtol=1e-13)
    assert np.all(r["gate"].sum(1)[~has] == 0)


def test_zero_rows_and_dz_rowsum(oracle64):
    prob = refs.tiny_problem(9, T=60, d=6, E=8, k=2, F=3, n_res=2)
    for gate_fn in (GATE_SOFTMAX, GATE_SIGMOID):
        r, y, b = run_oracle(oracle64, prob, gate_fn)
        none = (r["pair_row"] < 0).all(1)
        assert none.any() and np.all(y[none] == 0)            # rows with no kept pair are bit-zero
        assert np.all(b["dgate"][r["pair_row"] < 0] == 0)
        if gate_fn == GATE_SOFTMAX:
            np.testing.assert_allclose(b["dlogits"].sum(1), 0, atol=1e-15)
        else:                                                    # sigmoid: exactly zero dz / dx without a kept pair
            assert np.all(b["dlogits"][none] == 0) and np.all(b["dx"][none] == 0)
            assert np.all(b["dlogits"][:, np.setdiff1d(np.arange(8), prob["resident"])] == 0)


def test_token_equivariance(oracle64):
    prob = refs.tiny_problem(11, T=25, d=6, E=6, k=2, F=4, n_res=3, n_sh=1, F_sh=3)
    _, y, b = run_oracle(oracle64, prob)
    perm = np.random.default_rng(0).permutation(25)
    prob2 = dict(prob, x=prob["x"][perm], dy=prob["dy"][perm])
    _, y2, b2 = run_oracle(oracle64, prob2)
    np.testing.assert_allclose(y2, y[perm], rtol=1e-13, atol=1e-15)
    np.testing.assert_allclose(b2["dx"], b["dx"][perm], rtol=1e-13, atol=1e-15)
    for key in ("dw_router", "dw_gate", "dw_up", "dw_down", "d_sh_gate"):
        np.testing.assert_allclose(b2[key], b[key], rtol=1e-10, atol=1e-13)


def test_superset_of_residents_only_adds_terms(oracle64):
    """Making a ghost expert resident changes y only on tokens that selected it (skipped pairs contribute exactly zero)."""
    prob = refs.tiny_problem(12, T=50, d=6, E=6, k=2, F=4, n_res=3)
    r, y, _ = run_oracle(oracle64, prob, bwd=False)
    ghost = int(np.setdiff1d(np.arange(6), prob["resident"])[0])
    prob2 = dict(prob, resident=np.sort(np.append(prob["resident"], ghost)).astype(np.int32))
    _, y2, _ = run_oracle(oracle64, prob2, bwd=False)
    touched = (r["topk_idx"] == ghost).any(1)
    assert touched.any() and np.array_equal(y2[~touched], y[~touched]) and not np.allclose(y2[touched], y[touched])


def test_kept_fraction_matches_eq2(oracle32):
    """sigma_st = N_le/N_e under balanced routing (Eq. 2; 207), uniform C2-like draw."""
    from paper_2606_19025_b200 import workloads as W
    w = W.config("C2").with_(T=4096)
    r = oracle32.route(W.make_x(w), W.make_router(w), W.resident_set(w), w.k)
    assert abs(r["P"] / (w.T * w.k) - w.n_res / w.E) < 0.03


# ----------------------------------------------------------------------------------------------------
# f32 build agrees with f64 build; pack is one IEEE subtraction per word
# ----------------------------------------------------------------------------------------------------
def test_f32_build_matches_f64(oracle32, oracle64):
    prob = refs.tiny_problem(13, T=64, d=16, E=8, k=2, F=12, n_res=4, n_sh=1, F_sh=8, wscale=0.2)
    r64, y64, b64 = run_oracle(oracle64, prob)
    r32, y32, b32 = run_oracle(oracle32, prob)
    assert np.array_equal(r32["topk_idx"], r64["topk_idx"]) and np.array_equal(r32["pair_row"], r64["pair_row"])
    assert np.abs(y32 - y64).max() <= 1e-5 * np.abs(y64).max()
    for key in ("dx", "dw_router", "dw_gate", "dw_up", "dw_down"):
        assert np.abs(b32[key] - b64[key]).max() <= 1e-5 * np.abs(b64[key]).max(), key


def test_dw_sample_matches_full_backward(oracle64):
    """The sampled-row weight-gradient helper used by the full-size GPU tests equals the (autograd-pinned) full backward."""
    prob = refs.tiny_problem(21, T=90, d=10, E=6, k=2, F=9, n_res=3)
    wg, wu, wd = refs.resident_stacks(prob)
    r, _, b = run_oracle(oracle64, prob)
    f_idx = np.array([0, 4, 8], np.int32)
    for slot in range(3):
        g, u, dn = oracle64.dw_sample(prob["x"], prob["dy"], r, prob["resident"], slot, f_idx, wg[slot], wu[slot], wd[slot])
        np.testing.assert_allclose(g, b["dw_gate"][slot][f_idx], rtol=1e-11, atol=1e-13)
        np.testing.assert_allclose(u, b["dw_up"][slot][f_idx], rtol=1e-11, atol=1e-13)
        np.testing.assert_allclose(dn, b["dw_down"][slot][:, f_idx].T, rtol=1e-11, atol=1e-13)


def test_pack_bit_exact_and_layout(oracle64):
    rng = np.random.default_rng(2)
    n_res, F, d = 5, 6, 4
    now = [rng.standard_normal(s).astype(np.float32) for s in ((n_res, F, d), (n_res, F, d), (n_res, d, F))]
    start = [a + rng.standard_normal(a.shape).astype(np.float32) * np.float32(1e-3) for a in now]
    pay = oracle64.pack(now, start)
    assert pay.shape == (n_res, 3 * F * d) and pay.dtype == np.float32
    for s in range(n_res):   # blocks in ascending slot order, tensors gate|up|down at closed-form offsets
        for t in range(3):
            want = (start[t][s] - now[t][s]).ravel()
            assert np.array_equal(pay[s, t * F * d:(t + 1) * F * d].view(np.uint32), want.view(np.uint32))
    slots = np.array([3, 0], np.int32)
    sub = oracle64.pack(now, start, slots)
    assert np.array_equal(sub, pay[slots])
