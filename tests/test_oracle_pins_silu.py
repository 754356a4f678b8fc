"""Pins for the oracle's paper-form expert, E(x) = W_down silu(W_up x) (§B.3.1; payload = up + down,
PAPER.md:253), against things other than the oracle (-m "not gpu"): brute force over all experts x indicator, torch
autograd of the independent dense "W_down := 0 outside S" construction (fwd and bwd), central finite differences,
the E=1 closed form sigma(w.x) W_down silu(W_up x), independence from W_gate, the sampled-row helper, and the pack
layout without a gate block."""
import numpy as np
import pytest

import refs
from refs import EXPERT_SILU, GATE_SIGMOID, GATE_SOFTMAX, RULE_DROP_ONLY, RULE_RENORM_RESIDENT, RULE_RENORM_TOPK


def run_silu(o, prob, gate_fn=GATE_SIGMOID, rule=RULE_DROP_ONLY, tau=1.0, bwd=True):
    _, wu, wd = refs.resident_stacks(prob)
    shared = None if prob["shared"] is None else (None, prob["shared"][1], prob["shared"][2])
    r = o.route(prob["x"], prob["w_r"], prob["resident"], prob["k"], gate_fn, rule, tau)
    y = o.moe_fwd(prob["x"], r, prob["resident"], None, wu, wd, shared, expert_fn=EXPERT_SILU)
    b = None
    if bwd:
        b = o.moe_bwd(prob["x"], prob["dy"], prob["w_r"], r, prob["resident"], None, wu, wd, shared, gate_fn, rule, tau,
                      expert_fn=EXPERT_SILU)
    return r, y, b


@pytest.mark.parametrize("seed", range(3))
@pytest.mark.parametrize("gate_fn", [GATE_SOFTMAX, GATE_SIGMOID])
@pytest.mark.parametrize("rule", [RULE_DROP_ONLY, RULE_RENORM_TOPK, RULE_RENORM_RESIDENT])
def test_silu_forward_vs_brute_force(oracle64, seed, gate_fn, rule):
    prob = refs.tiny_problem(40 + seed, T=7, d=6, E=5, k=2, F=4, n_res=[2, 5, 3][seed], n_sh=[0, 1, 2][seed], F_sh=3)
    _, y, _ = run_silu(oracle64, prob, gate_fn, rule, bwd=False)
    np.testing.assert_allclose(y, refs.brute_force_fwd(prob, gate_fn, rule, expert_fn=EXPERT_SILU), rtol=1e-11, atol=1e-13)


@pytest.mark.parametrize("seed", range(3))
@pytest.mark.parametrize("gate_fn", [GATE_SOFTMAX, GATE_SIGMOID])
def test_silu_fwd_bwd_vs_torch_autograd(oracle64, seed, gate_fn):
    """Zeroed-down-projection identity with the paper's expert: forward and every gradient."""
    prob = refs.tiny_problem(50 + seed, T=29, d=11, E=8, k=[2, 4, 3][seed], F=9, n_res=[3, 8, 5][seed], n_sh=[0, 2, 1][seed], F_sh=6)
    _, y, b = run_silu(oracle64, prob, gate_fn)
    y_ref, g = refs.torch_dense_moe(prob, gate_fn, expert_fn=EXPERT_SILU)
    np.testing.assert_allclose(y, y_ref, rtol=1e-11, atol=1e-12)
    assert g["ghost_grad_max"] == 0.0 and "dw_gate" not in b
    for key in ("dx", "dw_router", "dw_up", "dw_down", "d_sh_up", "d_sh_down"):
        if key in g:
            np.testing.assert_allclose(b[key], g[key], rtol=1e-9, atol=1e-11, err_msg=key)


def test_silu_finite_differences(oracle64):
    prob = refs.tiny_problem(78, T=4, d=4, E=4, k=2, F=3, n_res=2, n_sh=1, F_sh=2)
    _, wu, wd = refs.resident_stacks(prob)
    shared = (None, prob["shared"][1], prob["shared"][2])
    _, _, b = run_silu(oracle64, prob)

    def loss(x=None, w_r=None, wu_=None, wd_=None):
        x = prob["x"] if x is None else x
        w_r = prob["w_r"] if w_r is None else w_r
        r = oracle64.route(x, w_r, prob["resident"], prob["k"], GATE_SIGMOID, RULE_DROP_ONLY)
        y = oracle64.moe_fwd(x, r, prob["resident"], None, wu if wu_ is None else wu_, wd if wd_ is None else wd_, shared,
                             expert_fn=EXPERT_SILU)
        return float((y * prob["dy"]).sum())

    eps = 1e-6
    rng = np.random.default_rng(1)
    for name, base, grad, kw in (("dx", prob["x"], b["dx"], "x"), ("dw_router", prob["w_r"], b["dw_router"], "w_r"),
                                 ("dw_up", wu, b["dw_up"], "wu_"), ("dw_down", wd, b["dw_down"], "wd_")):
        for _ in range(6):
            pos = tuple(rng.integers(0, s) for s in base.shape)
            hi, lo = base.copy(), base.copy()
            hi[pos] += eps
            lo[pos] -= eps
            fd = (loss(**{kw: hi}) - loss(**{kw: lo})) / (2 * eps)
            assert abs(fd - grad[pos]) <= 1e-6 * max(1.0, abs(fd)), (name, pos, fd, grad[pos])


def test_silu_single_expert_closed_form(oracle64):
    """E=1, k=1: y = sigmoid(w.x) * W_down silu(W_up x)   (Eq. 13 with one term, Eq. 17, §B.3.1)."""
    prob = refs.tiny_problem(4, T=9, d=6, E=1, k=1, F=5, n_res=1)
    _, y, _ = run_silu(oracle64, prob, bwd=False)
    f = prob["full"]
    v = prob["x"] @ f["w_up"][0].T
    want = (1 / (1 + np.exp(-(prob["x"] @ prob["w_r"])))) * ((v / (1 + np.exp(-v))) @ f["w_down"][0].T)
    np.testing.assert_allclose(y, want, rtol=1e-12)


def test_silu_does_not_read_w_gate(oracle64):
    """The paper's expert has two matrices: whatever is passed as W_gate must not matter."""
    prob = refs.tiny_problem(5, T=12, d=6, E=4, k=2, F=5, n_res=3)
    wg, wu, wd = refs.resident_stacks(prob)
    r = oracle64.route(prob["x"], prob["w_r"], prob["resident"], prob["k"], GATE_SIGMOID)
    y0 = oracle64.moe_fwd(prob["x"], r, prob["resident"], None, wu, wd, expert_fn=EXPERT_SILU)
    y1 = oracle64.moe_fwd(prob["x"], r, prob["resident"], 7.0 * wg, wu, wd, expert_fn=EXPERT_SILU)
    assert np.array_equal(y0, y1)


def test_silu_dw_sample_matches_full_backward(oracle64):
    prob = refs.tiny_problem(22, T=80, d=10, E=6, k=2, F=9, n_res=3)
    _, wu, wd = refs.resident_stacks(prob)
    r, _, b = run_silu(oracle64, prob)
    f_idx = np.array([1, 4, 8], np.int32)
    for slot in range(3):
        g, u, dn = oracle64.dw_sample(prob["x"], prob["dy"], r, prob["resident"], slot, f_idx, None, wu[slot], wd[slot],
                                      expert_fn=EXPERT_SILU)
        assert not g.any()
        np.testing.assert_allclose(u, b["dw_up"][slot][f_idx], rtol=1e-11, atol=1e-13)
        np.testing.assert_allclose(dn, b["dw_down"][slot][:, f_idx].T, rtol=1e-11, atol=1e-13)


def test_silu_pack_payload_is_up_then_down(oracle64):
    """Payload per expert = up + down projections: a gate block of zero elements."""
    rng = np.random.default_rng(3)
    now = [np.zeros((3, 0), np.float32), rng.standard_normal((3, 8)).astype(np.float32), rng.standard_normal((3, 8)).astype(np.float32)]
    start = [np.zeros((3, 0), np.float32), rng.standard_normal((3, 8)).astype(np.float32), rng.standard_normal((3, 8)).astype(np.float32)]
    pay = oracle64.pack(now, start)
    assert pay.shape == (3, 16)
    assert np.array_equal(pay[:, :8], start[1] - now[1]) and np.array_equal(pay[:, 8:], start[2] - now[2])


# ----------------------------------------------------------------------------------------------------
# forced-local routing (the paper's default mode): the partitioned router IS a standard
# top-k MoE over the resident experts with the router sliced to their columns
# ----------------------------------------------------------------------------------------------------
def _sliced(prob, k):
    S = prob["resident"]
    full = {key: v[S].copy() for key, v in prob["full"].items()}
    return dict(x=prob["x"], w_r=prob["w_r"][:, S].copy(), resident=np.arange(len(S), dtype=np.int32), full=full,
                shared=prob["shared"], dy=prob["dy"], k=k, E=len(S))


@pytest.mark.parametrize("seed", range(3))
@pytest.mark.parametrize("gate_fn", [GATE_SOFTMAX, GATE_SIGMOID])
@pytest.mark.parametrize("expert_fn", [0, EXPERT_SILU])
def test_forced_local_is_standard_moe_on_resident_slice(oracle64, seed, gate_fn, expert_fn):
    prob = refs.tiny_problem(60 + seed, T=31, d=9, E=8, k=2, F=6, n_res=[3, 5, 8][seed], n_sh=[0, 1, 0][seed], F_sh=4)
    S, k = prob["resident"], prob["k"]
    wg, wu, wd = refs.resident_stacks(prob)
    shared = prob["shared"]
    if expert_fn == EXPERT_SILU:
        wg = None
        shared = None if shared is None else (None, shared[1], shared[2])
    r = oracle64.route(prob["x"], prob["w_r"], S, k, gate_fn, RULE_DROP_ONLY, 1.0, None, route_mode=1)
    # every selected expert is resident, ghosts have probability 0 and logit -inf
    assert np.isin(r["topk_idx"], S).all() and (r["pair_row"] >= 0).all() and r["P"] == 31 * k
    ghost = np.setdiff1d(np.arange(8), S)
    assert np.all(r["probs"][:, ghost] == 0) and np.all(np.isneginf(r["logits"][:, ghost]))
    y = oracle64.moe_fwd(prob["x"], r, S, wg, wu, wd, shared, expert_fn=expert_fn)
    b = oracle64.moe_bwd(prob["x"], prob["dy"], prob["w_r"], r, S, wg, wu, wd, shared, gate_fn, RULE_DROP_ONLY, 1.0, expert_fn=expert_fn)
    # independent construction: torch autograd of the dense standard MoE over the resident slice
    y_ref, g = refs.torch_dense_moe(_sliced(prob, k), gate_fn, expert_fn=expert_fn)
    np.testing.assert_allclose(y, y_ref, rtol=1e-11, atol=1e-12)
    np.testing.assert_allclose(b["dx"], g["dx"], rtol=1e-9, atol=1e-11)
    np.testing.assert_allclose(b["dw_router"][:, S], g["dw_router"], rtol=1e-9, atol=1e-11)
    assert np.all(b["dw_router"][:, ghost] == 0)      # no router column, no gradient
    for key in ("dw_up", "dw_down") + (() if expert_fn == EXPERT_SILU else ("dw_gate",)):
        np.testing.assert_allclose(b[key], g[key], rtol=1e-9, atol=1e-11, err_msg=key)
    # and brute force over the slice
    np.testing.assert_allclose(y, refs.brute_force_fwd(_sliced(prob, k), gate_fn, expert_fn=expert_fn), rtol=1e-11, atol=1e-13)


def test_forced_local_all_resident_equals_skip_token(oracle64):
    prob = refs.tiny_problem(70, T=20, d=7, E=6, k=3, F=5, n_res=6)
    a = oracle64.route(prob["x"], prob["w_r"], prob["resident"], 3, GATE_SIGMOID, route_mode=0)
    b = oracle64.route(prob["x"], prob["w_r"], prob["resident"], 3, GATE_SIGMOID, route_mode=1)
    for key in ("topk_idx", "gate", "probs", "counts", "offsets", "row_token", "pair_row"):
        assert np.array_equal(a[key], b[key]), key


def test_forced_local_rejects_k_above_resident_count(oracle64):
    prob = refs.tiny_problem(71, T=5, d=4, E=6, k=3, F=3, n_res=2)
    with pytest.raises(ValueError):
        oracle64.route(prob["x"], prob["w_r"], prob["resident"], 3, GATE_SIGMOID, route_mode=1)
