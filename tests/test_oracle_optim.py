"""Pins for oracle/optim_oracle.py (-m "not gpu"): torch.optim.AdamW and torch.optim.SGD(nesterov=True) as independent
library routines, closed forms of the first step, and the pack / unpack round trip."""
import numpy as np
import torch

from oracle import optim_oracle as OO


def test_adamw_matches_torch_over_several_steps():
    rng = np.random.default_rng(0)
    w0 = rng.standard_normal(257)
    p = torch.nn.Parameter(torch.tensor(w0, dtype=torch.float64))
    opt = torch.optim.AdamW([p], lr=0.0131, betas=(0.9, 0.95), eps=1e-8, weight_decay=0.0)
    w, m, v = w0.copy(), np.zeros_like(w0), np.zeros_like(w0)
    for step in range(1, 6):
        g = rng.standard_normal(257)
        p.grad = torch.tensor(g, dtype=torch.float64)
        opt.step()
        w, m, v = OO.adamw_step(w, g, m, v, step, 0.0131)
        np.testing.assert_allclose(w, p.detach().numpy(), rtol=1e-12, atol=1e-14)


def test_adamw_weight_decay_matches_torch():
    rng = np.random.default_rng(1)
    w0, g = rng.standard_normal(64), rng.standard_normal(64)
    p = torch.nn.Parameter(torch.tensor(w0, dtype=torch.float64))
    opt = torch.optim.AdamW([p], lr=0.01, betas=(0.9, 0.95), eps=1e-8, weight_decay=0.1)
    p.grad = torch.tensor(g, dtype=torch.float64)
    opt.step()
    w, _, _ = OO.adamw_step(w0, g, np.zeros(64), np.zeros(64), 1, 0.01, weight_decay=0.1)
    np.testing.assert_allclose(w, p.detach().numpy(), rtol=1e-12)


def test_adamw_first_step_closed_form():
    """Step 1 from zero moments: m_hat = g, v_hat = g^2, so w moves by -lr * g / (|g| + eps) = -lr * sign(g) (eps -> 0)."""
    g = np.array([0.3, -2.0, 1e-3])
    w, m, v = OO.adamw_step(np.zeros(3), g, np.zeros(3), np.zeros(3), 1, 0.5, eps=0.0)
    np.testing.assert_allclose(w, -0.5 * np.sign(g), rtol=1e-12)
    np.testing.assert_allclose(m, 0.1 * g)
    np.testing.assert_allclose(v, 0.05 * g * g)


def test_outer_nesterov_matches_torch_sgd():
    """DiLoCo's outer optimizer: SGD(lr 0.7, momentum 0.9, nesterov) on the outer gradient delta."""
    rng = np.random.default_rng(2)
    w0 = rng.standard_normal(100)
    p = torch.nn.Parameter(torch.tensor(w0, dtype=torch.float64))
    opt = torch.optim.SGD([p], lr=0.7, momentum=0.9, nesterov=True)
    w, buf = w0.copy(), np.zeros_like(w0)
    for _ in range(4):
        delta = rng.standard_normal(100) * 0.01
        p.grad = torch.tensor(delta, dtype=torch.float64)
        opt.step()
        w, buf = OO.outer_nesterov_step(w, delta, buf)
        np.testing.assert_allclose(w, p.detach().numpy(), rtol=1e-12, atol=1e-14)


def test_outer_first_step_closed_form():
    w, buf = OO.outer_nesterov_step(np.ones(3), np.full(3, 0.1), np.zeros(3), lr=0.7, momentum=0.9)
    np.testing.assert_allclose(buf, 0.1)
    np.testing.assert_allclose(w, 1.0 - 0.7 * 0.1 * 1.9)


def test_unpack_inverts_pack(oracle64):
    rng = np.random.default_rng(3)
    now = [rng.standard_normal((5, n)).astype(np.float32) for n in (8, 8, 12)]
    start = [rng.standard_normal((5, n)).astype(np.float32) for n in (8, 8, 12)]
    slots = np.array([4, 1, 2], np.int32)
    pay = oracle64.pack(now, start, slots)
    outs, mask = OO.unpack_blocks(pay, (8, 8, 12), slots, 5)
    assert mask.tolist() == [False, True, True, False, True]
    for i in range(3):
        assert np.array_equal(outs[i][slots], (start[i] - now[i])[slots]) and not outs[i][~mask].any()
