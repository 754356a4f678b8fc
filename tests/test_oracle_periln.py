"""Pins for oracle/periln_oracle.py (-m "not gpu"): torch.nn.functional.layer_norm and autograd (library routine), closed
forms (zero mean / unit variance, shift and scale invariance), and Eq. 15 assembled end to end."""
import numpy as np
import torch

from oracle import periln_oracle as PO


def _rand(seed, T=7, d=12):
    r = np.random.default_rng(seed)
    return r.standard_normal((T, d)) * 2 + 0.5, r.standard_normal(d) + 1.0, r.standard_normal(d), r.standard_normal((T, d))


def test_ln_forward_matches_torch_and_normalises():
    x, g, b, _ = _rand(0)
    out, mean, rstd = PO.ln_fwd(x, g, b)
    ref = torch.nn.functional.layer_norm(torch.tensor(x), (x.shape[1],), torch.tensor(g), torch.tensor(b), 1e-5).numpy()
    np.testing.assert_allclose(out, ref, rtol=1e-12, atol=1e-13)
    xhat = (out - b) / g
    np.testing.assert_allclose(xhat.mean(1), 0, atol=1e-12)
    np.testing.assert_allclose((xhat ** 2).mean(1), 1, rtol=1e-4)        # up to eps
    np.testing.assert_allclose(PO.ln_fwd(3.0 * x + 7.0, g, b, eps=0.0)[0], PO.ln_fwd(x, g, b, eps=0.0)[0], rtol=1e-10, atol=1e-11)


def test_ln_backward_matches_autograd():
    x, g, b, dout = _rand(1)
    xt, gt, bt = (torch.tensor(a, requires_grad=True) for a in (x, g, b))
    y = torch.nn.functional.layer_norm(xt, (x.shape[1],), gt, bt, 1e-5)
    (y * torch.tensor(dout)).sum().backward()
    _, mean, rstd = PO.ln_fwd(x, g, b)
    dx, dg, db = PO.ln_bwd(dout, x, mean, rstd, g)
    np.testing.assert_allclose(dx, xt.grad.numpy(), rtol=1e-10, atol=1e-12)
    np.testing.assert_allclose(dg, gt.grad.numpy(), rtol=1e-10, atol=1e-12)
    np.testing.assert_allclose(db, bt.grad.numpy(), rtol=1e-10, atol=1e-12)


def test_eq15_block_end_to_end_against_autograd():
    """x_{l+1} = x + alpha LN2(F(LN1(x))) with F a fixed linear map standing in for the MoE block."""
    x, g1, b1, dout = _rand(2)
    _, g2, b2, _ = _rand(3)
    A = np.random.default_rng(4).standard_normal((x.shape[1], x.shape[1])) * 0.3
    alpha = 0.7
    xt, g1t, b1t, g2t, b2t = (torch.tensor(a, requires_grad=True) for a in (x, g1, b1, g2, b2))
    d = (x.shape[1],)
    yt = torch.nn.functional.layer_norm(xt, d, g1t, b1t, 1e-5) @ torch.tensor(A)
    outt = xt + alpha * torch.nn.functional.layer_norm(yt, d, g2t, b2t, 1e-5)
    (outt * torch.tensor(dout)).sum().backward()
    xn, m1, r1 = PO.ln_fwd(x, g1, b1)
    y = xn @ A
    out, m2, r2 = PO.periln_post_fwd(x, y, g2, b2, alpha)
    np.testing.assert_allclose(out, outt.detach().numpy(), rtol=1e-11, atol=1e-12)
    dy, dg2, db2 = PO.periln_post_bwd(dout, y, m2, r2, g2, alpha)
    dxn = dy @ A.T
    dx, dg1, db1 = PO.periln_pre_bwd(dxn, x, m1, r1, g1, dout)
    for got, want in ((dx, xt.grad), (dg1, g1t.grad), (db1, b1t.grad), (dg2, g2t.grad), (db2, b2t.grad)):
        np.testing.assert_allclose(got, want.numpy(), rtol=1e-9, atol=1e-11)
