"""fomoe_periln_bwd_noalloc — the Peri-LN backward (Eq. 15) whose partial-sum workspace is a static device array
inside libfomoe.so, for callers that cannot allocate — against the existing fomoe_periln_bwd (caller-owned workspace) on the
same inputs, twice in a row (the array keeps the previous call's contents), and against the oracle within the tolerances of
tests/test_periln_gpu.py.  Named test_zz_* so that pytest collects it last."""
import numpy as np
import pytest

import helpers as H
from oracle import periln_oracle as PO
from paper_2606_19025_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _inputs(dtype, T, d, seed):
    import torch
    rng = np.random.default_rng(seed)
    td = torch.bfloat16 if dtype == "bf16" else torch.float32
    st = (lambda a: W.bf16_round(a)) if dtype == "bf16" else (lambda a: a.astype(np.float32))
    x, res, dout = (st(rng.standard_normal((T, d)) * s + o) for s, o in ((2.0, 0.3), (1.0, 0.0), (1.0, 0.0)))
    gamma, beta = (rng.standard_normal(d) * 0.2 + 1.0).astype(np.float32), (rng.standard_normal(d) * 0.1).astype(np.float32)
    dev = lambda a, dt=td: torch.from_numpy(np.ascontiguousarray(a)).cuda().to(dt)
    return (x, res, dout, gamma, beta), (dev(x), dev(res), dev(dout), dev(gamma, torch.float32), dev(beta, torch.float32))


@pytest.mark.parametrize("dtype", ["bf16", "f32"])
def test_noalloc_matches_the_workspace_path_twice_in_a_row(dtype):
    """Two different problems back to back: the second call finds the first call's partial sums in the array (more CTAs and a
    wider row first, so stale entries lie beyond and between what the second call writes) and must not see them."""
    import torch
    from paper_2606_19025_b200 import binding as B
    tol = 2e-2 if dtype == "bf16" else 1e-4
    alpha = 0.6
    for T, d, seed in ((1500, 1024, 1), (333, 512, 2)):
        (x, res, dout, gamma, beta), (xd, rd, dd, gd, bd) = _inputs(dtype, T, d, seed)
        out, stats = torch.empty_like(xd), torch.empty((T, 2), dtype=torch.float32, device="cuda")
        B.fomoe_periln_fwd(xd, gd, bd, out, stats, residual=rd, alpha=alpha)
        # existing path: caller-owned workspace
        dx0, dg0, db0 = torch.empty_like(xd), torch.empty(d, device="cuda"), torch.empty(d, device="cuda")
        part = torch.empty(B.fomoe_periln_workspace_bytes(T, d), dtype=torch.uint8, device="cuda")
        B.fomoe_periln_bwd(dd, xd, stats, gd, dx0, dg0, db0, part, dresidual=rd, alpha=alpha)
        # new path: no workspace argument; outputs pre-filled with garbage
        dx1 = torch.full_like(xd, float("nan"))
        dg1, db1 = torch.full((d,), float("nan"), device="cuda"), torch.full((d,), float("nan"), device="cuda")
        B.fomoe_periln_bwd_noalloc(dd, xd, stats, gd, dx1, dg1, db1, dresidual=rd, alpha=alpha)
        torch.cuda.synchronize()
        # same kernels, same grid, same fixed-order reduction: identical bits, which is within any tolerance
        assert torch.equal(dx1, dx0) and torch.equal(dg1, dg0) and torch.equal(db1, db0)
        # and the oracle, at the tolerances of test_periln_gpu.py
        _, mean, rstd = PO.periln_post_fwd(res, x, gamma, beta, alpha)
        dxr, dgr, dbr = PO.ln_bwd(alpha * dout, x, mean, rstd, gamma)
        assert H.rel_err(H.t2n(dx1), dxr + res) <= tol
        assert H.rel_err(H.t2n(dg1), dgr) <= 1e-4 and H.rel_err(H.t2n(db1), dbr) <= 1e-4


def test_noalloc_rejects_sizes_beyond_the_static_array():
    import torch
    from paper_2606_19025_b200 import binding as B
    cap = B.fomoe_periln_bwd_noalloc_max_floats()
    assert cap == 4 << 20
    T, d = 4096, 8192          # 2 * min(T, 4 * SMs) * d floats > 4 Mi on any GPU with >= 65 SMs
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    assert 2 * min(T, 4 * sms) * d > cap
    xd = torch.zeros((T, d), dtype=torch.bfloat16, device="cuda")
    stats = torch.zeros((T, 2), dtype=torch.float32, device="cuda")
    g = torch.ones(d, device="cuda")
    dx, dg, db = torch.empty_like(xd), torch.empty(d, device="cuda"), torch.empty(d, device="cuda")
    with pytest.raises(B.FomoeError, match="FOMOE_ERR_UNSUPPORTED.*static array"):
        B.fomoe_periln_bwd_noalloc(xd, xd, stats, g, dx, dg, db)
    # the empty batch is fine and zeroes the parameter gradients, like fomoe_periln_bwd
    e = torch.zeros((0, 64), dtype=torch.bfloat16, device="cuda")
    dg, db = torch.full((64,), 7.0, device="cuda"), torch.full((64,), 7.0, device="cuda")
    B.fomoe_periln_bwd_noalloc(e, e, torch.zeros((0, 2), device="cuda"), torch.ones(64, device="cuda"), e.clone(), dg, db)
    torch.cuda.synchronize()
    assert float(dg.abs().max()) == 0.0 and float(db.abs().max()) == 0.0
