"""Parity of the round-boundary optimizer kernels (fomoe_adamw_resident, fomoe_outer_nesterov) against oracle/optim_oracle.py
(fp64 numpy) through the C ABI: fp32 arithmetic -> max|err|/max|ref| <= 1e-4 is the bar (measured ~1e-7); the compute-dtype
copy is exactly the rounding of the fp32 result; unpacked slots are untouched."""
import numpy as np
import pytest

import helpers as H
from oracle import optim_oracle as OO

pytestmark = pytest.mark.gpu


def _stacks(rng, n_res, elems, scale=1.0):
    return [None if e == 0 else (rng.standard_normal((n_res, e)) * scale).astype(np.float32) for e in elems]


@pytest.mark.parametrize("elems", [(4096 + 8, 4096 + 8, 1024), (0, 2052, 2052)])
@pytest.mark.parametrize("gdt", ["f32", "bf16"])
def test_adamw_resident(gdt, elems):
    import torch
    from paper_2606_19025_b200 import binding as B
    rng = np.random.default_rng(5)
    n_res = 3
    w = _stacks(rng, n_res, elems, 0.02)
    m = [None if a is None else np.zeros_like(a) for a in w]
    v = [None if a is None else np.zeros_like(a) for a in w]
    dev = lambda a, dt=torch.float32: None if a is None else torch.from_numpy(a).cuda().to(dt)
    wd_, md_, vd_ = [dev(a) for a in w], [dev(a) for a in m], [dev(a) for a in v]
    cdt = torch.bfloat16 if gdt == "bf16" else torch.float32     # `dtype` of the ABI call covers grad and w_compute alike
    wc = [None if a is None else torch.empty(a.shape, dtype=cdt, device="cuda") for a in w]
    ref = [None if a is None else (a.astype(np.float64), np.zeros(a.shape), np.zeros(a.shape)) for a in w]
    for step in range(1, 4):
        g = _stacks(rng, n_res, elems, 1e-3)
        gd = [dev(a, torch.bfloat16 if gdt == "bf16" else torch.float32) for a in g]
        B.fomoe_adamw_resident(wd_, gd, md_, vd_, wc, step, lr=0.0131, weight_decay=0.0 if step < 3 else 0.1)
        for i in range(3):
            if ref[i] is None:
                continue
            gi = H.t2n(gd[i]).astype(np.float64)      # the gradient values the kernel saw (bf16-rounded when gdt == bf16)
            ref[i] = OO.adamw_step(ref[i][0], gi, ref[i][1], ref[i][2], step, 0.0131, weight_decay=0.0 if step < 3 else 0.1)
    torch.cuda.synchronize()
    for i in range(3):
        if ref[i] is None:
            continue
        for got, want, name in ((wd_[i], ref[i][0], "w"), (md_[i], ref[i][1], "m"), (vd_[i], ref[i][2], "v")):
            assert H.rel_err(H.t2n(got), want) <= 1e-5, (i, name, H.rel_err(H.t2n(got), want))
        assert torch.equal(wc[i], wd_[i].to(cdt))


@pytest.mark.parametrize("elems", [(2048, 2048, 4100), (0, 1028, 1028)])
def test_pack_then_outer_nesterov(oracle64, elems):
    import torch
    from paper_2606_19025_b200 import binding as B
    from paper_2606_19025_b200.layer import pack_resident_deltas
    rng = np.random.default_rng(6)
    n_res = 5
    start = _stacks(rng, n_res, elems, 0.02)
    now = [None if a is None else a + (rng.standard_normal(a.shape) * 1e-3).astype(np.float32) for a in start]
    buf = _stacks(rng, n_res, elems, 1e-3)
    slots = np.array([4, 0, 2], np.int32)
    e0 = lambda a, e: torch.zeros((n_res, 0), dtype=torch.float32, device="cuda") if a is None else torch.from_numpy(a).cuda()
    sd, nd, bd = ([e0(a, e) for a, e in zip(t, elems)] for t in (start, now, buf))
    ps = torch.from_numpy(slots).cuda()
    payload = pack_resident_deltas(nd, sd, ps)                      # with one replica the group average is the payload itself
    z = lambda t: [np.zeros((n_res, 0), np.float32) if a is None else a for a in t]
    assert np.array_equal(payload.cpu().numpy().view(np.uint32), oracle64.pack(z(now), z(start), slots).view(np.uint32))
    wc = [None if a is None else torch.empty(a.shape, dtype=torch.bfloat16, device="cuda") for a in start]
    keep = [None if a is None else t.clone() for a, t in zip(start, nd)]
    B.fomoe_outer_nesterov([None if a is None else t for a, t in zip(start, sd)], [None if a is None else t for a, t in zip(start, nd)],
                           [None if a is None else t for a, t in zip(start, bd)], wc, payload, ps, lr=0.7, mu=0.9)
    torch.cuda.synchronize()
    deltas, mask = OO.unpack_blocks(payload.cpu().numpy(), elems, slots, n_res)
    for i in range(3):
        if start[i] is None:
            continue
        w_ref, b_ref = OO.outer_nesterov_step(start[i], deltas[i], buf[i])
        got_w, got_b = H.t2n(sd[i]), H.t2n(bd[i])
        assert H.rel_err(got_w[mask], w_ref[mask]) <= 1e-6 and H.rel_err(got_b[mask], b_ref[mask]) <= 1e-6
        assert torch.equal(sd[i][ps.long()], nd[i][ps.long()])                       # w_now = new round start
        assert np.array_equal(got_w[~mask], start[i][~mask]) and np.array_equal(got_b[~mask], buf[i][~mask])   # untouched
        assert torch.equal(nd[i][torch.from_numpy(~mask).cuda()], keep[i][torch.from_numpy(~mask).cuda()])
        assert torch.equal(wc[i][ps.long()], sd[i][ps.long()].to(torch.bfloat16))
