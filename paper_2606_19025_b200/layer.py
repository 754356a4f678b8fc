"""SkipTokenMoE: the call a user makes.  Owns the device tensors and workspaces of one partially resident MoE layer
and drives the C ABI (binding.py) — route, forward, backward, delta pack.  No arithmetic happens here.
"""
from __future__ import annotations

from typing import Optional

import numpy as np
import torch

from . import binding as B
from .workloads import MoEWorkload


def _dev(a: Optional[np.ndarray], dtype: torch.dtype, device) -> Optional[torch.Tensor]:
    if a is None:
        return None
    t = torch.from_numpy(np.ascontiguousarray(a))
    return t.to(device=device, dtype=dtype).contiguous()


class SkipTokenMoE:
    def __init__(self, w: MoEWorkload, resident: np.ndarray, w_router: np.ndarray, w_gate, w_up, w_down, shared=None,
                 router_bias: Optional[np.ndarray] = None, device="cuda"):
        """Arrays are numpy fp32 holding storage-dtype-exact values (workloads.py); experts are resident-compact stacks."""
        if not torch.cuda.is_available():
            raise B.FomoeError("SkipTokenMoE needs a CUDA device: there is no CPU fallback")
        B.lib()
        self.w = w
        self.device = torch.device(device)
        self.n_res = int(len(resident))
        self.tdtype = torch.bfloat16 if w.dtype == "bf16" else torch.float32
        self.cfg = B.make_config(w.T, w.d, w.E, w.k, w.F, w.n_sh, w.F_sh, B.FOMOE_BF16 if w.dtype == "bf16" else B.FOMOE_F32,
                                 w.gate_fn, w.gate_rule, w.temperature, w.expert_fn, w.route_mode)
        dv, td = self.device, self.tdtype
        self.resident = _dev(np.asarray(resident, np.int32), torch.int32, dv) if self.n_res else torch.empty(0, dtype=torch.int32, device=dv)
        self.w_router = _dev(w_router, torch.float32, dv)
        self.router_bias = _dev(router_bias, torch.float32, dv)
        self.w_gate, self.w_up, self.w_down = (_dev(a, td, dv) for a in (w_gate, w_up, w_down))
        self.shared = None if shared is None else tuple(_dev(a, td, dv) for a in shared)
        rb, ab, sb = B.fomoe_workspace_bytes(self.cfg, self.n_res)
        self.route_state = B.alloc_route_state(self.cfg, self.n_res, dv)
        self.saved_acts = torch.empty(ab, dtype=torch.uint8, device=dv)
        self.scratch = torch.empty(sb, dtype=torch.uint8, device=dv)
        self.y = torch.empty((w.T, w.d), dtype=td, device=dv)
        self.dx = torch.empty((w.T, w.d), dtype=td, device=dv)
        self.dw_router = torch.empty((w.d, w.E), dtype=torch.float32, device=dv)
        # (the paper's two-matrix expert has no W_gate: w_gate / shared[0] are None then, and so are their gradients)
        self.dw_gate, self.dw_up, self.dw_down = (None if t is None else torch.empty_like(t) for t in (self.w_gate, self.w_up, self.w_down))
        self.d_shared = None if self.shared is None else tuple(None if t is None else torch.empty_like(t) for t in self.shared)
        self.launches = 0

    def to_dev(self, a: np.ndarray) -> torch.Tensor:
        return _dev(a, self.tdtype, self.device)

    def route(self, x: torch.Tensor, stream=None):
        B.fomoe_route(self.cfg, x, self.w_router, self.router_bias, self.resident, self.n_res, self.route_state, stream)
        self.launches = B.fomoe_last_launch_count()
        return self.route_state

    def forward(self, x: torch.Tensor, stream=None) -> torch.Tensor:
        B.fomoe_moe_fwd(self.cfg, x, self.route_state, self.n_res, self.w_gate, self.w_up, self.w_down, self.shared, self.y,
                        self.saved_acts, self.scratch, stream)
        self.launches = B.fomoe_last_launch_count()
        return self.y

    def backward(self, dy: torch.Tensor, x: torch.Tensor, stream=None):
        B.fomoe_moe_bwd(self.cfg, dy, x, self.route_state, self.n_res, self.w_router, self.w_gate, self.w_up, self.w_down, self.shared,
                        self.saved_acts, self.dx, self.dw_router, self.dw_gate, self.dw_up, self.dw_down, self.d_shared, self.scratch,
                        stream)
        self.launches = B.fomoe_last_launch_count()
        return self.dx

    def forward_periln(self, xn: torch.Tensor, gamma, beta, residual, out, stats, alpha=1.0, eps=1e-5, stream=None) -> torch.Tensor:
        """Forward on the pre-LN output xn; the combine also writes out = residual + alpha LN(y) (Eq. 15)."""
        B.fomoe_moe_fwd_periln(self.cfg, xn, self.route_state, self.n_res, self.w_gate, self.w_up, self.w_down, self.shared, self.y,
                               self.saved_acts, self.scratch, gamma, beta, residual, out, stats, alpha, eps, stream)
        self.launches = B.fomoe_last_launch_count()
        return out

    def backward_periln(self, dy: torch.Tensor, xn: torch.Tensor, x_raw, stats, gamma, dresidual, dgamma, dbeta, partials, stream=None):
        """Backward whose final scatter-sum applies the pre-LN backward: self.dx = gradient w.r.t. the BLOCK input."""
        B.fomoe_moe_bwd_periln(self.cfg, dy, xn, self.route_state, self.n_res, self.w_router, self.w_gate, self.w_up, self.w_down,
                               self.shared, self.saved_acts, self.dx, self.dw_router, self.dw_gate, self.dw_up, self.dw_down, self.d_shared,
                               self.scratch, x_raw, stats, gamma, dresidual, dgamma, dbeta, partials, stream)
        self.launches = B.fomoe_last_launch_count()
        return self.dx

    def step(self, x: torch.Tensor, dy: torch.Tensor, stream=None) -> int:
        """route + forward + backward on device-resident inputs; returns the number of kernels launched."""
        n = 0
        self.route(x, stream); n += self.launches
        self.forward(x, stream); n += self.launches
        self.backward(dy, x, stream); n += self.launches
        self.launches = n
        return n

    def capture_step(self, x: torch.Tensor, dy: torch.Tensor):
        """Captures route + forward + backward on (x, dy) into a CUDA graph (no entry point syncs or reads back, so the
        whole step is capturable).  Returns a callable that replays it; inputs are read from the captured buffers."""
        s = torch.cuda.Stream()
        s.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(s):
            for _ in range(2):  # warm up: first-call attribute setup must not happen during capture
                n = self.step(x, dy)
        torch.cuda.current_stream().wait_stream(s)
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            self.step(x, dy)
        self.launches = n
        return g.replay

    def step_host(self, x_host, dy_host, y_host, dx_host, x_dev, dy_dev, stream=None, copy_stream=None, defer_join=False) -> int:
        """Whole step from pinned HOST buffers through fomoe_moe_step_host (uploads x, dy; downloads y, dx).  defer_join=True
        leaves the downloads running (call host_join() before reading y_host / dx_host): with alternating (x_dev, dy_dev) pairs
        consecutive steps then overlap their PCIe copies with each other's compute."""
        B.fomoe_moe_step_host(self.cfg, x_host, dy_host, y_host, dx_host, x_dev, dy_dev, self.y, self.dx, self.w_router,
                              self.router_bias, self.resident, self.n_res, self.route_state, self.w_gate, self.w_up, self.w_down,
                              self.shared, self.dw_router, self.dw_gate, self.dw_up, self.dw_down, self.d_shared, self.saved_acts,
                              self.scratch, stream, copy_stream, defer_join)
        self.launches = B.fomoe_last_launch_count()
        return self.launches

    def host_join(self, stream=None) -> None:
        B.fomoe_moe_step_host_join(stream)

    def routing_numpy(self) -> dict:
        """Device -> host copy of the public routing outputs (tests / diagnostics only)."""
        r = self.route_state
        out = {k: getattr(r, k).cpu().numpy() for k in ("topk_idx", "gate", "probs", "counts", "offsets", "row_token", "pair_row")}
        out["P"] = int(out["offsets"][-1])
        return out


    def routing_stats(self, stream=None) -> dict:
        """Routing diagnostics of the last route() (fomoe_routing_stats): device kernel, read back here."""
        load = torch.empty(self.w.E + 2, dtype=torch.int32, device=self.device)
        stats = torch.empty(8, dtype=torch.float32, device=self.device)
        B.fomoe_routing_stats(self.cfg, self.route_state, self.n_res, load, stats, stream)
        vals = stats.cpu().tolist()
        out = dict(zip(B.STAT_NAMES, vals))
        out["load"] = load[:self.w.E].cpu().numpy()
        return out


def pack_resident_deltas(w_now, w_start, pack_slots: Optional[torch.Tensor] = None, payload: Optional[torch.Tensor] = None,
                         stream=None) -> torch.Tensor:
    """fp32 payload [n_pack, elems_gate + elems_up + elems_down] = w_start - w_now per packed slot (fomoe_pack_resident_deltas)."""
    n_res = w_now[0].shape[0]
    n_pack = n_res if pack_slots is None else int(pack_slots.numel())
    block = sum(int(t[0].numel()) for t in w_now) if n_res else 0
    if payload is None:
        payload = torch.empty((n_pack, block), dtype=torch.float32, device=w_now[0].device)
    B.fomoe_pack_resident_deltas(w_now, w_start, pack_slots, payload, stream)
    return payload
