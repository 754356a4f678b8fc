"""Thin Python binding of libfomoe.so (include/fomoe.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI; PyTorch provides device memory and streams.
The functions keep the C names (fomoe_route, fomoe_moe_fwd, fomoe_moe_bwd, fomoe_pack_resident_deltas,
fomoe_moe_step_host, fomoe_workspace_bytes).  There is no CPU or eager fallback: if the shared library is missing
or a call fails, an exception is raised.
"""
from __future__ import annotations

import ctypes as C
from dataclasses import dataclass
from pathlib import Path
from typing import Optional

import torch

_HERE = Path(__file__).resolve().parent
LIB_PATH = _HERE / "libfomoe.so"

FOMOE_OK, FOMOE_ERR_BADARG, FOMOE_ERR_UNSUPPORTED, FOMOE_ERR_CUDA = 0, -1, -2, -3
FOMOE_F32, FOMOE_BF16 = 0, 1
FOMOE_GATE_SOFTMAX, FOMOE_GATE_SIGMOID = 0, 1
FOMOE_DROP_ONLY, FOMOE_RENORM_TOPK, FOMOE_RENORM_RESIDENT = 0, 1, 2
FOMOE_EXPERT_SWIGLU, FOMOE_EXPERT_SILU = 0, 1
FOMOE_ROUTE_SKIP_TOKEN, FOMOE_ROUTE_FORCED_LOCAL = 0, 1

EXPORTS = ("fomoe_workspace_bytes", "fomoe_route", "fomoe_moe_fwd", "fomoe_moe_bwd", "fomoe_pack_resident_deltas",
           "fomoe_adamw_resident", "fomoe_outer_nesterov", "fomoe_periln_workspace_bytes", "fomoe_periln_fwd", "fomoe_periln_bwd",
           "fomoe_moe_step_host", "fomoe_moe_step_host_join", "fomoe_last_launch_count", "fomoe_last_cuda_error", "fomoe_abi_version",
           "fomoe_set_force_simt", "fomoe_profile_enable", "fomoe_profile_collect", "fomoe_debug_validate_resident",
           "fomoe_routing_stats", "fomoe_moe_fwd_periln", "fomoe_moe_bwd_periln", "fomoe_periln_bwd_noalloc",
           "fomoe_periln_bwd_noalloc_max_floats")
STAT_NAMES = ("kept_fraction", "ghost_fraction", "zero_kept_tokens", "load_cv", "routing_entropy", "max_load", "min_load")


class fomoe_config(C.Structure):
    _fields_ = [("T", C.c_int32), ("d_model", C.c_int32), ("E", C.c_int32), ("top_k", C.c_int32), ("d_ff", C.c_int32),
                ("n_shared", C.c_int32), ("d_ff_shared", C.c_int32), ("dtype", C.c_int32), ("gate_fn", C.c_int32),
                ("gate_rule", C.c_int32), ("temperature", C.c_float), ("expert_fn", C.c_int32), ("route_mode", C.c_int32)]


class fomoe_route_state(C.Structure):
    _fields_ = [("topk_idx", C.c_void_p), ("gate", C.c_void_p), ("probs", C.c_void_p), ("counts", C.c_void_p),
                ("offsets", C.c_void_p), ("row_token", C.c_void_p), ("pair_row", C.c_void_p), ("internal", C.c_void_p)]


class fomoe_periln_post(C.Structure):
    _fields_ = [("gamma", C.c_void_p), ("beta", C.c_void_p), ("eps", C.c_float), ("alpha", C.c_float), ("residual", C.c_void_p),
                ("out", C.c_void_p), ("stats", C.c_void_p)]


class fomoe_periln_pre_bwd(C.Structure):
    _fields_ = [("x_raw", C.c_void_p), ("stats", C.c_void_p), ("gamma", C.c_void_p), ("dresidual", C.c_void_p), ("dgamma", C.c_void_p),
                ("dbeta", C.c_void_p), ("partials", C.c_void_p)]


class FomoeError(RuntimeError):
    pass


_lib = None


def lib() -> C.CDLL:
    """Loads libfomoe.so (built in-tree by paper_2606_19025_b200.build). Raises if it is missing: no fallback."""
    global _lib
    if _lib is None:
        if not LIB_PATH.exists():
            raise FomoeError(f"{LIB_PATH} is missing: build it with `python -m paper_2606_19025_b200.build` (no CPU fallback)")
        _lib = C.CDLL(str(LIB_PATH))
        for name in EXPORTS:
            getattr(_lib, name).restype = C.c_int
        _lib.fomoe_last_cuda_error.restype = C.c_char_p
        _lib.fomoe_periln_bwd_noalloc_max_floats.restype = C.c_size_t
        if _lib.fomoe_abi_version() != 5:
            raise FomoeError("libfomoe.so ABI version mismatch")
    return _lib


def _check(rc: int, what: str) -> None:
    if rc != FOMOE_OK:
        name = {FOMOE_ERR_BADARG: "FOMOE_ERR_BADARG", FOMOE_ERR_UNSUPPORTED: "FOMOE_ERR_UNSUPPORTED",
                FOMOE_ERR_CUDA: "FOMOE_ERR_CUDA"}.get(rc, str(rc))
        raise FomoeError(f"{what} failed: {name} {lib().fomoe_last_cuda_error().decode()}")


def _p(t: Optional[torch.Tensor]) -> C.c_void_p:
    if t is None:
        return C.c_void_p(0)
    assert t.is_contiguous(), "tensors crossing the C ABI must be contiguous"
    return C.c_void_p(t.data_ptr())


def _stream(stream=None) -> C.c_void_p:
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def make_config(T, d_model, E, top_k, d_ff, n_shared=0, d_ff_shared=0, dtype=FOMOE_BF16, gate_fn=FOMOE_GATE_SOFTMAX,
                gate_rule=FOMOE_DROP_ONLY, temperature=1.0, expert_fn=FOMOE_EXPERT_SWIGLU,
                route_mode=FOMOE_ROUTE_SKIP_TOKEN) -> fomoe_config:
    return fomoe_config(T, d_model, E, top_k, d_ff, n_shared, d_ff_shared, dtype, gate_fn, gate_rule, temperature, expert_fn, route_mode)


def fomoe_workspace_bytes(cfg: fomoe_config, n_res: int):
    r, a, s = C.c_size_t(0), C.c_size_t(0), C.c_size_t(0)
    _check(lib().fomoe_workspace_bytes(C.byref(cfg), C.c_int32(n_res), C.byref(r), C.byref(a), C.byref(s)), "fomoe_workspace_bytes")
    return r.value, a.value, s.value


@dataclass
class RouteState:
    """Device tensors behind a fomoe_route_state (caller-owned, as the ABI requires)."""
    topk_idx: torch.Tensor
    gate: torch.Tensor
    probs: torch.Tensor
    counts: torch.Tensor
    offsets: torch.Tensor
    row_token: torch.Tensor
    pair_row: torch.Tensor
    internal: torch.Tensor

    def c_struct(self) -> fomoe_route_state:
        return fomoe_route_state(*(t.data_ptr() for t in (self.topk_idx, self.gate, self.probs, self.counts, self.offsets,
                                                           self.row_token, self.pair_row, self.internal)))


def alloc_route_state(cfg: fomoe_config, n_res: int, device="cuda") -> RouteState:
    rb, _, _ = fomoe_workspace_bytes(cfg, n_res)
    T, k, E = cfg.T, cfg.top_k, cfg.E
    i32 = dict(dtype=torch.int32, device=device)
    return RouteState(
        topk_idx=torch.empty((T, k), **i32), gate=torch.empty((T, k), dtype=torch.float32, device=device),
        probs=torch.empty((T, E), dtype=torch.float32, device=device), counts=torch.empty(max(n_res, 1), **i32)[:n_res],
        offsets=torch.empty(n_res + 1, **i32), row_token=torch.empty(max(T * k, 1), **i32)[:T * k],
        pair_row=torch.empty((T, k), **i32), internal=torch.empty(rb, dtype=torch.uint8, device=device))


def fomoe_route(cfg, x, w_router, router_bias, resident_ids, n_res, route: RouteState, stream=None) -> None:
    rs = route.c_struct()
    _check(lib().fomoe_route(C.byref(cfg), _p(x), _p(w_router), _p(router_bias), _p(resident_ids), C.c_int32(n_res), C.byref(rs),
                             _stream(stream)), "fomoe_route")


def fomoe_moe_fwd(cfg, x, route: RouteState, n_res, w_gate, w_up, w_down, shared, y, saved_acts, scratch, stream=None) -> None:
    rs = route.c_struct()
    sg, su, sd = shared if shared is not None else (None, None, None)
    _check(lib().fomoe_moe_fwd(C.byref(cfg), _p(x), C.byref(rs), C.c_int32(n_res), _p(w_gate), _p(w_up), _p(w_down), _p(sg), _p(su),
                               _p(sd), _p(y), _p(saved_acts), _p(scratch), _stream(stream)), "fomoe_moe_fwd")


def fomoe_moe_bwd(cfg, dy, x, route: RouteState, n_res, w_router, w_gate, w_up, w_down, shared, saved_acts, dx, dw_router, dw_gate,
                  dw_up, dw_down, d_shared, scratch, stream=None) -> None:
    rs = route.c_struct()
    sg, su, sd = shared if shared is not None else (None, None, None)
    dsg, dsu, dsd = d_shared if d_shared is not None else (None, None, None)
    _check(lib().fomoe_moe_bwd(C.byref(cfg), _p(dy), _p(x), C.byref(rs), C.c_int32(n_res), _p(w_router), _p(w_gate), _p(w_up),
                               _p(w_down), _p(sg), _p(su), _p(sd), _p(saved_acts), _p(dx), _p(dw_router), _p(dw_gate), _p(dw_up),
                               _p(dw_down), _p(dsg), _p(dsu), _p(dsd), _p(scratch), _stream(stream)), "fomoe_moe_bwd")


def fomoe_periln_fused_supported(cfg) -> bool:
    """Whether d_model fits the register-resident row shape of the fused Peri-LN forms (host-side shape rule of fomoe.h)."""
    vn = 8 if cfg.dtype == FOMOE_BF16 else 4
    return cfg.d_model % vn == 0 and cfg.d_model // vn <= 1024


def _dp(t: Optional[torch.Tensor]):
    return None if t is None else t.data_ptr()


def fomoe_moe_fwd_periln(cfg, x, route: RouteState, n_res, w_gate, w_up, w_down, shared, y, saved_acts, scratch, gamma, beta, residual,
                         out, stats, alpha=1.0, eps=1e-5, stream=None) -> None:
    """fomoe_moe_fwd whose combine also applies the post-LN, the depth multiplier and the residual (Eq. 15)."""
    rs = route.c_struct()
    sg, su, sd = shared if shared is not None else (None, None, None)
    ln = fomoe_periln_post(_dp(gamma), _dp(beta), eps, alpha, _dp(residual), _dp(out), _dp(stats))
    _check(lib().fomoe_moe_fwd_periln(C.byref(cfg), _p(x), C.byref(rs), C.c_int32(n_res), _p(w_gate), _p(w_up), _p(w_down), _p(sg), _p(su),
                                      _p(sd), _p(y), _p(saved_acts), _p(scratch), C.byref(ln), _stream(stream)), "fomoe_moe_fwd_periln")


def fomoe_moe_bwd_periln(cfg, dy, x, route: RouteState, n_res, w_router, w_gate, w_up, w_down, shared, saved_acts, dx, dw_router, dw_gate,
                         dw_up, dw_down, d_shared, scratch, x_raw, stats, gamma, dresidual, dgamma, dbeta, partials, stream=None) -> None:
    """fomoe_moe_bwd whose scatter-sum also applies the pre-LN backward and adds the residual-branch gradient."""
    rs = route.c_struct()
    sg, su, sd = shared if shared is not None else (None, None, None)
    dsg, dsu, dsd = d_shared if d_shared is not None else (None, None, None)
    ln = fomoe_periln_pre_bwd(_dp(x_raw), _dp(stats), _dp(gamma), _dp(dresidual), _dp(dgamma), _dp(dbeta), _dp(partials))
    _check(lib().fomoe_moe_bwd_periln(C.byref(cfg), _p(dy), _p(x), C.byref(rs), C.c_int32(n_res), _p(w_router), _p(w_gate), _p(w_up),
                                      _p(w_down), _p(sg), _p(su), _p(sd), _p(saved_acts), _p(dx), _p(dw_router), _p(dw_gate), _p(dw_up),
                                      _p(dw_down), _p(dsg), _p(dsu), _p(dsd), _p(scratch), C.byref(ln), _stream(stream)),
           "fomoe_moe_bwd_periln")


def fomoe_pack_resident_deltas(w_now, w_start, pack_slots, payload, stream=None) -> None:
    """w_now / w_start: 3-tuples of fp32 device tensors [n_res, ...] (gate, up, down); payload fp32 [n_pack, block]."""
    n_res = w_now[0].shape[0]
    elems = [int(t[0].numel()) if n_res else 0 for t in w_now]
    arr3 = C.c_void_p * 3
    now = arr3(*(t.data_ptr() for t in w_now))
    start = arr3(*(t.data_ptr() for t in w_start))
    n_pack = n_res if pack_slots is None else int(pack_slots.numel())
    _check(lib().fomoe_pack_resident_deltas(now, start, C.c_int32(n_res), C.c_int64(elems[0]), C.c_int64(elems[1]),
                                            C.c_int64(elems[2]), _p(pack_slots), C.c_int32(n_pack), _p(payload), _stream(stream)),
           "fomoe_pack_resident_deltas")


def _dt(t: torch.Tensor) -> int:
    return FOMOE_BF16 if t.dtype == torch.bfloat16 else FOMOE_F32


def fomoe_periln_workspace_bytes(T: int, d_model: int) -> int:
    n = C.c_size_t(0)
    _check(lib().fomoe_periln_workspace_bytes(C.c_int32(T), C.c_int32(d_model), C.byref(n)), "fomoe_periln_workspace_bytes")
    return n.value


def fomoe_periln_fwd(x, gamma, beta, out, stats, residual=None, alpha=1.0, eps=1e-5, stream=None) -> None:
    T, d = x.shape
    _check(lib().fomoe_periln_fwd(C.c_int32(T), C.c_int32(d), C.c_int32(_dt(x)), _p(x), _p(gamma), _p(beta), C.c_float(eps), _p(residual),
                                  C.c_float(alpha), _p(out), _p(stats), _stream(stream)), "fomoe_periln_fwd")


def fomoe_periln_bwd(dout, x, stats, gamma, dx, dgamma, dbeta, partials, dresidual=None, alpha=1.0, stream=None) -> None:
    T, d = x.shape
    _check(lib().fomoe_periln_bwd(C.c_int32(T), C.c_int32(d), C.c_int32(_dt(x)), _p(dout), _p(x), _p(stats), _p(gamma), C.c_float(alpha),
                                  _p(dresidual), _p(dx), _p(dgamma), _p(dbeta), _p(partials), _stream(stream)), "fomoe_periln_bwd")


def fomoe_periln_bwd_noalloc(dout, x, stats, gamma, dx, dgamma, dbeta, dresidual=None, alpha=1.0, stream=None) -> None:
    """fomoe_periln_bwd with its partial-sum workspace in the library's static device array (no allocation anywhere)."""
    T, d = x.shape
    _check(lib().fomoe_periln_bwd_noalloc(C.c_int32(T), C.c_int32(d), C.c_int32(_dt(x)), _p(dout), _p(x), _p(stats), _p(gamma),
                                          C.c_float(alpha), _p(dresidual), _p(dx), _p(dgamma), _p(dbeta), _stream(stream)),
           "fomoe_periln_bwd_noalloc")


def fomoe_periln_bwd_noalloc_max_floats() -> int:
    return int(lib().fomoe_periln_bwd_noalloc_max_floats())


def _arr3(ts):
    """Host array of 3 device pointers; None entries (zero-element tensors, two-matrix expert) become NULL."""
    return (C.c_void_p * 3)(*(0 if t is None or t.numel() == 0 else t.data_ptr() for t in ts))


def _elems3(ts):
    return [0 if t is None or t.shape[0] == 0 else int(t[0].numel()) for t in ts]


def fomoe_adamw_resident(w_master, grad, m, v, w_compute, step, lr, beta1=0.9, beta2=0.95, eps=1e-8, weight_decay=0.0,
                         stream=None) -> None:
    """3-tuples (gate, up, down) of device tensors [n_res, ...]: fp32 master / moments, grads in f32 or bf16."""
    n_res = next(t.shape[0] for t in w_master if t is not None)
    e = _elems3(w_master)
    gd = next(t for t in grad if t is not None).dtype
    dtype = FOMOE_BF16 if gd == torch.bfloat16 else FOMOE_F32
    wc = _arr3(w_compute) if w_compute is not None else None
    assert w_compute is None or all(t is None or t.dtype == gd for t in w_compute), "w_compute must have the gradients' dtype"
    _check(lib().fomoe_adamw_resident(_arr3(w_master), _arr3(grad), _arr3(m), _arr3(v), wc, C.c_int32(dtype), C.c_int32(n_res),
                                      C.c_int64(e[0]), C.c_int64(e[1]), C.c_int64(e[2]), C.c_int32(step), C.c_float(lr),
                                      C.c_float(beta1), C.c_float(beta2), C.c_float(eps), C.c_float(weight_decay), _stream(stream)),
           "fomoe_adamw_resident")


def fomoe_outer_nesterov(w_start, w_now, momentum, w_compute, payload_avg, pack_slots=None, lr=0.7, mu=0.9, stream=None) -> None:
    n_res = next(t.shape[0] for t in w_start if t is not None)
    e = _elems3(w_start)
    dtype = FOMOE_F32
    wc = None
    if w_compute is not None:
        wc = _arr3(w_compute)
        dtype = FOMOE_BF16 if next(t for t in w_compute if t is not None).dtype == torch.bfloat16 else FOMOE_F32
    n_pack = n_res if pack_slots is None else int(pack_slots.numel())
    _check(lib().fomoe_outer_nesterov(_arr3(w_start), _arr3(w_now), _arr3(momentum), wc, C.c_int32(dtype), _p(payload_avg),
                                      C.c_int32(n_res), C.c_int64(e[0]), C.c_int64(e[1]), C.c_int64(e[2]), _p(pack_slots),
                                      C.c_int32(n_pack), C.c_float(lr), C.c_float(mu), _stream(stream)), "fomoe_outer_nesterov")


def fomoe_moe_step_host(cfg, x_host, dy_host, y_host, dx_host, x_dev, dy_dev, y_dev, dx_dev, w_router, router_bias, resident_ids,
                        n_res, route: RouteState, w_gate, w_up, w_down, shared, dw_router, dw_gate, dw_up, dw_down, d_shared,
                        saved_acts, scratch, stream=None, copy_stream=None, defer_join=False) -> None:
    rs = route.c_struct()
    sg, su, sd = shared if shared is not None else (None, None, None)
    dsg, dsu, dsd = d_shared if d_shared is not None else (None, None, None)
    _check(lib().fomoe_moe_step_host(
        C.byref(cfg), _p(x_host), _p(dy_host), _p(y_host), _p(dx_host), _p(x_dev), _p(dy_dev), _p(y_dev), _p(dx_dev), _p(w_router),
        _p(router_bias), _p(resident_ids), C.c_int32(n_res), C.byref(rs), _p(w_gate), _p(w_up), _p(w_down), _p(sg), _p(su), _p(sd),
        _p(dw_router), _p(dw_gate), _p(dw_up), _p(dw_down), _p(dsg), _p(dsu), _p(dsd), _p(saved_acts), _p(scratch),
        _stream(stream), _stream(copy_stream if copy_stream is not None else stream), C.c_int32(1 if defer_join else 0)),
        "fomoe_moe_step_host")


def fomoe_moe_step_host_join(stream=None) -> None:
    _check(lib().fomoe_moe_step_host_join(_stream(stream)), "fomoe_moe_step_host_join")


def fomoe_debug_validate_resident(resident_ids, E: int, stream=None) -> None:
    """Synchronising content check of the resident set; raises FomoeError (BADARG) on out-of-range / duplicate / unsorted ids."""
    _check(lib().fomoe_debug_validate_resident(_p(resident_ids), C.c_int32(int(resident_ids.numel())), C.c_int32(E), _stream(stream)),
           "fomoe_debug_validate_resident")


def fomoe_routing_stats(cfg, route: RouteState, n_res: int, load: torch.Tensor, stats: torch.Tensor, stream=None) -> None:
    """load: int32 [E + 2], stats: fp32 [8] device tensors (see include/fomoe.h)."""
    rs = route.c_struct()
    _check(lib().fomoe_routing_stats(C.byref(cfg), C.byref(rs), C.c_int32(n_res), _p(load), _p(stats), _stream(stream)),
           "fomoe_routing_stats")


def fomoe_last_launch_count() -> int:
    return int(lib().fomoe_last_launch_count())


def fomoe_set_force_simt(on: bool) -> bool:
    return bool(lib().fomoe_set_force_simt(C.c_int(1 if on else 0)))


def fomoe_profile_enable(on: bool) -> None:
    _check(lib().fomoe_profile_enable(C.c_int(1 if on else 0)), "fomoe_profile_enable")


def fomoe_profile_collect(cap: int = 4096):
    """Returns [(kernel name, ms), ...] recorded since fomoe_profile_enable(True)."""
    names = (C.c_char_p * cap)()
    ms = (C.c_float * cap)()
    n = lib().fomoe_profile_collect(names, ms, C.c_int(cap))
    return [(names[i].decode(), float(ms[i])) for i in range(min(n, cap))]
