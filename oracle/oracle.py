"""ORACLE — TEST INFRASTRUCTURE, NOT THE PRODUCT (see the header of fomoe_oracle.c).

ctypes loader for the plain-C CPU oracle.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module.  It imports nothing from the CUDA package.

`Oracle("f64")` is the parity reference (and the finite-difference build); `Oracle("f32")` is the plain
fp32 implementation that is timed as the CPU baseline.  Arrays in / out are numpy, C-contiguous.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "fomoe_oracle.c"
_LIBS = {"f64": ("liboracle_f64.so", "double", np.float64), "f32": ("liboracle_f32.so", "float", np.float32)}


def build(force: bool = False) -> None:
    """gcc -O3 -fopenmp, one shared object per REAL type."""
    for name, (lib, ctype, _) in _LIBS.items():
        out = _HERE / lib
        if not force and out.exists() and out.stat().st_mtime >= _SRC.stat().st_mtime:
            continue
        cmd = ["gcc", "-O3", "-march=x86-64-v3", "-fopenmp", "-fPIC", "-shared", "-std=c11", f"-DREAL={ctype}",
               str(_SRC), "-o", str(out), "-lm"]
        subprocess.run(cmd, check=True)


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


class Oracle:
    def __init__(self, real: str = "f64"):
        build()
        lib, _, self.dt = _LIBS[real]
        self.real = real
        self.lib = C.CDLL(str(_HERE / lib))
        assert self.lib.oracle_real_bytes() == np.dtype(self.dt).itemsize
        for fn in ("oracle_route", "oracle_moe_fwd", "oracle_moe_bwd", "oracle_pack_resident_deltas", "oracle_dw_sample"):
            getattr(self.lib, fn).restype = C.c_int

    @staticmethod
    def threads() -> int:
        return int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))

    def _r(self, a):
        return None if a is None else np.ascontiguousarray(a, dtype=self.dt)

    # ---- steps 1-6 -------------------------------------------------------------------------------
    def route(self, x, w_r, resident, k, gate_fn=0, gate_rule=0, tau=1.0, bias=None, route_mode=0):
        """route_mode 0 = skip-token (top-k over all E, ghosts dropped), 1 = forced-local (router over resident experts only)."""
        x, w_r, bias = self._r(x), self._r(w_r), self._r(bias)
        resident = np.ascontiguousarray(resident, dtype=np.int32)
        T, d = x.shape
        E = w_r.shape[1]
        n_res = len(resident)
        out = dict(
            logits=np.empty((T, E), self.dt), probs=np.empty((T, E), self.dt),
            topk_idx=np.empty((T, k), np.int32), gate=np.empty((T, k), self.dt),
            counts=np.zeros(n_res, np.int32), offsets=np.zeros(n_res + 1, np.int32),
            row_token=np.empty(T * k, np.int32), pair_row=np.empty((T, k), np.int32))
        rc = self.lib.oracle_route(C.c_int(T), C.c_int(d), C.c_int(E), C.c_int(k), C.c_int(gate_fn), C.c_int(gate_rule),
                                   C.c_double(tau), C.c_int(route_mode), _ptr(x), _ptr(w_r), _ptr(bias), _ptr(resident), C.c_int(n_res),
                                   _ptr(out["logits"]), _ptr(out["probs"]), _ptr(out["topk_idx"]), _ptr(out["gate"]),
                                   _ptr(out["counts"]), _ptr(out["offsets"]), _ptr(out["row_token"]), _ptr(out["pair_row"]))
        if rc != 0:
            raise ValueError(f"oracle_route rc={rc}")
        out["P"] = int(out["offsets"][-1])
        return out

    # ---- steps 7-8 -------------------------------------------------------------------------------
    def moe_fwd(self, x, route, resident, w_gate, w_up, w_down, shared=None, E=None, expert_fn=0):
        """expert_fn 0 = SwiGLU, 1 = the paper's W_down silu(W_up x) (w_gate and shared[0] are None then)."""
        x = self._r(x)
        resident = np.ascontiguousarray(resident, dtype=np.int32)
        T, d = x.shape
        k = route["topk_idx"].shape[1]
        E = route["probs"].shape[1] if E is None else E
        wg, wu, wd = self._r(w_gate), self._r(w_up), self._r(w_down)
        F = wu.shape[1] if wu.ndim == 3 and wu.shape[0] > 0 else (wd.shape[2] if wd.ndim == 3 else 0)
        sg = su = sd = None
        n_sh = F_sh = 0
        if shared is not None:
            sg, su, sd = (self._r(s) for s in shared)
            n_sh, F_sh = su.shape[0], su.shape[1]
        y = np.empty((T, d), self.dt)
        rc = self.lib.oracle_moe_fwd(C.c_int(T), C.c_int(d), C.c_int(E), C.c_int(k), C.c_int(F), C.c_int(n_sh), C.c_int(F_sh),
                                     C.c_int(expert_fn), _ptr(x), _ptr(route["topk_idx"]), _ptr(self._r(route["gate"])),
                                     _ptr(resident), C.c_int(len(resident)), _ptr(wg), _ptr(wu), _ptr(wd),
                                     _ptr(sg), _ptr(su), _ptr(sd), _ptr(y))
        if rc != 0:
            raise ValueError(f"oracle_moe_fwd rc={rc}")
        return y

    # ---- step 9 ----------------------------------------------------------------------------------
    def moe_bwd(self, x, dy, w_r, route, resident, w_gate, w_up, w_down, shared=None,
                gate_fn=0, gate_rule=0, tau=1.0, expert_fn=0):
        x, dy, w_r = self._r(x), self._r(dy), self._r(w_r)
        resident = np.ascontiguousarray(resident, dtype=np.int32)
        T, d = x.shape
        E = w_r.shape[1]
        k = route["topk_idx"].shape[1]
        wg, wu, wd = self._r(w_gate), self._r(w_up), self._r(w_down)
        n_res = len(resident)
        F = wu.shape[1]
        sg = su = sd = None
        n_sh = F_sh = 0
        if shared is not None:
            sg, su, sd = (self._r(s) for s in shared)
            n_sh, F_sh = su.shape[0], su.shape[1]
        out = dict(dx=np.empty((T, d), self.dt), dw_router=np.empty((d, E), self.dt),
                   dw_up=np.empty((n_res, F, d), self.dt), dw_down=np.empty((n_res, d, F), self.dt),
                   dgate=np.empty((T, k), self.dt), dlogits=np.empty((T, E), self.dt))
        if wg is not None:
            out["dw_gate"] = np.empty((n_res, F, d), self.dt)
        if shared is not None:
            out.update(d_sh_up=np.empty_like(su), d_sh_down=np.empty_like(sd))
            if sg is not None:
                out["d_sh_gate"] = np.empty_like(sg)
        rc = self.lib.oracle_moe_bwd(
            C.c_int(T), C.c_int(d), C.c_int(E), C.c_int(k), C.c_int(F), C.c_int(n_sh), C.c_int(F_sh), C.c_int(expert_fn),
            C.c_int(gate_fn), C.c_int(gate_rule), C.c_double(tau),
            _ptr(x), _ptr(dy), _ptr(w_r), _ptr(self._r(route["probs"])), _ptr(route["topk_idx"]), _ptr(self._r(route["gate"])),
            _ptr(resident), C.c_int(n_res), _ptr(route["offsets"]), _ptr(route["row_token"]),
            _ptr(wg), _ptr(wu), _ptr(wd), _ptr(sg), _ptr(su), _ptr(sd),
            _ptr(out["dx"]), _ptr(out["dw_router"]), _ptr(out.get("dw_gate")), _ptr(out["dw_up"]), _ptr(out["dw_down"]),
            _ptr(out.get("d_sh_gate")), _ptr(out.get("d_sh_up")), _ptr(out.get("d_sh_down")),
            _ptr(out["dgate"]), _ptr(out["dlogits"]))
        if rc != 0:
            raise ValueError(f"oracle_moe_bwd rc={rc}")
        return out

    # ---- sampled weight gradients (full-size parity) -----------------------------------------------
    def dw_sample(self, x, dy, route, resident, slot, f_idx, w_gate_s, w_up_s, w_down_s, expert_fn=0):
        """dW_gate[slot, f, :], dW_up[slot, f, :], dW_down[slot, :, f] for f in f_idx; weights are that slot's matrices."""
        x, dy = self._r(x), self._r(dy)
        wg, wu, wd = self._r(w_gate_s), self._r(w_up_s), self._r(w_down_s)
        F, d = wu.shape
        k = route["topk_idx"].shape[1]
        f_idx = np.ascontiguousarray(f_idx, dtype=np.int32)
        outs = [np.empty((len(f_idx), d), self.dt) for _ in range(3)]
        rc = self.lib.oracle_dw_sample(C.c_int(d), C.c_int(k), C.c_int(F), C.c_int(expert_fn), _ptr(x), _ptr(dy), _ptr(route["topk_idx"]),
                                       _ptr(self._r(route["gate"])), C.c_int(int(resident[slot])),
                                       C.c_int(int(route["offsets"][slot])), C.c_int(int(route["offsets"][slot + 1])),
                                       _ptr(route["row_token"]), _ptr(wg), _ptr(wu), _ptr(wd), _ptr(f_idx), C.c_int(len(f_idx)),
                                       _ptr(outs[0]), _ptr(outs[1]), _ptr(outs[2]))
        if rc != 0:
            raise ValueError(f"oracle_dw_sample rc={rc}")
        return outs

    # ---- step 10 ---------------------------------------------------------------------------------
    def pack(self, w_now, w_start, pack_slots=None):
        """w_now / w_start: 3-tuples of fp32 [n_res, ...] stacks (gate, up, down). Returns fp32 payload [n_pack, block]."""
        now = [np.ascontiguousarray(a, dtype=np.float32) for a in w_now]
        start = [np.ascontiguousarray(a, dtype=np.float32) for a in w_start]
        n_res = now[0].shape[0]
        elems = [int(np.prod(a.shape[1:])) for a in now]
        slots = None if pack_slots is None else np.ascontiguousarray(pack_slots, dtype=np.int32)
        n_pack = n_res if slots is None else len(slots)
        payload = np.empty((n_pack, sum(elems)), np.float32)
        rc = self.lib.oracle_pack_resident_deltas(_ptr(now[0]), _ptr(now[1]), _ptr(now[2]),
                                                  _ptr(start[0]), _ptr(start[1]), _ptr(start[2]),
                                                  C.c_int(n_res), C.c_int64(elems[0]), C.c_int64(elems[1]), C.c_int64(elems[2]),
                                                  _ptr(slots), C.c_int(n_pack), _ptr(payload))
        if rc != 0:
            raise ValueError(f"oracle_pack rc={rc}")
        return payload
