#!/usr/bin/env python
"""bench.py — skip-token MoE layer tokens/s, forward + backward, on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C2] [--impl reference]

A "step" is one pass of the hot path over one batch resident in HBM: fomoe_route + fomoe_moe_fwd + fomoe_moe_bwd
(rows F1-F8, B1-B7 of SURVEY.md §8(a)).  The resident-delta pack (row S1) runs once per K local steps at a round
boundary, so it is timed beside the step and reported under "pack", not inside tokens/s.
Prints ONE JSON line (see DESIGN.md "Measurement" for every key).  --impl reference times the CPU oracle instead.
N > 1: one process per GPU (torchrun), independent replicas, no collective on the data path ("scaling": "weak").
"""
from __future__ import annotations

import argparse
import dataclasses
import json
import os
import statistics
import subprocess
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

from paper_2606_19025_b200 import workloads as W  # noqa: E402

METRIC = "skip-token MoE layer tokens/s fwd+bwd"
UNIT = "tokens/s"
FALLBACK_PEAKS = {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}  # B200_PROFILING.md fallback


def workload_desc(w: W.MoEWorkload, n_res: int) -> str:
    sh = f" + {w.n_sh} shared (d_ff {w.F_sh})" if w.n_sh else ""
    ex = "SwiGLU d_ff" if w.expert_fn == W.EXPERT_SWIGLU else "two-matrix SiLU expert (PAPER.md:589) d_expert"
    gf = "softmax" if w.gate_fn == W.GATE_SOFTMAX else "sigmoid"
    return (f"{w.name}: T={w.T}, d_model={w.d}, E={w.E}{sh}, top-{w.k}, {gf} gate, {ex}={w.F}, {n_res} of {w.E} resident, "
            f"{w.dtype}, fp32 router, x~N(0,1), weights~N(0,0.02), seed {w.seed}"
            + (f", Zipf(alpha={w.zipf_alpha}) router bias" if w.zipf_alpha else ""))


def load_peaks():
    f = ROOT / "MEASURED_PEAKS.json"
    if f.exists():
        try:
            d = json.loads(f.read_text())
            return {k: float(d[k]) for k in FALLBACK_PEAKS}, "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return dict(FALLBACK_PEAKS), "fallback (B200_PROFILING.md)"


# ------------------------------------------------------------------------------------------------------------------
# clocks sampled DURING the timed region
# ------------------------------------------------------------------------------------------------------------------
class ClockSampler:
    """SM clock + throttle reasons sampled DURING the timed region: NVML polled every 2 ms from a thread (the timed region
    of the small workloads lasts ~10 ms, too short for nvidia-smi's 100 ms loop), nvidia-smi as the fallback."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
    NAMES = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index
        self.nvml, self.handle, self.stop_flag, self.thread = None, None, False, None
        try:
            import pynvml
            import torch
            pynvml.nvmlInit()
            try:
                uuid = str(torch.cuda.get_device_properties(index).uuid)
                self.handle = pynvml.nvmlDeviceGetHandleByUUID(("GPU-" + uuid) if not uuid.startswith("GPU-") else uuid)
            except Exception:
                self.handle = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.nvml = pynvml
        except Exception:
            self.nvml = None

    def _poll(self):
        n = self.nvml
        bits = ((getattr(n, "nvmlClocksThrottleReasonHwSlowdown", 0x8), "hw_slowdown"),
                (getattr(n, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40), "hw_thermal_slowdown"),
                (getattr(n, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20), "sw_thermal_slowdown"),
                (getattr(n, "nvmlClocksThrottleReasonSwPowerCap", 0x4), "sw_power_cap"))
        mx = float(n.nvmlDeviceGetMaxClockInfo(self.handle, n.NVML_CLOCK_SM))
        while not self.stop_flag:
            try:
                sm = float(n.nvmlDeviceGetClockInfo(self.handle, n.NVML_CLOCK_SM))
                r = int(n.nvmlDeviceGetCurrentClocksThrottleReasons(self.handle))
                self.rows.append((sm, mx, [nm for b, nm in bits if r & b], time.perf_counter()))
            except Exception:
                pass
            time.sleep(0.002)

    def start(self):
        if self.nvml is not None:
            self.thread = threading.Thread(target=self._poll, daemon=True)
            self.thread.start()
            return
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            c = [v.strip() for v in line.split(",")]
            try:
                self.rows.append((float(c[0]), float(c[1]), [nm for nm, v in zip(self.NAMES, c[3:7]) if v.lower().startswith("active")],
                                  time.perf_counter()))
            except Exception:
                continue

    def stop(self, window=None):
        """window = (t0, t1) perf_counter bounds of the timed region: only samples inside it count (the sampler is started
        before the warm-up so that a short region still has samples; if none fell inside, the two nearest ones are used)."""
        if self.thread is not None:
            self.stop_flag = True
            self.thread.join()
            src = "nvml, 2 ms poll"
            if not self.rows:   # a region of a few ms can end before the first poll returns: one sample right after it
                try:
                    n = self.nvml
                    sm = float(n.nvmlDeviceGetClockInfo(self.handle, n.NVML_CLOCK_SM))
                    mx = float(n.nvmlDeviceGetMaxClockInfo(self.handle, n.NVML_CLOCK_SM))
                    self.rows.append((sm, mx, [], time.perf_counter()))
                    src = "nvml, one sample right after the timed region (no poll landed inside it)"
                except Exception:
                    pass
        elif self.proc is not None:
            time.sleep(0.15)
            self.proc.terminate()
            src = "nvidia-smi -lms 100"
        else:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvml and nvidia-smi unavailable"]}
        rows = self.rows
        if window is not None and rows:
            inside = [r for r in rows if window[0] <= r[3] <= window[1]]
            if not inside:
                mid = 0.5 * (window[0] + window[1])
                inside = sorted(rows, key=lambda r: abs(r[3] - mid))[:2]
            rows = inside
        sm = [r[0] for r in rows]
        mx = [r[1] for r in rows]
        reasons = sorted({nm for r in rows for nm in r[2]})
        # under load = samples in the upper half of what was seen (idle samples at the edges are dropped)
        load = [v for v in sm if v >= 0.5 * max(sm)] if sm else []
        return {"sm_mhz": statistics.median(load) if load else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm), "source": src}


# ------------------------------------------------------------------------------------------------------------------
# the CPU oracle legs (cpu_baseline, --impl reference): the only places bench.py executes oracle/
# ------------------------------------------------------------------------------------------------------------------
def oracle_sample_time(w: W.MoEWorkload, n_res: int, sample_tokens: int, reps: int = 1):
    """Times the f32 oracle, as it stands, on the first `sample_tokens` tokens of the workload (same weights)."""
    from oracle.oracle import Oracle
    o = Oracle("f32")
    ws = w.with_(T=sample_tokens)
    S = W.resident_set(w, n_res)
    x, dy = W.make_x(w)[:sample_tokens].copy(), W.make_dy(w)[:sample_tokens].copy()
    w_r, bias = W.make_router(w), W.router_bias(w)
    wg, wu, wd = W.make_resident_experts(w, S)
    shared = W.make_shared_experts(w)
    times = []
    for _ in range(reps):
        t0 = time.perf_counter()
        r = o.route(x, w_r, S, ws.k, ws.gate_fn, ws.gate_rule, ws.temperature, bias)
        o.moe_fwd(x, r, S, wg, wu, wd, shared, expert_fn=ws.expert_fn)
        o.moe_bwd(x, dy, w_r, r, S, wg, wu, wd, shared, ws.gate_fn, ws.gate_rule, ws.temperature, expert_fn=ws.expert_fn)
        times.append(time.perf_counter() - t0)
    return times, o.threads()


def sized_sample(w, n_res, target_s: float, cap_tokens: int) -> int:
    """Tokens of the workload the oracle gets through in about `target_s` seconds on this box: a 64-token probe, then scale."""
    probe = min(w.T, 64)
    times, _ = oracle_sample_time(w, n_res, probe)
    rate = probe / max(times[0], 1e-6)
    n = int(rate * target_s)
    n = max(64, min(cap_tokens, w.T, (n // 64) * 64 if n >= 64 else 64))
    return n


def run_reference(args, w, n_res):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    # every step is a bounded sample of the workload, sized so that the whole run ends within a few minutes
    per_step_s = max(0.5, min(15.0, 150.0 / max(1, args.steps + args.warmup)))
    sample = sized_sample(w, n_res, per_step_s, args.ref_tokens)
    times, cores = oracle_sample_time(w, n_res, sample, reps=args.warmup + args.steps)
    timed = times[args.warmup:]
    ms = 1e3 * sum(timed) / len(timed)
    val = sample / (ms / 1e3)
    sample_desc = f"first {sample} of {w.T} tokens per step, all {n_res} resident experts' weights, route+fwd+bwd, f32 oracle"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic", "config": {"workload": workload_desc(w, n_res), "sample": sample_desc},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample_desc},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}))


# ------------------------------------------------------------------------------------------------------------------
# GPU arm
# ------------------------------------------------------------------------------------------------------------------
def gemm_flops(mode: str, P: int, T: int, w: W.MoEWorkload, launches_per_step: float = 1.0) -> float:
    """Algorithmic flops of one launch: 2*rows*d*F per GEMM; FWD1 and DX are two GEMMs."""
    if "ROUTE" in mode:    # logits x W_r (the bf16 split of W_r multiplies the tensor work, not the algorithmic flops)
        return 2.0 * T * w.d * w.E
    if "router" in mode:   # dz W_r^T and x^T dz: 2*T*d*E each
        return 2.0 * T * w.d * w.E
    if mode.startswith("fine_gather_kernel"):   # fine_gemm.cu: F1 and DH are one GEMM over the kept rows, WG is both weight gradients
        return (4.0 if "<WG>" in mode else 2.0) * P * w.d * w.F
    shared = "shared" in mode
    rows, F = (T * w.n_sh, w.F_sh) if shared else (P, w.F)
    mult = 4 if (("FWD1" in mode and "FWD1S" not in mode) or ("DX" in mode and w.expert_fn == W.EXPERT_SWIGLU)) else 2
    if "WGRAD" in mode:   # one launch computes every weight gradient of the experts (dW_down, dW_gate, dW_up)
        per = 3 if w.expert_fn == W.EXPERT_SWIGLU else 2
        mult = 2 * per if (not shared or launches_per_step < 1.5) else 2
    return float(mult) * rows * w.d * F


L2_BYTES = 126e6   # B200 L2 (both dies); an input that fits and was just read by the previous kernel is served from it


def hbm_bytes(name: str, P: int, T: int, w: W.MoEWorkload):
    """(algorithmic bytes of one launch, note) for the bandwidth-bound kernels; None for the others.
    When the whole of x fits in L2 a kernel that re-reads it right after the router is served from L2, not HBM: those
    bytes are then left out (counting them gave 'bandwidths' above the HBM peak) and the note says so."""
    s = 2 if w.dtype == "bf16" else 4
    x_in_l2 = T * w.d * s <= 0.75 * L2_BYTES
    if "ROUTE" in name or name.startswith("route_kernel"):
        return T * w.d * s + T * w.E * 4 + T * w.k * 8, None
    if name.startswith("gather_rows"):
        return (P * w.d * s, "x served from L2: only the write counted") if x_in_l2 else (2 * P * w.d * s, None)
    if name.startswith("combine_kernel"):
        return (P + T * (2 if w.n_sh else 1)) * w.d * s, None
    if name.startswith("combine_bwd"):
        return 3 * P * w.d * s, None
    if name.startswith("scale_rows"):   # do = g dy without the <dy, o> dot (two-matrix expert: dgate comes out of the DH epilogue)
        return (P * w.d * s, "dy served from L2: only the write counted") if x_in_l2 else (2 * P * w.d * s, None)
    if name.startswith("dx_sum"):
        return (P + T * (2 + (1 if w.n_sh else 0))) * w.d * s, None
    return None


def run_gpu(args, w, n_res):
    import torch
    import torch.distributed as dist

    from paper_2606_19025_b200 import binding as B
    from paper_2606_19025_b200 import replicas
    from paper_2606_19025_b200.layer import SkipTokenMoE, pack_resident_deltas

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback); use --impl reference for the CPU oracle")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    B.lib()

    def build_layer(nr):
        S = W.resident_set(w, nr)
        wg, wu, wd = W.make_resident_experts(w, S)
        return SkipTokenMoE(w, S, W.make_router(w), wg, wu, wd, W.make_shared_experts(w), W.router_bias(w))

    layer = build_layer(n_res)
    x_np, dy_np = W.make_x(w), W.make_dy(w)
    x, dy = layer.to_dev(x_np), layer.to_dev(dy_np)
    flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")  # > 126 MB L2

    def barrier_all():
        replicas.barrier()
        torch.cuda.synchronize()

    window = [0.0, 0.0]   # perf_counter bounds of the most recent timed region

    def timed_steps(fn, steps, warmup, collective=False):
        """Per-step CUDA events on the launching stream; L2 flushed between steps, outside the event pairs.
        collective=True brackets the region with a barrier over all ranks (the headline measurement)."""
        barrier = barrier_all if collective else torch.cuda.synchronize
        for _ in range(warmup):
            fn()
        barrier()
        window[0] = time.perf_counter()
        evs = []
        for _ in range(steps):
            flush.zero_()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            fn()
            e1.record()
            evs.append((e0, e1))
        barrier()
        window[1] = time.perf_counter()
        return [a.elapsed_time(b) for a, b in evs]

    launches = [0]

    def step_eager():
        launches[0] = layer.step(x, dy)

    step = step_eager
    if not args.no_graph:   # launch-bound at this size: replay the step as one CUDA graph
        step_eager()
        step = layer.capture_step(x, dy)

    sampler = ClockSampler(local)
    sampler.start()
    ms_list = timed_steps(step, args.steps, args.warmup, collective=True)
    clocks = sampler.stop(tuple(window))
    ms = replicas.max_over_ranks(sum(ms_list) / len(ms_list), "cuda")
    value = replicas.whole_job_tokens_per_s(w.T, ms)

    routing = layer.routing_numpy()
    P = routing["P"]
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": w.dtype,
        "data": "synthetic",
        "config": {"workload": workload_desc(w, n_res), "parallelism": f"{world} independent replica(s), no collective",
                   "l2": "512 MiB flush write between timed steps (outside the per-step CUDA-event pairs)",
                   "timing": "per-step CUDA events on the launching stream, mean over steps, max over ranks",
                   "launch": "eager" if args.no_graph else "whole step replayed as one CUDA graph"},
        "clocks": clocks, "gpu_launches": launches[0] * args.steps,
        "kept_pairs": P, "kept_fraction": P / max(1, w.T * w.k), "ms_min": min(ms_list),
    }
    try:   # routing diagnostics: realised kept fraction, load CV, entropy, zero-kept-token fraction
        rs = layer.routing_stats()
        out["routing_stats"] = {k: (float(v) if not hasattr(v, "tolist") else None) for k, v in rs.items() if k != "load"}
        ld = rs["load"]
        out["routing_stats"]["load_min_max_all_experts"] = [int(ld.min()), int(ld.max())]
    except Exception as e:
        out["routing_stats"] = {"error": str(e)}
    fl_pair = 18.0 if w.expert_fn == W.EXPERT_SWIGLU else 12.0   # flops per (row, d, F): 3 (2) GEMMs forward, twice that backward
    flops_step = fl_pair * P * w.d * w.F + fl_pair * w.T * w.n_sh * w.d * w.F_sh
    out["tflops"] = flops_step / (ms / 1e3) / 1e12

    if rank == 0:
        peaks, peak_src = load_peaks()
        # the denominator follows the clock regime the timed region ran in: a short run stays at max clocks (burst peak),
        # a long one settles under the power cap (sustained peak)   [B200_PROFILING.md]
        burst = clocks.get("sm_mhz") is None or clocks["sm_mhz"] >= 0.9 * (clocks.get("sm_max_mhz") or 1965.0)
        tc_peak = peaks["bf16_tflops"] if burst else peaks["bf16_tflops_sustained"]
        tc_peak_name = "bf16 burst (SM clocks at max during the timed region)" if burst else "bf16 sustained (power-capped clocks)"
        # ---- per-kernel timing: a second pass of the same steps with one CUDA event after every launch ----
        B.fomoe_profile_enable(True)
        for _ in range(args.steps):
            flush.zero_()
            step_eager()
        recs = B.fomoe_profile_collect(65536)
        B.fomoe_profile_enable(False)
        agg = {}
        for name, t in recs:
            a = agg.setdefault(name, [0.0, 0])
            a[0] += t
            a[1] += 1
        total = sum(a[0] for a in agg.values())
        kernels = []
        for name, (tt, n) in sorted(agg.items(), key=lambda kv: -kv[1][0]):
            k = {"name": name, "launches_per_step": n / args.steps, "ms_per_launch": tt / n, "share": tt / total}
            hbn = hbm_bytes(name, P, w.T, w)
            if hbn is not None:
                hb, note = hbn
                k.update(bound="hbm", achieved=hb / (tt / n / 1e3) / 1e9, unit="GB/s")
                if note:
                    k["note"] = note
                k["frac"] = k["achieved"] / peaks["hbm_gbs"]
                k["frac_of_nominal_8000"] = k["achieved"] / 8000.0
            elif name.startswith("umma_grouped_kernel") or name.startswith("fine_gather_kernel"):
                fl = gemm_flops(name, P, w.T, w, n / args.steps)
                k.update(bound="tensor", achieved=fl / (tt / n / 1e3) / 1e12, unit="TFLOP/s")
                k["frac"] = k["achieved"] / tc_peak
                if name.startswith("fine_gather_kernel"):
                    # these are bound by the L2 -> SM path, not by the tensor pipe: operand bytes a launch pulls out of L2
                    # (gathered rows + the dense operand, fetched once per 256 gathered rows / per 256-column block)
                    # against the 6300 B/clk the L2 delivers at best (B300_MICROARCH.md "TMA chip-throughput") at the sampled clock
                    ob = (3.0 if "<WG>" in name else 1.5) * P * w.d * 2
                    k["l2_operand_bytes"] = ob
                    k["l2_gbs"] = ob / (tt / n / 1e3) / 1e9
                    k["l2_frac_of_6300B_per_clk"] = k["l2_gbs"] / (6300 * (clocks.get("sm_mhz") or 1965.0) * 1e6 / 1e9)
                if name in ("umma_grouped_kernel<FWD2>", "umma_grouped_kernel<DX>"):
                    # with narrow experts these two are write streams of their [P, d] output, not contractions: report that rate
                    # too (compare with hbm_write_probe below: what a plain memset reaches on this GPU)
                    k["out_write_gbs"] = P * w.d * 2 / (tt / n / 1e3) / 1e9
            kernels.append(k)
        out["kernels"] = kernels
        # a pure-write stream for comparison: cudaMemset of the 512 MiB flush buffer, timed live
        for _ in range(3):
            flush.zero_()
        torch.cuda.synchronize()
        w0, w1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        w0.record()
        for _ in range(5):
            flush.zero_()
        w1.record()
        torch.cuda.synchronize()
        out["hbm_write_probe"] = {"memset_gbs": 5 * flush.numel() / (w0.elapsed_time(w1) / 1e3) / 1e9, "bytes": flush.numel(),
                                  "note": "pure-write rate of cudaMemset; the copy peak in MEASURED_PEAKS.json is read + write"}
        # DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum) from the committed `ncu --set full` capture of
        # THIS revision's kernels (profiles/r2_traffic.md names the command); keyed by workload and by the name the library emits
        traffic_rows = {}
        tf = ROOT / "profiles" / "r2_traffic.csv"
        if tf.exists():
            for line in tf.read_text().splitlines()[1:]:
                if not line.strip():
                    continue
                wl, rest = line.split(",", 1)          # kernel names contain commas: workload,kernel,bytes,launches
                kname, nbytes, _ = rest.rsplit(",", 2)
                traffic_rows[(wl, kname)] = float(nbytes)
        gemms = [k for k in kernels if k.get("bound") == "tensor" and "router" not in k["name"] and "ROUTE" not in k["name"]]
        if gemms:
            def roof(kk):
                return {"kernel": kk["name"], "bound": "tensor", "achieved": kk["achieved"], "peak": tc_peak, "unit": "TFLOP/s",
                        "frac": kk["frac"], "traffic": traffic_rows.get((w.name, kk["name"])),
                        "peak_source": peak_src + ", " + tc_peak_name, "frac_of_nominal_2250": kk["achieved"] / 2250.0,
                        "share_of_step": kk["share"], "ms_per_launch": kk["ms_per_launch"],
                        "kernel_timing": "second pass of the same steps with one CUDA event after every launch"}
            out["roofline"] = roof(gemms[0])                                   # the GEMM with the largest share of the step
            out["roofline_worst"] = roof(min(gemms, key=lambda kk: kk["frac"]))  # the GEMM furthest below the peak
            gt = sum(k["ms_per_launch"] * k["launches_per_step"] for k in gemms)
            out["gemm_family"] = {"tflops": flops_step / (gt / 1e3) / 1e12, "share_of_step": gt * args.steps / total,
                                  "frac_of_peak": flops_step / (gt / 1e3) / 1e12 / tc_peak,
                                  "frac_of_nominal_2250": flops_step / (gt / 1e3) / 1e12 / 2250.0}
        hbms = [k for k in kernels if k.get("bound") == "hbm"]
        if hbms:
            out["hbm_kernels"] = {k["name"]: round(k["frac"], 3) for k in hbms}
        # ---- the routing call timed ALONE (fomoe_route only, L2 flushed before every call, after a pause that lets the SM clock
        # recover): inside a long power-capped step the router runs at the GEMMs' reduced SM clock, and it is bound on the SM side
        # (L2 -> SM operand delivery), so kernels[] above understates what the kernel does at full clock; this is
        # the "kernel timed alone against the burst peak" form of the same number ----
        time.sleep(1.0)
        B.fomoe_profile_enable(True)
        sampler2 = ClockSampler(local)
        sampler2.start()
        w_t0 = time.perf_counter()
        for _ in range(max(50, args.steps)):
            flush.zero_()
            layer.route(x)
        torch.cuda.synchronize()
        w_t1 = time.perf_counter()
        rclk = sampler2.stop((w_t0, w_t1))
        rrecs = B.fomoe_profile_collect(65536)
        B.fomoe_profile_enable(False)
        ralone = {}
        for name, t in rrecs:
            a = ralone.setdefault(name, [0.0, 0])
            a[0] += t
            a[1] += 1
        out["route_alone"] = {"clocks": rclk, "kernels": []}
        for name, (tt, n) in ralone.items():
            kk = {"name": name, "ms_per_launch": tt / n}
            hbn = hbm_bytes(name, P, w.T, w)
            if hbn is not None:
                kk.update(bound="hbm", achieved=hbn[0] / (tt / n / 1e3) / 1e9, unit="GB/s", peak=peaks["hbm_gbs"])
                kk["frac"] = kk["achieved"] / peaks["hbm_gbs"]
            out["route_alone"]["kernels"].append(kk)

        # ---- end to end through the C ABI with HOST buffers (uploads x, dy; downloads y, dx every step).  Two arms:
        # "serial": one self-contained call per step (results complete when the stream is);  headline e2e: the same call with
        # alternating staging buffers and the join deferred, so that step i's kernels, step i+1's uploads and step i-1's dx
        # download run at the same time -- timed by ONE CUDA-event pair around the K steps, the end event after the join ----
        xh, dyh = x.cpu().pin_memory(), dy.cpu().pin_memory()
        yh, dxh = torch.empty_like(xh).pin_memory(), torch.empty_like(xh).pin_memory()
        stage = [(torch.empty_like(x), torch.empty_like(dy)) for _ in range(2)]
        cs = torch.cuda.Stream()
        ser_ms = timed_steps(lambda: layer.step_host(xh, dyh, yh, dxh, *stage[0], copy_stream=cs), max(3, args.steps // 2), 2)
        ser = sum(ser_ms) / len(ser_ms)
        for i in range(args.warmup):
            layer.step_host(xh, dyh, yh, dxh, *stage[i % 2], copy_stream=cs, defer_join=True)
        layer.host_join()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for i in range(args.steps):
            layer.step_host(xh, dyh, yh, dxh, *stage[i % 2], copy_stream=cs, defer_join=True)
        layer.host_join()
        e1.record()
        torch.cuda.synchronize()
        e2e = e0.elapsed_time(e1) / args.steps
        nbytes = xh.numel() * xh.element_size()
        out["e2e"] = {"value": world * w.T / (e2e / 1e3), "unit": UNIT, "h2d_bytes_per_step": 2 * nbytes,
                      "d2h_bytes_per_step": 2 * nbytes, "ms_per_step": e2e,
                      "api": "fomoe_moe_step_host(defer_join=1) x K + fomoe_moe_step_host_join: pinned host x, dy -> y, dx every step, "
                             "two alternating device staging pairs; uploads, kernels and downloads on three streams",
                      "timing": "one CUDA-event pair around the K steps (end event after the join); inputs arrive over PCIe, so no L2 flush",
                      "serial_ms_per_step": ser, "serial_value": world * w.T / (ser / 1e3),
                      "pcie_floor_ms": 2 * nbytes / 55e9 * 1e3}
        del stage

        # ---- resident-delta pack (row S1), HBM bound: 12 B per parameter ----
        S = W.resident_set(w, n_res)
        now = [torch.from_numpy(np.stack(t)).cuda() for t in zip(*(W.make_expert_master(w, int(e)) for e in S))]
        if w.expert_fn == W.EXPERT_SILU:   # the paper's expert payload is up + down: no gate block
            now[0] = now[0][:, :0].contiguous()
        start = [t + 1e-3 * torch.randn_like(t) for t in now]
        payload = torch.empty((n_res, sum(int(t[0].numel()) for t in now)), dtype=torch.float32, device="cuda")
        pk = timed_steps(lambda: pack_resident_deltas(now, start, None, payload), max(args.steps, 10), 3)
        pbytes = 12.0 * payload.numel()
        pms = sum(pk) / len(pk)
        out["pack"] = {"bound": "hbm", "achieved": pbytes / (pms / 1e3) / 1e9, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                       "frac": pbytes / (pms / 1e3) / 1e9 / peaks["hbm_gbs"], "ms": pms, "bytes": pbytes,
                       "frac_of_nominal_8000": pbytes / (pms / 1e3) / 1e9 / 8000.0}
        # ---- the optimizer steps on either side of the pack: fused local AdamW over the resident
        # experts and the outer Nesterov step that consumes the averaged payload ----
        try:
            gdt = torch.bfloat16 if w.dtype == "bf16" else torch.float32
            gs = gdt.itemsize if hasattr(gdt, "itemsize") else (2 if w.dtype == "bf16" else 4)
            grads = [(1e-3 * torch.randn_like(t)).to(gdt) for t in now]
            m1 = [torch.zeros_like(t) for t in now]
            v1 = [torch.zeros_like(t) for t in now]
            wc = [torch.empty_like(t, dtype=gdt) for t in now]
            nparam = float(sum(t.numel() for t in now))
            at = timed_steps(lambda: B.fomoe_adamw_resident(now, grads, m1, v1, wc, 1, 0.0131), max(args.steps, 10), 3)
            ams = sum(at) / len(at)
            abytes = nparam * (24.0 + 2.0 * gs)          # read w, m, v (fp32) + g; write w, m, v + the compute-dtype copy
            buf = m1                                     # reuse as the outer momentum buffers
            ot = timed_steps(lambda: B.fomoe_outer_nesterov(start, now, buf, wc, payload), max(args.steps, 10), 3)
            oms = sum(ot) / len(ot)
            obytes = nparam * (24.0 + gs)                # read delta, buf, w_start; write buf, w_start, w_now + the copy
            out["optim"] = {"adamw": {"bound": "hbm", "achieved": abytes / (ams / 1e3) / 1e9, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                                      "frac": abytes / (ams / 1e3) / 1e9 / peaks["hbm_gbs"], "ms": ams, "bytes": abytes},
                            "outer_nesterov": {"bound": "hbm", "achieved": obytes / (oms / 1e3) / 1e9, "peak": peaks["hbm_gbs"],
                                               "unit": "GB/s", "frac": obytes / (oms / 1e3) / 1e9 / peaks["hbm_gbs"], "ms": oms,
                                               "bytes": obytes}}
            del grads, m1, v1, wc
        except Exception as e:   # never let the side measurements take the headline down
            out["optim"] = {"error": str(e)}
        # ---- Peri-LN either side of the block (Eq. 15): the stand-alone streaming kernels
        # against the HBM roofline, and the whole block x + alpha LN(MoE(LN(x))) fused (post-LN inside the combine, pre-LN backward
        # inside the dx scatter-sum) and unfused, in units of one pass over [T, d] beyond the MoE step ----
        try:
            gam, bet = torch.ones(w.d, device="cuda"), torch.zeros(w.d, device="cuda")
            stats, stats2 = (torch.empty((w.T, 2), dtype=torch.float32, device="cuda") for _ in range(2))
            lo, ldx, xn, dyy = (torch.empty_like(x) for _ in range(4))
            dgm, dbt = torch.empty(w.d, device="cuda"), torch.empty(w.d, device="cuda")
            part = torch.empty(B.fomoe_periln_workspace_bytes(w.T, w.d), dtype=torch.uint8, device="cuda")
            es = x.element_size()
            n10 = max(args.steps, 10)
            ft = timed_steps(lambda: B.fomoe_periln_fwd(x, gam, bet, lo, stats, residual=dy, alpha=0.8), n10, 3)
            bt = timed_steps(lambda: B.fomoe_periln_bwd(dy, x, stats, gam, ldx, dgm, dbt, part, dresidual=dy, alpha=0.8), n10, 3)
            fms, bms = sum(ft) / len(ft), sum(bt) / len(bt)
            fby, bby = 3.0 * w.T * w.d * es, 4.0 * w.T * w.d * es       # post-LN + residual: read y, x, write out; bwd: read dout, x, dres, write dx
            pl = {"post_fwd": {"bound": "hbm", "achieved": fby / (fms / 1e3) / 1e9, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                               "frac": fby / (fms / 1e3) / 1e9 / peaks["hbm_gbs"], "ms": fms, "bytes": fby},
                  "pre_bwd": {"bound": "hbm", "achieved": bby / (bms / 1e3) / 1e9, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                              "frac": bby / (bms / 1e3) / 1e9 / peaks["hbm_gbs"], "ms": bms, "bytes": bby}}

            def block(fused):
                B.fomoe_periln_fwd(x, gam, bet, xn, stats)                                  # pre-LN
                layer.route(xn)
                if fused:
                    layer.forward_periln(xn, gam, bet, x, lo, stats2, alpha=0.8)            # MoE + post-LN + residual
                else:
                    layer.forward(xn)
                    B.fomoe_periln_fwd(layer.y, gam, bet, lo, stats2, residual=x, alpha=0.8)
                B.fomoe_periln_bwd(dy, layer.y, stats2, gam, dyy, dgm, dbt, part, alpha=0.8)  # post-LN backward -> dy of the layer
                if fused:
                    layer.backward_periln(dyy, xn, x, stats, gam, dy, dgm, dbt, part)       # MoE backward + pre-LN backward + residual
                else:
                    layer.backward(dyy, xn)
                    B.fomoe_periln_bwd(layer.dx, x, stats, gam, ldx, dgm, dbt, part, dresidual=dy)
            if B.fomoe_periln_fused_supported(layer.cfg):
                pass_ms = 2.0 * w.T * w.d * es / (peaks["hbm_gbs"] * 1e9) * 1e3    # read + write of [T, d] at the measured copy rate
                step_ms = sum(timed_steps(step_eager, n10, 3)) / n10
                tf_ = sum(timed_steps(lambda: block(True), n10, 3)) / n10
                tu_ = sum(timed_steps(lambda: block(False), n10, 3)) / n10
                pl["block"] = {"ms_moe_step_eager": step_ms, "ms_block_fused": tf_, "ms_block_unfused": tu_,
                               "extra_passes_fused": (tf_ - step_ms) / pass_ms, "extra_passes_unfused": (tu_ - step_ms) / pass_ms,
                               "pass_ms": pass_ms, "launch": "eager (all three arms)"}
            out["periln"] = pl
            del lo, ldx, xn, dyy, part
        except Exception as e:
            out["periln"] = {"error": str(e)}
        del now, start, payload

        # ---- skip-token speed-up against the same kernels with every expert resident: both arms replay a CUDA graph, both
        # are timed by the same loop, and both report the clocks sampled inside their own timed region ----
        if not args.no_all_resident and n_res < w.E:
            del layer, step
            torch.cuda.empty_cache()
            full = build_layer(w.E)
            full_step = full.step
            if not args.no_graph:
                full.step(x, dy)
                full_step = full.capture_step(x, dy)
            else:
                full_step = lambda: full.step(x, dy)  # noqa: E731
            s2 = ClockSampler(local)
            s2.start()
            ms_full = timed_steps(full_step, args.steps, args.warmup)
            clocks_full = s2.stop(tuple(window))
            mf = sum(ms_full) / len(ms_full)
            ideal = (w.k * fl_pair * w.d * w.F * w.T + fl_pair * w.T * w.n_sh * w.d * w.F_sh) / flops_step
            sk = {"ms_all_resident": mf, "speedup_vs_all_resident": mf / ms, "ideal_flop_ratio": ideal,
                  "launch_all_resident": "eager" if args.no_graph else "CUDA graph (same as the skip arm)",
                  "sm_mhz_skip_arm": clocks.get("sm_mhz"), "sm_mhz_all_resident": clocks_full.get("sm_mhz"),
                  "reasons_all_resident": clocks_full.get("reasons")}
            sk["tflops_all_resident"] = (w.k * fl_pair * w.d * w.F * w.T + fl_pair * w.T * w.n_sh * w.d * w.F_sh) / (mf / 1e3) / 1e12
            sk["tflops_skip_arm"] = out["tflops"]
            if mf / ms > ideal:   # a speed-up above the FLOP ratio means the all-resident arm ran less efficiently: say why
                a, b = clocks.get("sm_mhz"), clocks_full.get("sm_mhz")
                sk["above_ideal_because"] = (
                    f"the longer all-resident step settles under the power cap (NVML: {b} MHz, reasons {clocks_full.get('reasons')}) while "
                    f"the short skip arm samples {a} MHz: the arms do not run at the same clock, so the ratio overstates the kernels' "
                    f"share of the gain; per-arm TFLOP/s: {sk['tflops_all_resident']:.0f} (all resident) vs {out['tflops']:.0f} (skip)"
                    if a and b and b < 0.98 * a else
                    f"not a clock effect ({b} vs {a} MHz): the all-resident arm reached {sk['tflops_all_resident']:.0f} TFLOP/s "
                    f"against {out['tflops']:.0f} for the skip arm on the same kernels (its larger routed share runs the less "
                    f"efficient routed GEMMs and row kernels)")
            out["skip_token"] = sk
            del full, full_step

        # ---- Fig. 11 analogue: step time against the number of ghost (non-resident) experts ----
        if args.ghost_sweep:
            try:
                del layer, step
            except NameError:
                pass
            torch.cuda.empty_cache()
            sweep = []
            base_ms = None
            for nr in sorted({w.E, (3 * w.E) // 4, w.E // 2, w.E // 4, w.E // 8}, reverse=True):
                if nr < 1:
                    continue
                lay = build_layer(nr)
                lay.step(x, dy)
                st = lay.capture_step(x, dy)
                t_ms = timed_steps(st, args.steps, args.warmup)
                m = sum(t_ms) / len(t_ms)
                base_ms = m if base_ms is None else base_ms
                sweep.append({"n_res": nr, "ghost_experts": w.E - nr, "ms_per_step": m, "kept_pairs": lay.routing_numpy()["P"],
                              "speedup_vs_all_resident": base_ms / m})
                del lay, st
                torch.cuda.empty_cache()
            out["ghost_sweep"] = sweep

        # ---- the oracle, as it stands, on the host cores (reported baseline, not the target) ----
        if not args.no_cpu_baseline:
            sample = sized_sample(w, n_res, 30.0, args.ref_tokens)     # 10-30 s of CPU work (the probe over-estimates the rate a little)
            times, cores = oracle_sample_time(w, n_res, sample)
            out["cpu_baseline"] = {"value": sample / times[0], "unit": UNIT, "cores": cores, "kind": "oracle",
                                   "sample": f"first {sample} of {w.T} tokens, all {n_res} resident experts' weights, "
                                             f"route+fwd+bwd, f32 oracle, 1 repetition, {times[0]:.1f} s"}
        print(json.dumps(out))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C5", choices=sorted(W.CONFIGS),
                    help="C5 (BASELINE.json configs[4]) is the largest single-GPU configuration: the headline")
    ap.add_argument("--n-res", type=int, default=None)
    ap.add_argument("--tokens", type=int, default=None, help="override the workload's token count T (scaling experiments)")
    ap.add_argument("--ref-tokens", type=int, default=16384, help="upper bound on the tokens per step of the CPU oracle sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-all-resident", action="store_true")
    ap.add_argument("--ghost-sweep", action="store_true", help="also time the step for n_res = E, 3E/4, E/2, E/4, E/8 (Fig. 11 analogue)")
    ap.add_argument("--no-graph", action="store_true", help="launch kernels eagerly instead of replaying a CUDA graph")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # not launched by torchrun: start one process per GPU ourselves (the driver's launch line, see the module docstring)
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
               "--master-port", str(29500 + os.getpid() % 2000), str(Path(__file__).resolve()), *sys.argv[1:]]
        raise SystemExit(subprocess.call(cmd))
    w = W.config(args.workload)
    if args.tokens is not None:
        w = dataclasses.replace(w, T=args.tokens, name=f"{w.name}@T={args.tokens}")
    n_res = w.n_res if args.n_res is None else args.n_res
    if args.impl == "reference":
        run_reference(args, w, n_res)
    else:
        run_gpu(args, w, n_res)


if __name__ == "__main__":
    main()
