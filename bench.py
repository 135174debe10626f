#!/usr/bin/env python
"""bench.py -- X-engine throughput on B200 (BASELINE.json metric: Tops/s at 8 ops per complex MAC).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg2] [--impl reference]

A "step" is one pass of the whole hot path (S0-S3 of SURVEY 8(a): staging if needed, tile schedule,
tcgen05 X-engine, packing epilogue) over one synthetic input block through the C-ABI library.
Default workload = BASELINE.json configs[1] (N=128, F=1024, T=1000).  Prints ONE JSON line.

  value        whole-job Tops/s, inputs resident in HBM (ops = 8 * F * T * N(2N+1), Eq. 5)
  e2e          same metric through xc_correlate_host with HOST buffers (H2D + X-engine + D2H per step)
  roofline     dominant kernel against the measured HBM / int8-tensor peak (MEASURED_PEAKS.json)
  cpu_baseline the oracle (oracle/xo_oracle.c, as it stands) on the box's host cores, bounded sample
  by_config    kernel-only Tops/s for the other BASELINE configs (the metric is "vs N stations")

N > 1 (torchrun): every rank runs its own block of F channels (channels are independent, PAPER.md:65,
285): no data-path collective, "scaling": "weak"; time = max over ranks.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

NOMINAL_I8_OVER_BF16 = 2.0          # 4.5 / 2.25 PFLOP/s dense (B200_PROFILING.md nominal table)
FALLBACK_HBM_GBS, FALLBACK_BF16_TF = 6650.0, 1590.0


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as fh:
            m = json.load(fh)
        return {"hbm_gbs": float(m["hbm_gbs"]), "bf16_burst": float(m["bf16_tflops"]),
                "bf16_sustained": float(m.get("bf16_tflops_sustained", m["bf16_tflops"])), "source": "measured"}
    return {"hbm_gbs": FALLBACK_HBM_GBS, "bf16_burst": FALLBACK_BF16_TF, "bf16_sustained": 1400.0,
            "source": "fallback"}


class ClockSampler:
    """SM clock and throttle reasons sampled through NVML (pynvml) every ~1 ms by a thread, DURING the
    timed region (the recipe's clocks line, without nvidia-smi's start-up latency)."""
    REASONS = {"hw_slowdown": 0x8, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20, "sw_power_cap": 0x4}

    def __init__(self, index: int):
        self.rows, self.ok, self._stop = [], False, False
        try:
            import pynvml
            pynvml.nvmlInit()
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            phys = int(vis.split(",")[index]) if vis and vis.split(",")[index].isdigit() else index
            self.nv, self.h = pynvml, pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.max_sm = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
            self.thr = threading.Thread(target=self._run, daemon=True)
            self.thr.start()
        except Exception as e:  # noqa: BLE001 -- report, never fail the bench for a missing NVML
            self.err = repr(e)

    def _run(self):
        nv, h = self.nv, self.h
        while not self._stop:
            try:
                sm = nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM)
                try:
                    rs = nv.nvmlDeviceGetCurrentClocksEventReasons(h)
                except AttributeError:
                    rs = nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                pw = nv.nvmlDeviceGetPowerUsage(h) / 1000.0
                self.rows.append((time.perf_counter(), float(sm), int(rs), pw))
            except Exception:  # noqa: BLE001
                pass
            time.sleep(0.001)

    def window(self, t0, t1):
        if not self.ok:
            return {"sm_mhz": None, "sm_max_mhz": None, "samples": 0, "reasons": [], "error": getattr(self, "err", "")}
        rows = [r for r in self.rows if t0 <= r[0] <= t1]
        where = "timed region"
        if not rows:  # region shorter than one sampling period: take the samples right after it
            rows = [r for r in self.rows if t1 < r[0] <= t1 + 0.02][:3]
            where = "first samples after the timed region (region shorter than the sampling period)"
        sm = sorted(r[1] for r in rows)
        bits = 0
        for r in rows:
            bits |= r[2]
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": self.max_sm, "samples": len(sm),
                "power_w_max": max((r[3] for r in rows), default=None),
                "reasons": sorted(n for n, b in self.REASONS.items() if bits & b), "window": where}

    def stop(self):
        self._stop = True


def workload_desc(w):
    return (f"{w.name}: N={w.N} stations x 2 pol, F={w.F} channels, T={w.T} samples, int8 {w.kind} "
            f"sigma={w.sigma}, seed {w.seed}, layout [t][f][station][pol][re,im]")


def cpu_sample(w, x, target_s=12.0):
    """Oracle on a bounded sample of channels of the same workload; returns (Tops/s, cores, text)."""
    from oracle import xo
    cores = xo.num_threads()
    per_ch = w.T * w.N * (2 * w.N + 1)
    t0 = time.perf_counter()
    xo.channels_i8(x, list(range(min(cores, w.F))))
    dt = time.perf_counter() - t0
    n0 = min(cores, w.F)
    rate = n0 * per_ch / dt
    nsel = int(max(n0, min(w.F, (target_s * rate / per_ch) // cores * cores)))
    t0 = time.perf_counter()
    xo.channels_i8(x, list(range(nsel)))
    dt = time.perf_counter() - t0
    tops = 8.0 * nsel * per_ch / dt / 1e12
    return tops, cores, f"{nsel} of {w.F} channels of {w.name}, all baselines, {dt:.1f} s"


def run_reference(args, rank):
    """--impl reference: the CPU oracle as it stands, on the host cores (rank 0 only)."""
    if rank != 0:
        return
    import xc_workloads as wl
    from oracle import xo
    w = wl.CONFIGS[args.workload]
    cores = xo.num_threads()
    per_ch = w.T * w.N * (2 * w.N + 1)
    # a step = `nch` channels of the workload (bounded sample; channels are independent)
    nch = max(1, min(w.F, cores))
    sub = wl.Workload(w.name, w.N, nch, w.T, w.kind, w.sigma, w.seed)
    x = wl.make_input(sub)
    sel = list(range(nch))
    for _ in range(args.warmup):
        xo.channels_i8(x, sel)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        xo.channels_i8(x, sel)
    dt = time.perf_counter() - t0
    tops = 8.0 * args.steps * nch * per_ch / dt / 1e12
    sample = f"{nch} of {w.F} channels of {w.name} per step, all baselines"
    print(json.dumps({
        "impl": "reference", "metric": "X-engine Tops/s (8 ops per cMAC)", "value": tops, "unit": "Tops/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "int8", "data": "synthetic",
        "config": {"workload": workload_desc(w), "sample": sample},
        "cpu_baseline": {"value": tops, "unit": "Tops/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": tops, "unit": "Tops/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def time_kernel(p, xd, vis, stream, steps, warmup):
    """Per-launch durations (ms) with CUDA events on the launching stream."""
    import torch
    with torch.cuda.stream(stream):
        for _ in range(warmup):
            p.correlate(xd, vis, stream=stream)
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        stream.synchronize()
        for a, b in evs:
            a.record(stream)
            p.correlate(xd, vis, stream=stream)
            b.record(stream)
        stream.synchronize()
    return [a.elapsed_time(b) for a, b in evs]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="cfg2")
    ap.add_argument("--impl", default="native", choices=["native", "reference"])
    ap.add_argument("--no-sweep", action="store_true", help="skip the by_config sweep")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--f32-only", type=int, default=0, metavar="F",
                    help="profiling aid: run only xc_correlate_f32 on config 3's values cut to F channels, 4 launches")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "native" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    if args.impl == "reference":
        run_reference(args, rank)
        return

    import numpy as np
    import torch
    import torch.distributed as dist

    import paper_1107_4264_b200 as xcb
    import xc_workloads as wl
    from paper_1107_4264_b200 import build as xc_build

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the X-engine has no CPU path")
    if rank == 0:
        xc_build.build()
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
        dist.barrier()
    xcb.load_library()

    if args.f32_only:
        w3 = wl.CONFIGS["cfg3"]
        sub = wl.Workload("cfg3_f32", w3.N, args.f32_only, w3.T, w3.kind, w3.sigma, w3.seed)
        x3 = torch.from_numpy(wl.make_input(sub)).cuda().to(torch.float32)
        p3 = xcb.Plan(sub.N, sub.F, sub.T)
        v3 = p3.new_vis(torch.float32)
        e = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        p3.correlate_f32(x3, v3)
        e[0].record()
        for _ in range(3):
            p3.correlate_f32(x3, v3)
        e[1].record()
        torch.cuda.synchronize()
        ms = e[0].elapsed_time(e[1]) / 3
        print(json.dumps({"f32_only": True, "N": sub.N, "F": sub.F, "T": sub.T, "kernel_ms": ms,
                          "tflops": sub.ops / (ms * 1e-3) / 1e12}))
        return

    peaks = load_peaks()
    w = wl.CONFIGS[args.workload]
    # weak scaling: every rank holds its own block of F channels (seed differs per rank)
    x_np = wl.make_input(w, seed=w.seed + 7919 * rank)
    p = xcb.Plan(w.N, w.F, w.T)
    stream = torch.cuda.Stream()
    xh = torch.from_numpy(x_np).pin_memory()
    xd = xh.cuda()
    vis = p.new_vis()
    torch.cuda.synchronize()

    # ---- device-resident timing: exactly K steps between barrier + synchronize ----------------
    sampler = ClockSampler(torch.cuda.current_device())
    with torch.cuda.stream(stream):
        for _ in range(args.warmup):
            p.correlate(xd, vis, stream=stream)
    launches_per_step = p.last_launches
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    t_wall0 = time.perf_counter()
    with torch.cuda.stream(stream):
        e0.record(stream)
        for _ in range(args.steps):
            p.correlate(xd, vis, stream=stream)
        e1.record(stream)
    torch.cuda.synchronize()
    t_wall1 = time.perf_counter()
    ms_total = e0.elapsed_time(e1)
    if world > 1:
        t = torch.tensor([ms_total], device="cuda", dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_total = float(t.item())
        dist.barrier()
    clocks = sampler.window(t_wall0, t_wall1)
    ms_step = ms_total / args.steps
    tops = world * w.ops / (ms_step * 1e-3) / 1e12

    # ---- per-launch duration of the dominant kernel (events around each launch) -------------
    per = time_kernel(p, xd, vis, stream, min(args.steps, 50), 1)
    k_ms = sum(per) / len(per)
    alg_bytes = w.in_bytes + w.vis_bytes                      # input once + output once
    i8_peak = peaks["bf16_burst"] * NOMINAL_I8_OVER_BF16      # Tops/s: measured bf16 x nominal int8/bf16 ratio
    t_hbm = alg_bytes / (peaks["hbm_gbs"] * 1e9)
    t_tc = w.ops / (i8_peak * 1e12)
    traffic = TRAFFIC_NCU.get(w.name)
    if t_hbm >= t_tc:
        ach = alg_bytes / (k_ms * 1e-3) / 1e9
        roof = {"bound": "hbm", "achieved": ach, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                "frac": ach / peaks["hbm_gbs"], "traffic": traffic}
    else:
        ach = w.ops / (k_ms * 1e-3) / 1e12
        roof = {"bound": "tensor", "achieved": ach, "peak": i8_peak, "unit": "Tops/s", "frac": ach / i8_peak,
                "traffic": traffic}
    roof.update({"kernel": "xc_i8_tc_kernel", "kernel_ms": k_ms, "peak_source": peaks["source"] +
                 (" hbm_gbs" if roof["bound"] == "hbm" else " bf16_tflops (burst) x 2 (nominal int8/bf16)"),
                 "algorithmic_bytes": alg_bytes, "algorithmic_ops": w.ops,
                 "other_roof_frac": (w.ops / (k_ms * 1e-3) / 1e12 / i8_peak) if roof["bound"] == "hbm"
                 else (alg_bytes / (k_ms * 1e-3) / 1e9 / peaks["hbm_gbs"])})

    # ---- the SM clock the kernel REALLY ran at: CTA 0 stamps (clock64, globaltimer) at start and end ----------
    # (NVML keeps reporting clocks.max.sm while the chip's power management already runs the tensor-heavy kernel
    # slower; measured 1.2-1.6 GHz.  Reported beside the NVML figures, which stay in the contract's keys.)
    probe = torch.zeros(xcb.TRACE_WORDS, dtype=torch.int64, device="cuda")
    p.set_trace(probe)
    mhz = []
    with torch.cuda.stream(stream):
        for _ in range(20):
            p.correlate(xd, vis, stream=stream)
            stream.synchronize()
            t4 = probe[-4:].tolist()
            if t4[3] > t4[1]:
                mhz.append((t4[2] - t4[0]) / (t4[3] - t4[1]) * 1e3)
    p.set_trace(None)
    mhz.sort()
    clocks["sm_mhz_in_kernel"] = mhz[len(mhz) // 2] if mhz else None
    clocks["sm_mhz_in_kernel_how"] = ("clock64 / globaltimer stamped by CTA 0 of xc_i8_tc_kernel at its start and end, "
                                      "median of 20 back-to-back launches after the timed region")

    # ---- end to end through the C ABI with HOST buffers ---------------------------------------
    vh = torch.empty(p.vis_shape(), dtype=torch.int32).pin_memory()
    e2e_steps = max(3, min(args.steps, 10))
    p.correlate_host(xh, vh, xd, vis, stream=stream)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        p.correlate_host(xh, vh, xd, vis, stream=stream)       # synchronises the stream itself
    e2e_s = (time.perf_counter() - t0) / e2e_steps
    if world > 1:
        t = torch.tensor([e2e_s], device="cuda", dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e_s = float(t.item())
    e2e = {"value": world * w.ops / e2e_s / 1e12, "unit": "Tops/s", "h2d_bytes_per_step": world * w.in_bytes,
           "d2h_bytes_per_step": world * w.vis_bytes, "ms_per_step": 1e3 * e2e_s, "steps": e2e_steps,
           "api": "xc_correlate_host (pinned host in/out)"}

    # ---- the metric "vs N stations": kernel-only numbers for the other configs (rank 0, N=1) -----
    by_config = {}
    if rank == 0 and world == 1 and not args.no_sweep:
        del xd, vis, xh, vh
        torch.cuda.empty_cache()
        for name in ["cfg1", "cfg3", "cfg4", "cfg5_N32", "cfg5_N64", "cfg5_N100", "cfg5_N500", "cfg5_N1024"]:
            if name == args.workload:
                continue
            ww = wl.CONFIGS[name]
            xx = torch.from_numpy(wl.make_input(ww)).cuda()
            pp = xcb.Plan(ww.N, ww.F, ww.T)
            vv = pp.new_vis()
            d = time_kernel(pp, xx, vv, stream, 10, 3)
            ms = sorted(d)[len(d) // 2]
            # the same launch 20 times back to back between two events: what a caller streaming blocks sees (the
            # kernels are launched with programmatic stream serialization, so launch latency and prologue overlap
            # the previous kernel's tail -- the difference matters for the microsecond-scale small-N configs)
            with torch.cuda.stream(stream):
                b0, b1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                stream.synchronize()
                b0.record(stream)
                for _ in range(20):
                    pp.correlate(xx, vv, stream=stream)
                b1.record(stream)
                stream.synchronize()
            ms_b2b = b0.elapsed_time(b1) / 20
            by_config[name] = {"N": ww.N, "F": ww.F, "T": ww.T, "kernel_ms": ms,
                               "back_to_back_ms": ms_b2b, "tops_back_to_back": ww.ops / (ms_b2b * 1e-3) / 1e12,
                               "tops": ww.ops / (ms * 1e-3) / 1e12,
                               "frac_i8_peak": ww.ops / (ms * 1e-3) / 1e12 / i8_peak,
                               "hbm_gbs": (ww.in_bytes + ww.vis_bytes) / (ms * 1e-3) / 1e9,
                               "l2": "cold (input > L2)" if ww.in_bytes > 126e6 else "warm (input fits L2)"}
            pp.close()
            del xx, vv
            torch.cuda.empty_cache()

    # ---- S5 / S6 of the scope table: fp32 variant and two-stream pipeline (rank 0, N=1) -------------
    extras = {}
    if rank == 0 and world == 1 and not args.no_sweep:
        # fp32-input variant on config 3's values (BASELINE.json configs[2]); ALU-bound: peak = SMs x 128 FMA x 2 x f_max
        w3 = wl.CONFIGS["cfg3"]
        x3 = torch.from_numpy(wl.make_input(w3)).cuda().to(torch.float32)
        p3 = xcb.Plan(w3.N, w3.F, w3.T)
        v3 = p3.new_vis(torch.float32)
        for _ in range(3):
            p3.correlate_f32(x3, v3, stream=stream)
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        stream.synchronize()
        ev[0].record(stream)
        for _ in range(5):
            p3.correlate_f32(x3, v3, stream=stream)
        ev[1].record(stream)
        stream.synchronize()
        ms = ev[0].elapsed_time(ev[1]) / 5
        sms = torch.cuda.get_device_properties(0).multi_processor_count
        fp32_peak = sms * 128 * 2 * (clocks.get("sm_max_mhz") or 1965.0) * 1e6 / 1e12
        extras["f32"] = {"workload": "cfg3 values as float32 through xc_correlate_f32", "kernel_ms": ms,
                         "tflops": w3.ops / (ms * 1e-3) / 1e12, "bound": "alu", "peak_tflops": fp32_peak,
                         "frac": w3.ops / (ms * 1e-3) / 1e12 / fp32_peak,
                         "peak_source": "SMs x 128 FMA/clk x 2 x clocks.max.sm (derived, DESIGN.md 5.2)",
                         "context": "pure-register FFMA2 streams on this pool: 65.2 TFLOPS (constant operands), 57.7 TFLOPS "
                                    "(this kernel's operand pattern); round-1 probe, DESIGN.md 5.2"}
        p3.close()
        del x3, v3
        torch.cuda.empty_cache()
        # 4-bit samples on config 2's shape: device-resident (unpack + X-engine) and
        # end to end with host buffers (half the H2D bytes of the int8 call)
        w2 = wl.CONFIGS["cfg2"]
        x4h = torch.from_numpy(wl.packed_i4(w2.N, w2.F, w2.T, seed=2002)).pin_memory()
        x4d = x4h.cuda()
        p4 = xcb.Plan(w2.N, w2.F, w2.T)
        v4 = p4.new_vis()
        v4h = torch.empty(p4.vis_shape(), dtype=torch.int32).pin_memory()
        for _ in range(3):
            p4.correlate_i4(x4d, v4, stream=stream)
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        stream.synchronize()
        ev[0].record(stream)
        for _ in range(20):
            p4.correlate_i4(x4d, v4, stream=stream)
        ev[1].record(stream)
        stream.synchronize()
        ms4 = ev[0].elapsed_time(ev[1]) / 20
        p4.correlate_host_i4(x4h, v4h, x4d, v4, stream=stream)
        t0 = time.perf_counter()
        for _ in range(5):
            p4.correlate_host_i4(x4h, v4h, x4d, v4, stream=stream)
        e4 = (time.perf_counter() - t0) / 5
        extras["i4"] = {"workload": "config 2's shape with 4-bit complex samples (uniform nibbles), xc_correlate_i4 / xc_correlate_host_i4",
                        "device_ms": ms4, "tops": w2.ops / (ms4 * 1e-3) / 1e12, "launches_per_step": 2,
                        "e2e_ms": 1e3 * e4, "e2e_tops": w2.ops / e4 / 1e12, "h2d_bytes_per_step": w2.in_bytes // 2,
                        "d2h_bytes_per_step": w2.vis_bytes}
        p4.close()
        del x4h, x4d, v4, v4h
        torch.cuda.empty_cache()
        # two-stream run of config 5: 8 host blocks (the same seeded block 8 times: only the timing matters here;
        # parity of the 8-distinct-block run is tests/test_xc_gpu.py::test_cfg5_two_stream_eight_blocks)
        w5 = wl.CONFIGS["cfg5_N1024"]
        blk = torch.from_numpy(wl.make_input(w5))
        host = torch.empty((8,) + tuple(blk.shape), dtype=torch.int8).pin_memory()
        for k in range(8):
            host[k].copy_(blk)
        p5 = xcb.Plan(w5.N, w5.F, w5.T)
        dev2 = torch.empty(2 * p5.in_bytes, dtype=torch.int8, device="cuda")
        v5 = p5.new_vis()
        s2 = torch.cuda.Stream()
        p5.correlate_pipelined(host, dev2, v5, stream, s2)
        stream.synchronize()
        t0 = time.perf_counter()
        p5.correlate_pipelined(host, dev2, v5, stream, s2)
        stream.synchronize()
        tot = time.perf_counter() - t0
        t0 = time.perf_counter()
        for k in range(8):
            dev2[:p5.in_bytes].view(torch.int8).copy_(host[k].view(-1), non_blocking=True)
        torch.cuda.synchronize()
        t_copy = time.perf_counter() - t0
        xk = dev2[:p5.in_bytes].view(w5.T, w5.F, w5.N, 2, 2)
        t_comp = 8e-3 * sorted(time_kernel(p5, xk, v5, stream, 5, 2))[2]
        extras["two_stream"] = {"workload": "cfg5_N1024 x 8 pinned host blocks, xc_correlate_pipelined (Algorithm 1)",
                                "total_ms": 1e3 * tot, "copy_alone_ms": 1e3 * t_copy, "compute_alone_ms": 1e3 * t_comp,
                                "h2d_gbs": 8 * w5.in_bytes / tot / 1e9, "tops": 8 * w5.ops / tot / 1e12,
                                "overlap_efficiency": max(t_copy, t_comp) / tot}
        # the integrated run (Fig. 7): the same 8 blocks through xc_integrate -- int64 widening of the
        # int32 partial sums and the copy of the result back to the host inside the timed region
        v64 = torch.empty(p5.vis_shape(), dtype=torch.int64, device="cuda")
        v64h = torch.empty(p5.vis_shape(), dtype=torch.int64).pin_memory()
        p5.integrate(host, dev2, v5, v64, stream, s2, vis64_host=v64h)
        stream.synchronize()
        t0 = time.perf_counter()
        p5.integrate(host, dev2, v5, v64, stream, s2, vis64_host=v64h)
        stream.synchronize()
        tot_i = time.perf_counter() - t0
        extras["integrated"] = {"workload": "cfg5_N1024 x 8 pinned host blocks (16384 samples), xc_integrate: H2D pipeline, "
                                            "X-engine, int64 widening, D2H of the int64 result",
                                "total_ms": 1e3 * tot_i, "tops": 8 * w5.ops / tot_i / 1e12,
                                "h2d_bytes": 8 * w5.in_bytes, "d2h_bytes": 2 * w5.vis_bytes,
                                "pcie_floor_ms": 1e3 * (t_copy + 2 * w5.vis_bytes / (8 * w5.in_bytes / t_copy))}
        del v64, v64h
        p5.close()
        del host, dev2, v5
        torch.cuda.empty_cache()

    # ---- CPU baseline: the oracle on a bounded sample (rank 0 at N=1 only) --------------------
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu:
        v, cores, sample = cpu_sample(w, x_np)
        cpu = {"value": v, "unit": "Tops/s", "cores": cores, "kind": "oracle", "sample": sample}
    sampler.stop()

    if rank == 0:
        out = {
            "metric": "X-engine Tops/s (8 ops per cMAC)", "value": tops, "unit": "Tops/s", "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "int8", "data": "synthetic",
            "config": {"workload": workload_desc(w), "global_channels": world * w.F,
                       "parallelism": f"channel-sharded x{world}, no collective",
                       "l2": "input block (%.0f MB) + output (%.0f MB) exceed the 126 MB L2: every step is cold"
                             % (w.in_bytes / 1e6, w.vis_bytes / 1e6)},
            "clocks": clocks, "e2e": e2e, "gpu_launches": args.steps * launches_per_step,
            "roofline": roof, "cpu_baseline": cpu, "by_config": by_config, "extras": extras,
            "frac_of_int8_peak": tops / world / i8_peak, "int8_peak_tops": i8_peak,
            "paper_context": "1058 GFLOPS = 79% of fp32 peak on a GeForce GTX 480 (PAPER.md:267); other hardware",
        }
        print(json.dumps(out))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


# dram__bytes_read.sum + dram__bytes_write.sum per launch of xc_i8_tc_kernel from `ncu --set full`
# captures (see profiles/*.md for the command and the raw numbers); null until captured.
TRAFFIC_NCU: dict = {
    "cfg2": 524557824 + 237699584,        # profiles/r1_ncu_full_cfg2.md
    "cfg4": 524457216 + 1019722000,       # profiles/r1_ncu_full_cfg4.md
    "cfg5_N1024": 537382656 + 1022897000,  # profiles/r1_ncu_full_cfg5N1024.md
}

if __name__ == "__main__":
    main()
