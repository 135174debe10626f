#!/usr/bin/env python
"""bench.py -- X-engine throughput on B200 (BASELINE.json metric: Tops/s at 8 ops per complex MAC, vs N stations).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg5_N1024] [--impl reference]

A "step" is one pass of the whole hot path (S0-S4 of SURVEY 8(a): staging if needed, tile schedule, tcgen05 X-engine,
packing epilogue) over one synthetic input block through the C-ABI library.  Default workload = the largest single-GPU
configuration of BASELINE.json (configs[4], N = 1024: the regime north_star's target is defined on).  Prints ONE JSON line.

  value        whole-job Tops/s, inputs resident in HBM (ops = 8 * F * T * N(2N+1), Eq. 5), K steps back to back
  e2e          same metric through xc_correlate_host with HOST buffers (H2D + X-engine + D2H per step)
  roofline     the dominant kernel (xc_i8_tc_kernel) of the headline workload: burst (isolated launches, duration from the
               kernel's own globaltimer stamps) against the burst peak, `sustained` (>= 2 s of back-to-back launches, NVML
               power / clock trace) against the sustained peak, and `per_config`: the same for every BASELINE config
  cpu_baseline the oracle (oracle/xo_oracle.c, as it stands) on the box's host cores, bounded sample
  extras       fp32 variant, 4-bit samples, two-stream pipeline, integrated run, pitched N = 500, F-engine + FX chain

N > 1 (torchrun): every rank runs its own block of F channels (channels are independent): no data-path
collective, "scaling": "weak"; time = max over ranks.
"""
from __future__ import annotations

import argparse
import csv
import glob
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

NOMINAL_I8_OVER_BF16 = 2.0          # 4.5 / 2.25 PFLOP/s dense (B200_PROFILING.md nominal table)
NOMINAL_I8_TOPS = 4500.0            # dense int8 = fp8 nominal (B200_PROFILING.md)
FALLBACK_HBM_GBS, FALLBACK_BF16_TF = 6650.0, 1590.0
NCU_CAPTURE_COMMIT = ("headline cfg5_N1024: round 3's build (2026-11-06, profiles/r3_ncu_cfg5_N1024.csv); other configs: 0f76063 "
                      "(2026-11-05, profiles/r2_ncu_*.csv; the X-engine kernel source is unchanged since)")
SWEEP = ["cfg1", "cfg2", "cfg3", "cfg4", "cfg5_N32", "cfg5_N64", "cfg5_N100", "cfg5_N500", "cfg5_N1024"]
SUSTAINED = {"cfg2", "cfg3", "cfg4", "cfg5_N500", "cfg5_N1024"}      # the configs north_star's target speaks about (+ cfg2)


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as fh:
            m = json.load(fh)
        return {"hbm_gbs": float(m["hbm_gbs"]), "bf16_burst": float(m["bf16_tflops"]),
                "bf16_sustained": float(m.get("bf16_tflops_sustained", m["bf16_tflops"])), "source": "measured"}
    return {"hbm_gbs": FALLBACK_HBM_GBS, "bf16_burst": FALLBACK_BF16_TF, "bf16_sustained": 1400.0,
            "source": "fallback"}


def ncu_profile(workload, kernel="xc_i8_tc_kernel"):
    """Counters of xc_i8_tc_kernel from the tracked ncu export profiles/r2_ncu_<workload>.csv (written by
    `ncu -i <rep> --page raw --csv --print-units base --metrics ...`; the .md beside it names the commands).  Returns
    {} when no capture of this round exists: nothing is hard-coded here."""
    path = os.path.join(ROOT, "profiles", f"r3_ncu_{workload}.csv")       # this round's capture where one was made
    if not os.path.exists(path):
        path = os.path.join(ROOT, "profiles", f"r2_ncu_{workload}.csv")   # else round 2's (the kernel source is unchanged)
    if not os.path.exists(path):
        return {}
    with open(path, newline="") as fh:
        rows = list(csv.reader(fh))
    rows = [r for r in rows if r and r[0].strip('"') not in ("",) or (r and len(r) > 4)]
    hdr = next((r for r in rows if "Kernel Name" in r), None)
    if hdr is None:
        return {}
    ki = hdr.index("Kernel Name")
    data = [r for r in rows if len(r) == len(hdr) and kernel in r[ki]]
    if not data:
        return {}

    def col(name):
        if name not in hdr:
            return None
        vals = [float(r[hdr.index(name)]) for r in data if r[hdr.index(name)] not in ("", "n/a")]
        return sum(vals) / len(vals) if vals else None
    rd, wr = col("dram__bytes_read.sum"), col("dram__bytes_write.sum")
    out = {"file": os.path.relpath(path, ROOT), "launches": len(data),
           "dram_bytes": (rd + wr) if rd is not None and wr is not None else None,
           "duration_us": (col("gpu__time_duration.sum") or 0) / 1e3 or None,
           "tensor_pipe_active_pct": col("sm__pipe_tensor_cycles_active.avg.pct_of_peak_sustained_elapsed"),
           "l2_to_sm_read_bytes": col("l1tex__m_xbar2l1tex_read_bytes.sum"),
           "sm_ghz": (col("sm__cycles_elapsed.avg.per_second") or 0) / 1e9 or None}
    return out


class ClockSampler:
    """SM clock, power and throttle reasons sampled through NVML (pynvml) every ~1 ms by a thread, DURING the timed
    regions (the recipe's clocks line, without nvidia-smi's start-up latency)."""
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
        pw = sorted(r[3] for r in rows)
        bits = 0
        for r in rows:
            bits |= r[2]
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": self.max_sm, "samples": len(sm),
                "power_w_median": pw[len(pw) // 2] if pw else None, "power_w_max": pw[-1] if pw else None,
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
    """--impl reference: the CPU oracle as it stands, on the host cores (rank 0 only).  A step = a bounded sample of the
    workload: `cores` channels (the oracle parallelises over channels only) and as many time samples as the oracle does in
    about 2 s, so that the driver's --steps 20 --warmup 5 ends within a few minutes at every N."""
    if rank != 0:
        return
    import xc_workloads as wl
    from oracle import xo
    w = wl.CONFIGS[args.workload]
    cores = xo.num_threads()
    nch = max(1, min(w.F, cores))
    sel = list(range(nch))
    per_sample = nch * w.N * (2 * w.N + 1)                         # cMACs per time sample of the step
    t_cal = min(w.T, 32)
    x_cal = wl.make_input(wl.Workload(w.name, w.N, nch, t_cal, w.kind, w.sigma, w.seed))
    xo.channels_i8(x_cal, sel)
    t0 = time.perf_counter()
    xo.channels_i8(x_cal, sel)
    rate = t_cal * per_sample / (time.perf_counter() - t0)
    T_s = int(max(1, min(w.T, 2.0 * rate / per_sample)))
    x = wl.make_input(wl.Workload(w.name, w.N, nch, T_s, w.kind, w.sigma, w.seed))
    for _ in range(args.warmup):
        xo.channels_i8(x, sel)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        xo.channels_i8(x, sel)
    dt = time.perf_counter() - t0
    tops = 8.0 * args.steps * T_s * per_sample / dt / 1e12
    sample = f"{nch} of {w.F} channels x {T_s} of {w.T} time samples of {w.name} per step, all baselines"
    print(json.dumps({
        "impl": "reference", "metric": "X-engine Tops/s (8 ops per cMAC)", "value": tops, "unit": "Tops/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "int8", "data": "synthetic",
        "config": {"workload": workload_desc(w), "sample": sample},
        "cpu_baseline": {"value": tops, "unit": "Tops/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": tops, "unit": "Tops/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


# ------------------------------------------------------------------------------------------------------------------
# timing helpers (all on the launching stream)
# ------------------------------------------------------------------------------------------------------------------

def kernel_durations(p, xd, vis, stream, n):
    """n isolated launches; per launch (a) the duration from the kernel's own globaltimer stamps (min over CTAs at entry,
    max at exit: xc_set_timing_buffer), (b) the CUDA-event time around the call (includes the launch gap), (c) the SM clock
    from CTA 0's cycle counter.  Returns medians: (kernel_ms, event_ms, sm_mhz_in_kernel)."""
    import torch
    import paper_1107_4264_b200 as xcb
    init = torch.tensor([2 ** 62, 0, 0, 0, 0, 0], dtype=torch.int64, device="cuda")
    st = init.repeat(n, 1).contiguous()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n)]
    with torch.cuda.stream(stream):
        p.correlate(xd, vis, stream=stream)
        stream.synchronize()
        for k, (a, b) in enumerate(evs):
            p.set_timing_buffer(st[k])
            a.record(stream)
            p.correlate(xd, vis, stream=stream)
            b.record(stream)
            stream.synchronize()                      # isolated: nothing overlaps the next launch's prologue
    p.set_timing_buffer(None)
    rows = st.tolist()
    dur = sorted((r[1] - r[0]) / 1e6 for r in rows)
    ev = sorted(a.elapsed_time(b) for a, b in evs)
    mhz = sorted((r[4] - r[2]) / (r[5] - r[3]) * 1e3 for r in rows if r[5] > r[3])
    assert xcb.TIMING_WORDS == 6
    return dur[len(dur) // 2], ev[len(ev) // 2], (mhz[len(mhz) // 2] if mhz else None)


def back_to_back(p, xd, vis, stream, n):
    import torch
    with torch.cuda.stream(stream):
        b0, b1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        stream.synchronize()
        b0.record(stream)
        for _ in range(n):
            p.correlate(xd, vis, stream=stream)
        b1.record(stream)
        stream.synchronize()
    return b0.elapsed_time(b1) / n


def sustained_leg(p, xd, vis, stream, sampler, seconds, est_ms, fn=None):
    """>= `seconds` of back-to-back launches; throughput, power and clocks over the SECOND half (steady state under the
    power cap).  Returns dict with ms per launch and the NVML summary."""
    import torch
    batch = max(8, min(2000, int(0.1 / (est_ms * 1e-3))))            # ~0.1 s of work per batch
    marks = []
    call = fn or (lambda: p.correlate(xd, vis, stream=stream))
    with torch.cuda.stream(stream):
        stream.synchronize()
        t_begin = time.perf_counter()
        e_prev = torch.cuda.Event(enable_timing=True)
        e_prev.record(stream)
        queued = 0
        while True:
            for _ in range(batch):
                call()
            e = torch.cuda.Event(enable_timing=True)
            e.record(stream)
            queued += 1
            marks.append((e_prev, e, None))
            e_prev = e
            if queued >= 2:                                            # keep at most two batches in flight
                marks[queued - 2][1].synchronize()
                marks[queued - 2] = (marks[queued - 2][0], marks[queued - 2][1], time.perf_counter())
            if time.perf_counter() - t_begin >= seconds and queued >= 4:
                break
        stream.synchronize()
        t_end = time.perf_counter()
    marks[-1] = (marks[-1][0], marks[-1][1], t_end)
    if marks[-2][2] is None:
        marks[-2] = (marks[-2][0], marks[-2][1], t_end)
    half = len(marks) // 2
    ms = sum(a.elapsed_time(b) for a, b, _ in marks[half:]) / (batch * (len(marks) - half))
    first_ms = marks[0][0].elapsed_time(marks[0][1]) / batch
    t_half = marks[half - 1][2] if half >= 1 and marks[half - 1][2] else t_begin
    nv = sampler.window(t_half, t_end)
    return {"seconds": t_end - t_begin, "launches": batch * len(marks), "ms_per_launch": ms, "first_batch_ms_per_launch": first_ms,
            "nvml": {k: nv.get(k) for k in ("sm_mhz", "power_w_median", "power_w_max", "reasons", "samples")}}


def roofline_entry(w, k_ms, peaks, i8_burst, prof):
    """algorithmic bytes = input once + output once; algorithmic ops = Eq. 5.  The bound is the roof that
    takes longer at its measured peak."""
    alg_bytes = w.in_bytes + w.vis_bytes
    t_hbm = alg_bytes / (peaks["hbm_gbs"] * 1e9)
    t_tc = w.ops / (i8_burst * 1e12)
    tops = w.ops / (k_ms * 1e-3) / 1e12
    gbs = alg_bytes / (k_ms * 1e-3) / 1e9
    if t_hbm >= t_tc:
        e = {"bound": "hbm", "achieved": gbs, "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": gbs / peaks["hbm_gbs"]}
    else:
        e = {"bound": "tensor", "achieved": tops, "peak": i8_burst, "unit": "Tops/s", "frac": tops / i8_burst}
    e.update({"traffic": prof.get("dram_bytes"), "kernel_ms": k_ms, "tops": tops, "hbm_gbs": gbs,
              "frac_tensor_burst_peak": tops / i8_burst, "frac_tensor_nominal_4500": tops / NOMINAL_I8_TOPS,
              "frac_hbm_peak": gbs / peaks["hbm_gbs"], "algorithmic_bytes": alg_bytes, "algorithmic_ops": w.ops})
    if prof:
        e["ncu"] = prof
    return e


def flat_roofline_keys(per_config, extras, denominators):
    """Scalar copies of the per-config fractions, directly under `roofline` (a reader that keeps only the scalar keys of
    `roofline` still sees a fraction for every config north_star's target names, Fig. 5: rate against N).
    frac_<cfg> = burst fraction of the config's own bound (the `bound_<cfg>` key says which: tensor = bf16 burst x 2, hbm =
    measured copy bandwidth); frac_<cfg>_hbm = algorithmic bytes / in-kernel time over the HBM peak whatever the bound;
    sustained_frac_<cfg> = >= 1.5 s back to back against bf16 sustained x 2."""
    flat = {}
    for name, e in per_config.items():
        flat[f"frac_{name}"] = e.get("frac")
        flat[f"bound_{name}"] = e.get("bound")
        flat[f"tops_{name}"] = e.get("tops")
        flat[f"frac_{name}_hbm"] = e.get("frac_hbm_peak")
        if "sustained" in e:
            flat[f"sustained_frac_{name}"] = e["sustained"].get("frac")
        if denominators.get("cublas_int8_burst") and e.get("bound") == "tensor":
            flat[f"frac_vs_cublas_int8_{name}"] = e["tops"] / denominators["cublas_int8_burst"]
        if e.get("tensor_pipe_active_ncu_pct") is not None:
            flat[f"ncu_tensor_pipe_pct_{name}"] = e["tensor_pipe_active_ncu_pct"]
    fx = extras.get("fx") or {}
    flat["fengine_frac_hbm"] = fx.get("frac_hbm")
    flat["fengine_ms"] = fx.get("fengine_ms")
    f32 = extras.get("f32") or {}
    flat["f32tc_tflops"] = f32.get("tflops")
    flat["f32tc_frac"] = f32.get("frac")
    flat["f32tc_tensor_pipe_pct"] = ncu_profile("f32tc", kernel="xc_f32_tc_kernel").get("tensor_pipe_active_pct")
    i4 = extras.get("i4") or {}
    flat["i4_tops"] = i4.get("tops")
    # the ncu-derived numbers (traffic, tensor_pipe) describe the build that was profiled, not the one timed in this run
    flat["traffic_captured_at_commit"] = NCU_CAPTURE_COMMIT
    return flat


def useful_over_raw(p, w):
    """Stored baselines / baselines the scheduled tiles compute (the paper's wasted-work measure); with an
    origin shift the tile count is the mean over the channel classes of the last call."""
    tiles = p.tiles()
    si, sj = tiles[0][2:]
    cls = p.origin_shift
    n = sum(t for _, t in cls) / len(cls) if cls and cls[0][1] else len(tiles)
    return (w.N * (w.N + 1) / 2) / (n * si * sj)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="cfg5_N1024")
    ap.add_argument("--impl", default="native", choices=["native", "reference"])
    ap.add_argument("--no-sweep", action="store_true", help="skip roofline.per_config and the extras")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--no-sustained", action="store_true", help="skip the sustained legs")
    ap.add_argument("--sustained-seconds", type=float, default=2.0)
    ap.add_argument("--pitch", type=int, default=0, help="profiling aid: run the workload from a block with this row pitch")
    ap.add_argument("--only", default="", choices=["", "f32", "f32tc", "fengine", "trace", "noalloc"],
                    help="profiling aid: run only a few launches of that leg (for ncu) and print a short JSON line; trace = pipeline "
                         "timeline of CTA 0 from the -DXC_PROFILE build")
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
    import bench_legs

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the X-engine has no CPU path")
    if rank == 0:
        xc_build.build()
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
        dist.barrier()
    xcb.load_library()
    stream = torch.cuda.Stream()

    if args.only:
        print(json.dumps(bench_legs.only_leg(args.only, args.workload, stream)))
        return

    peaks = load_peaks()
    i8_burst = peaks["bf16_burst"] * NOMINAL_I8_OVER_BF16          # Tops/s: measured bf16 burst x nominal int8/bf16 ratio
    i8_sustained = peaks["bf16_sustained"] * NOMINAL_I8_OVER_BF16
    w = wl.CONFIGS[args.workload]
    # weak scaling: every rank holds its own block of F channels (seed differs per rank)
    x_np = wl.make_input(w, seed=w.seed + 7919 * rank)
    p = xcb.Plan(w.N, w.F, w.T)
    xh = torch.from_numpy(x_np).pin_memory()
    if args.pitch:
        p.set_in_pitch(args.pitch)
        xd = torch.zeros((w.T, w.F, args.pitch), dtype=torch.int8, device="cuda")
        xd[:, :, :4 * w.N] = xh.cuda().view(w.T, w.F, 4 * w.N)
    else:
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

    # ---- the dominant kernel: duration from its own stamps, burst roofline ---------------------
    k_ms, ev_ms, mhz_k = kernel_durations(p, xd, vis, stream, min(max(args.steps, 5), 20))
    roof = roofline_entry(w, k_ms, peaks, i8_burst, ncu_profile(w.name))
    roof.update({
        "kernel": "xc_i8_tc_kernel", "event_ms": ev_ms, "useful_over_raw": useful_over_raw(p, w),
        "kernel_ms_how": "median over isolated launches of (max over CTAs of globaltimer at exit) - (min at entry), written by "
                         "the kernel itself (xc_set_timing_buffer); event_ms = CUDA events around the same call (adds the launch gap)",
        "peak_source": peaks["source"] + (" hbm_gbs (MEASURED_PEAKS.json)" if roof["bound"] == "hbm" else
                                          " bf16_tflops (burst, MEASURED_PEAKS.json) x 2 (nominal int8/bf16 ratio): NOT a measured int8 number"),
        "traffic_source": roof.get("ncu", {}).get("file"),
    })
    clocks["sm_mhz_in_kernel"] = mhz_k
    clocks["sm_mhz_in_kernel_how"] = "clock64 / globaltimer stamped by CTA 0 of xc_i8_tc_kernel at entry and exit, median of isolated launches"

    # ---- other denominators for "% of int8 tensor peak": measured cuBLAS int8 GEMM, nominal -----------
    denominators = {"bf16_burst_x2": i8_burst, "bf16_sustained_x2": i8_sustained, "nominal_dense_int8": NOMINAL_I8_TOPS}
    if rank == 0 and not args.no_sweep:
        denominators.update(bench_legs.cublas_int8_peak(stream))
    roof["denominators_tops"] = denominators
    if denominators.get("cublas_int8_burst"):
        roof["frac_vs_cublas_int8_burst"] = roof["tops"] / denominators["cublas_int8_burst"]

    # ---- sustained leg of the headline workload ------------------------------------------------------------------
    if not args.no_sustained:
        s = sustained_leg(p, xd, vis, stream, sampler, args.sustained_seconds, k_ms)
        s_tops = w.ops / (s["ms_per_launch"] * 1e-3) / 1e12
        s.update({"tops": s_tops, "peak": i8_sustained, "frac": s_tops / i8_sustained,
                  "peak_source": peaks["source"] + " bf16_tflops_sustained x 2 (nominal int8/bf16 ratio)",
                  "frac_hbm_peak": (w.in_bytes + w.vis_bytes) / (s["ms_per_launch"] * 1e-3) / 1e9 / peaks["hbm_gbs"]})
        if denominators.get("cublas_int8_sustained"):
            s["frac_vs_cublas_int8_sustained"] = s_tops / denominators["cublas_int8_sustained"]
        roof["sustained"] = s

    # ---- end to end through the C ABI with HOST buffers ---------------------------------------
    vh = torch.empty(p.vis_shape(), dtype=torch.int32).pin_memory()
    scratch = p.new_scratch()
    if args.pitch:
        p.set_in_pitch(0)
    e2e_steps = max(3, min(args.steps, 10))
    p.correlate_host(xh, vh, scratch, vis, stream=stream)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        p.correlate_host(xh, vh, scratch, vis, stream=stream)       # synchronises the stream itself
    e2e_s = (time.perf_counter() - t0) / e2e_steps
    if world > 1:
        t = torch.tensor([e2e_s], device="cuda", dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e_s = float(t.item())
    e2e = {"value": world * w.ops / e2e_s / 1e12, "unit": "Tops/s", "h2d_bytes_per_step": world * w.in_bytes,
           "d2h_bytes_per_step": world * w.vis_bytes, "ms_per_step": 1e3 * e2e_s, "steps": e2e_steps,
           "api": "xc_correlate_host (pinned host in/out)",
           "pcie_floor_ms": 1e3 * max(w.in_bytes, w.vis_bytes) / 55e9}
    del scratch, vh

    # ---- the metric "vs N stations": every BASELINE config, kernel only (rank 0, N=1) --------------------------
    per_config = {}
    extras = {}
    if rank == 0 and world == 1 and not args.no_sweep:
        per_config[w.name] = {k: roof[k] for k in ("bound", "achieved", "peak", "unit", "frac", "traffic", "kernel_ms", "event_ms", "tops",
                                                   "hbm_gbs", "frac_tensor_burst_peak", "frac_tensor_nominal_4500", "frac_hbm_peak",
                                                   "useful_over_raw")}
        per_config[w.name]["back_to_back_ms"] = ms_step
        if "sustained" in roof:
            per_config[w.name]["sustained"] = {k: roof["sustained"][k] for k in ("ms_per_launch", "tops", "frac", "nvml")}
        if "ncu" in roof:
            per_config[w.name]["tensor_pipe_active_ncu_pct"] = roof["ncu"].get("tensor_pipe_active_pct")
        del xd, vis, xh
        torch.cuda.empty_cache()
        for name in SWEEP:
            if name == w.name:
                continue
            ww = wl.CONFIGS[name]
            xx = torch.from_numpy(wl.make_input(ww)).cuda()
            pp = xcb.Plan(ww.N, ww.F, ww.T)
            vv = pp.new_vis()
            time.sleep(0.5)          # the previous config's sustained leg must not set this one's burst clocks
            km, em, mhz = kernel_durations(pp, xx, vv, stream, 10)
            prof = ncu_profile(name)
            ent = roofline_entry(ww, km, peaks, i8_burst, prof)
            ent.pop("ncu", None)
            ent.update({"N": ww.N, "F": ww.F, "T": ww.T, "event_ms": em, "sm_mhz_in_kernel": mhz,
                        "back_to_back_ms": back_to_back(pp, xx, vv, stream, 20 if ww.in_bytes > 60e6 else 200),
                        "useful_over_raw": useful_over_raw(pp, ww), "tile": pp.tiles()[0][2:], "t_split": pp.t_split,
                        "origin_shift_bytes_tiles": pp.origin_shift,
                        "tensor_pipe_active_ncu_pct": prof.get("tensor_pipe_active_pct"),
                        "l2": "cold (input > L2)" if ww.in_bytes > 126e6 else "warm (input fits L2)"})
            ent["tops_back_to_back"] = ww.ops / (ent["back_to_back_ms"] * 1e-3) / 1e12
            if name in SUSTAINED and not args.no_sustained:
                s = sustained_leg(pp, xx, vv, stream, sampler, min(args.sustained_seconds, 1.5), km)
                s_tops = ww.ops / (s["ms_per_launch"] * 1e-3) / 1e12
                ent["sustained"] = {"ms_per_launch": s["ms_per_launch"], "tops": s_tops, "frac": s_tops / i8_sustained, "nvml": s["nvml"]}
            per_config[name] = ent
            if name in ("cfg5_N500", "cfg5_N100"):
                # the same dense block with the tile grids left unshifted (XC_OPT_ORIGIN_SHIFT = 0: round 1's schedule)
                pp.set_option(xcb.OPT_ORIGIN_SHIFT, 0)
                time.sleep(0.5)
                ent["origin_shift_off_kernel_ms"] = kernel_durations(pp, xx, vv, stream, 10)[0]
                pp.set_option(xcb.OPT_ORIGIN_SHIFT, 1)
            if name == "cfg5_N500":
                # the same values in a block whose rows are xc_scratch_pitch() = 2048 bytes apart (xc_set_in_pitch): what the
                # F-engine and the host-buffer calls hand to the X-engine (line-aligned rows)
                pitch = pp.scratch_pitch
                xp = torch.zeros((ww.T, ww.F, pitch), dtype=torch.int8, device="cuda")
                xp[:, :, :4 * ww.N] = xx.view(ww.T, ww.F, 4 * ww.N)
                pp.set_in_pitch(pitch)
                time.sleep(0.5)
                km2, em2, mhz2 = kernel_durations(pp, xp, vv, stream, 10)
                ent2 = roofline_entry(ww, km2, peaks, i8_burst, ncu_profile(name + "_p2048"))
                ent2.pop("ncu", None)
                ent2.update({"N": ww.N, "F": ww.F, "T": ww.T, "row_pitch_bytes": pitch, "event_ms": em2, "sm_mhz_in_kernel": mhz2,
                             "back_to_back_ms": back_to_back(pp, xp, vv, stream, 20),
                             "tensor_pipe_active_ncu_pct": ncu_profile(name + "_p2048").get("tensor_pipe_active_pct")})
                if not args.no_sustained:
                    s = sustained_leg(pp, xp, vv, stream, sampler, min(args.sustained_seconds, 1.5), km2)
                    s_tops = ww.ops / (s["ms_per_launch"] * 1e-3) / 1e12
                    ent2["sustained"] = {"ms_per_launch": s["ms_per_launch"], "tops": s_tops, "frac": s_tops / i8_sustained, "nvml": s["nvml"]}
                per_config["cfg5_N500_pitch2048"] = ent2
                del xp
            pp.close()
            del xx, vv
            torch.cuda.empty_cache()
        roof["per_config"] = per_config
        roof["per_config_note"] = ("burst: isolated launches, in-kernel duration, peak = bf16 burst x 2 (tensor) or measured HBM copy; "
                                   "sustained: >= 1.5 s back to back, frac against bf16 sustained x 2; tensor_pipe_active_ncu_pct from the "
                                   "tracked ncu exports under profiles/ (null = no capture this round)")
        extras = bench_legs.extras(stream, clocks, sampler, peaks)
        roof.update(flat_roofline_keys(per_config, extras, denominators))
    else:
        del xd, vis, xh

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
            "roofline": roof, "cpu_baseline": cpu, "extras": extras,
            "paper_context": "1058 GFLOPS = 79% of fp32 peak on a GeForce GTX 480 (PAPER.md:267); other hardware",
        }
        print(json.dumps(out))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
