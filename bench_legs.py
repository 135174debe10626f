"""bench_legs.py -- the secondary legs of bench.py (rank 0, one GPU): the other steps of SURVEY 8(a)/(f) beside the int8
X-engine -- fp32 variant (S5), two-stream pipeline (S6), integrated run, 4-bit samples, pitched N = 500 input, F-engine and
FX chain -- and the measured cuBLAS int8 GEMM rate used as an extra roofline denominator.  Everything here goes through the
C-ABI library exactly as bench.py's main leg does; nothing imports the oracle."""
from __future__ import annotations

import time


def _timed(fn, stream, n, warm=3):
    """Mean ms of n back-to-back calls of fn() between two events on `stream`."""
    import torch
    with torch.cuda.stream(stream):
        for _ in range(warm):
            fn()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        stream.synchronize()
        e0.record(stream)
        for _ in range(n):
            fn()
        e1.record(stream)
        stream.synchronize()
    return e0.elapsed_time(e1) / n


def cublas_int8_peak(stream):
    """cuBLAS int8 GEMM (torch._int_mm, 8192^3, int32 accumulate) on this very GPU: best of 10 (burst) and the mean of a
    ~1.5 s back-to-back loop (sustained).  A LIBRARY kernel used only as a denominator: what a vendor GEMM of the same
    dtype reaches, next to bf16 x 2 and the nominal 4500 Tops."""
    import torch
    try:
        n = 8192
        a = torch.randint(-127, 128, (n, n), dtype=torch.int8, device="cuda")
        b = torch.randint(-127, 128, (n, n), dtype=torch.int8, device="cuda")
        ops = 2.0 * n ** 3
        with torch.cuda.stream(stream):
            for _ in range(3):
                torch._int_mm(a, b)
            best = 1e9
            for _ in range(10):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                torch._int_mm(a, b)
                e1.record(stream)
                stream.synchronize()
                best = min(best, e0.elapsed_time(e1))
            reps = max(50, int(1.5 / (best * 1e-3)))
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            for _ in range(reps):
                torch._int_mm(a, b)
            e1.record(stream)
            stream.synchronize()
            sus = e0.elapsed_time(e1) / reps
        del a, b
        torch.cuda.empty_cache()
        return {"cublas_int8_burst": ops / (best * 1e-3) / 1e12, "cublas_int8_sustained": ops / (sus * 1e-3) / 1e12,
                "cublas_int8_how": "torch._int_mm 8192^3 measured in this run: best of 10 / mean over ~1.5 s back to back"}
    except Exception as e:  # noqa: BLE001 -- a missing library routine must not fail the bench
        return {"cublas_int8_burst": None, "cublas_int8_sustained": None, "cublas_int8_how": f"unavailable: {e!r}"}


def f32_leg(stream, clocks, F=None, launches=5, peaks=None, kernel=None, sampler=None):
    """xc_correlate_f32 on config 3's values as float32: the tensor-core kernel (three TF32 MMAs per product; what AUTO runs at
    this N) with a tensor roofline, and the CUDA-core kernel (packed FMAs, the paper's scheme) with its ALU roofline.
    kernel = "tc" / "cuda_cores": only that one (ncu captures)."""
    import torch
    import paper_1107_4264_b200 as xcb
    import xc_workloads as wl
    w3 = wl.CONFIGS["cfg3"]
    if F:
        w3 = wl.Workload("cfg3_f32", w3.N, F, w3.T, w3.kind, w3.sigma, w3.seed)
    x3 = torch.from_numpy(wl.make_input(w3)).cuda().to(torch.float32)
    p3 = xcb.Plan(w3.N, w3.F, w3.T)
    v3 = p3.new_vis(torch.float32)
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    out = {"workload": f"cfg3 values (N={w3.N}, F={w3.F}, T={w3.T}) as float32 through xc_correlate_f32"}
    in_bytes, vis_bytes = 16.0 * w3.N * w3.F * w3.T, 32.0 * (w3.N * (w3.N + 1) // 2) * w3.F
    if kernel in (None, "tc"):
        p3.set_option(xcb.OPT_F32_KERNEL, xcb.F32_KERNEL_TC)
        ms = _timed(lambda: p3.correlate_f32(x3, v3, stream=stream), stream, launches)
        bf16 = (peaks or {}).get("bf16_burst") or 1590.0
        tf32x3 = bf16 * 0.5 / 3.0
        out.update({"kernel": "xc_f32_tc_kernel (tcgen05 kind::tf32, hi/lo split: 3 MMAs per product)", "kernel_ms": ms,
                    "tflops": w3.ops / (ms * 1e-3) / 1e12, "bound": "tensor", "peak_tflops": tf32x3,
                    "frac": w3.ops / (ms * 1e-3) / 1e12 / tf32x3,
                    "peak_source": "bf16_tflops (burst, MEASURED_PEAKS.json) x 0.5 (nominal tf32/bf16 ratio) / 3 (MMAs per product): "
                                   "useful fp32-equivalent flops; NOT a measured tf32 number",
                    "frac_tensor_nominal": w3.ops / (ms * 1e-3) / 1e12 / (1125.0 / 3.0),
                    "frac_note": "frac may exceed 1: the denominator is derived from the cuBLAS bf16 measurement (0.73 of the nominal bf16 "
                                 "peak); frac_tensor_nominal is against the nominal dense TF32 rate 1125 TFLOPS / 3",
                    "hbm_gbs": (in_bytes + vis_bytes) / (ms * 1e-3) / 1e9, "algorithmic_bytes": in_bytes + vis_bytes})
        if sampler is not None:
            from bench import sustained_leg
            sus = sustained_leg(None, None, None, stream, sampler, 1.5, ms, fn=lambda: p3.correlate_f32(x3, v3, stream=stream))
            s_tf = w3.ops / (sus["ms_per_launch"] * 1e-3) / 1e12
            s_peak = ((peaks or {}).get("bf16_sustained") or 1400.0) * 0.5 / 3.0
            out["sustained"] = {"ms_per_launch": sus["ms_per_launch"], "tflops": s_tf, "peak_tflops": s_peak, "frac": s_tf / s_peak,
                                "peak_source": "bf16_tflops_sustained x 0.5 / 3 (derived)", "nvml": sus["nvml"]}
    if kernel in (None, "cuda_cores"):
        if sampler is not None:
            time.sleep(0.5)                                  # after the sustained leg
        p3.set_option(xcb.OPT_F32_KERNEL, xcb.F32_KERNEL_CUDA_CORES)
        ms = _timed(lambda: p3.correlate_f32(x3, v3, stream=stream), stream, launches)
        fp32_peak = sms * 128 * 2 * ((clocks or {}).get("sm_max_mhz") or 1965.0) * 1e6 / 1e12
        cc = {"kernel": "xc_f32_kernel (CUDA cores, packed fma.rn.f32x2; the paper's register tiling)", "kernel_ms": ms,
              "tflops": w3.ops / (ms * 1e-3) / 1e12, "bound": "alu", "peak_tflops": fp32_peak,
              "frac": w3.ops / (ms * 1e-3) / 1e12 / fp32_peak,
              "peak_source": "SMs x 128 FMA/clk x 2 x clocks.max.sm (derived, DESIGN.md 5.2)"}
        if F is None:
            cc["fma_issue_probe"] = fma_probe()
        out["cuda_cores"] = cc
    p3.close()
    del x3, v3
    torch.cuda.empty_cache()
    if kernel is None and F is None:
        # the tensor-core kernel against N (T = 2048, F N = 8192: 268 MB of float samples each; random normal floats)
        sweep = {}
        for N in (64, 128, 256, 512, 1024):
            Fn, T = 8192 // N, 2048
            x = torch.randn((T, Fn, N, 2, 2), device="cuda")
            p = xcb.Plan(N, Fn, T)
            v = p.new_vis(torch.float32)
            ms = _timed(lambda: p.correlate_f32(x, v, stream=stream), stream, launches)
            ops = 8.0 * Fn * T * N * (2 * N + 1)
            sweep[f"N{N}"] = {"F": Fn, "T": T, "kernel_ms": ms, "tflops": ops / (ms * 1e-3) / 1e12,
                              "frac": ops / (ms * 1e-3) / 1e12 / out["peak_tflops"]}
            p.close()
            del x, v
            torch.cuda.empty_cache()
        out["tensor_core_vs_N"] = sweep
    return out


def build_probe(force=False):
    """nvcc bench_probe.cu -> libbench_probe.so (sm_100a), next to this file: a bench aid, not part of the library."""
    import os
    import subprocess
    here = os.path.dirname(os.path.abspath(__file__))
    src, lib = os.path.join(here, "bench_probe.cu"), os.path.join(here, "libbench_probe.so")
    if force or not os.path.exists(lib) or os.path.getmtime(lib) < os.path.getmtime(src):
        nvcc = os.path.join(os.environ.get("CUDA_HOME", "/usr/local/cuda"), "bin", "nvcc")
        tmp = lib + f".tmp{os.getpid()}"
        subprocess.check_call([nvcc if os.path.exists(nvcc) else "nvcc", "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a",
                               "-lineinfo", "-shared", "-Xcompiler", "-fPIC", "-o", tmp, src])
        os.replace(tmp, lib)
    return lib


def f32_pitch_leg(stream, launches=5):
    """Float samples at ragged N (rows aligned to the memory line): the tensor-core fp32 kernel on a dense
    block whose 16N-byte rows straddle 128-byte lines (N % 8 != 0) against the same values in rows padded to a multiple of
    128 bytes (xc_set_in_pitch_f32).  T = 2048, F N ~ 8192: ~268 MB of random normal floats each."""
    import torch
    import paper_1107_4264_b200 as xcb
    out = {}
    for N in (100, 500):
        Fn, T = 8192 // N, 2048
        x = torch.randn((T, Fn, 4 * N), device="cuda")
        p = xcb.Plan(N, Fn, T)
        v = p.new_vis(torch.float32)
        ops = 8.0 * Fn * T * N * (2 * N + 1)
        ms_d = _timed(lambda: p.correlate_f32(x.view(T, Fn, N, 2, 2), v, stream=stream), stream, launches)
        pitch = (16 * N + 127) // 128 * 128
        xp = torch.zeros((T, Fn, pitch // 4), device="cuda")
        xp[:, :, :4 * N] = x
        p.set_in_pitch_f32(pitch)
        ms_p = _timed(lambda: p.correlate_f32(xp, v, stream=stream), stream, launches)
        out[f"N{N}"] = {"F": Fn, "T": T, "dense_row_bytes": 16 * N, "dense_ms": ms_d, "dense_tflops": ops / (ms_d * 1e-3) / 1e12,
                        "pitch_bytes": pitch, "pitched_ms": ms_p, "pitched_tflops": ops / (ms_p * 1e-3) / 1e12}
        p.close()
        del x, xp, v
        torch.cuda.empty_cache()
    return out


def two_stream_vs_n(stream, s2, names=("cfg5_N32", "cfg5_N64", "cfg5_N100", "cfg5_N500"), blocks=4):
    """The paper's Fig. 4 / Fig. 7 analogue over N (kernel time against host-to-device time, "the
    transfer is hidden for N > ..."; the integrated run): per config of the N sweep, `blocks` pinned host blocks
    through xc_correlate_pipelined (Algorithm 1) and through xc_integrate (+ int64 widening + D2H of the result), next to the
    copies alone and the X-engine alone.  compute_over_copy > 1 means PCIe is hidden behind the X-engine."""
    import torch
    import paper_1107_4264_b200 as xcb
    import xc_workloads as wl
    out = {}
    for name in names:
        w = wl.CONFIGS[name]
        blk = torch.from_numpy(wl.make_input(w))
        host = torch.empty((blocks,) + tuple(blk.shape), dtype=torch.int8).pin_memory()
        for k in range(blocks):
            host[k].copy_(blk)
        p = xcb.Plan(w.N, w.F, w.T)
        dev2, v = p.new_scratch(2), p.new_vis()
        v64 = torch.empty(p.vis_shape(), dtype=torch.int64, device="cuda")
        v64h = torch.empty(p.vis_shape(), dtype=torch.int64).pin_memory()

        def wall(fn, reps=3):
            fn()
            stream.synchronize()
            t0 = time.perf_counter()
            for _ in range(reps):
                fn()
                stream.synchronize()
            return (time.perf_counter() - t0) / reps
        tot = wall(lambda: p.correlate_pipelined(host, dev2, v, stream, s2))
        tot_i = wall(lambda: p.integrate(host, dev2, v, v64, stream, s2, vis64_host=v64h))
        dense = dev2[:4 * w.N * w.F * w.T]

        def copies():
            with torch.cuda.stream(stream):
                for k in range(blocks):
                    dense.copy_(host[k].view(-1), non_blocking=True)
        t_copy = wall(copies)
        xd = torch.from_numpy(wl.make_input(w)).cuda()
        t_comp = blocks * 1e-3 * _timed(lambda: p.correlate(xd, v, stream=stream), stream, 20, warm=3)
        out[name] = {"N": w.N, "F": w.F, "T": w.T, "blocks": blocks, "two_stream_ms": 1e3 * tot, "integrated_ms": 1e3 * tot_i,
                     "copy_alone_ms": 1e3 * t_copy, "compute_alone_ms": 1e3 * t_comp, "compute_over_copy": t_comp / t_copy,
                     "h2d_gbs": blocks * w.in_bytes / tot / 1e9, "tops": blocks * w.ops / tot / 1e12,
                     "tops_integrated": blocks * w.ops / tot_i / 1e12, "overlap_efficiency": max(t_copy, t_comp) / tot}
        p.close()
        del host, dev2, v, v64, v64h, xd, dense
        torch.cuda.empty_cache()
    return out


def fma_probe(iters=100000):
    """Pure-register FFMA2 / FFMA streams (bench_probe.cu beside this file, built on demand as libbench_probe.so): what the fp32 pipe delivers for the
    kernel's operand pattern with no memory traffic at all -- the practical ceiling next to which the kernel's rate is read."""
    import ctypes
    names = ["kernel statement order (ptxas schedule)", "scalar FFMA", "FFMA2, all operands re-used", "FFMA2 pair x pair",
             "FFMA2 a-stationary (pinned)", "FFMA2 b-stationary (pinned)"]
    try:
        L = ctypes.CDLL(build_probe())
        L.xc_probe_fma.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.POINTER(ctypes.c_double)]
        res = {}
        for mode, nm in enumerate(names):
            o = (ctypes.c_double * 4)()
            rc = L.xc_probe_fma(mode, iters, o)
            res[nm] = {"rc": rc} if rc else {"ms": o[0], "fma_per_clk_per_sm": o[1], "sm_mhz": o[2], "tflops": o[3]}
        res["how"] = "2 x 256 threads per SM, 64 accumulators per thread, no memory traffic; fma_per_clk_per_sm from the SM cycle counter (peak 128)"
        return res
    except Exception as e:  # noqa: BLE001
        return {"unavailable": repr(e)}


def trace_leg(workload, stream, debug_skip=0):
    """Pipeline timeline of CTA 0 of xc_i8_tc_kernel from the PROFILING build (libxc_profile.so, -DXC_PROFILE): clock64 stamps
    of the TMA producer, the MMA issuer and one epilogue warp, relative to the CTA's start, for the first tiles of `workload`.
    Returns per-role lists of cycle stamps and the derived per-stage periods."""
    import torch
    import paper_1107_4264_b200 as xcb
    import xc_workloads as wl
    from paper_1107_4264_b200 import build as xc_build
    xcb.load_library(xc_build.build(profile=True))
    w = wl.CONFIGS[workload]
    x = torch.from_numpy(wl.make_input(w)).cuda()
    p = xcb.Plan(w.N, w.F, w.T)
    p.set_option(xcb.OPT_DEBUG_SKIP, debug_skip)      # profiling build only: 1 no TMA loads, 2 no MMAs, 4 no stores, 8 stores to an 8 MB window
    v = p.new_vis()
    tr = torch.zeros(xcb.TRACE_WORDS, dtype=torch.int64, device="cuda")
    st = torch.zeros(xcb.TIMING_WORDS, dtype=torch.int64, device="cuda")
    with torch.cuda.stream(stream):
        for _ in range(5):
            p.correlate(x, v, stream=stream)
        stream.synchronize()
        p.set_trace(tr)
        p.set_timing_buffer(st)
        st[0] = 2 ** 62
        stream.synchronize()
        p.correlate(x, v, stream=stream)
        stream.synchronize()
    t = tr.cpu().view(3, 256, 4)
    s6 = st.tolist()
    c0 = s6[2]
    tile = p.tiles()[0][2]
    bk = 128 if tile == 64 else 256
    kb = (w.T + bk - 1) // bk
    n = min(256, 3 * kb)
    rel = lambda a: [int(q - c0) if q else None for q in a]
    mma = [rel(t[1, i].tolist()) for i in range(n) if t[1, i, 0]]
    prod = [rel(t[0, i, :3].tolist()) for i in range(n) if t[0, i, 0]]
    epi = [rel(t[2, i, :3].tolist()) for i in range(4) if t[2, i, 0]]
    per = [mma[i + 1][0] - mma[i][0] for i in range(len(mma) - 1)]
    out = {"workload": workload, "debug_skip": debug_skip, "tile_stations": tile, "stages_per_tile": kb, "samples_per_stage": bk,
           "kernel_ns": s6[1] - s6[0], "cta0_cycles": s6[4] - s6[2], "sm_mhz": (s6[4] - s6[2]) / max(1, s6[5] - s6[3]) * 1e3,
           "producer_first_issue_cycle": prod[0][2] if prod else None, "first_data_ready_cycle": mma[0][1] if mma else None,
           "mma_stage_period_cycles_tile0": per[:kb - 1], "mma_stage_period_cycles_tile1": per[kb:2 * kb - 1],
           "mma_stage_breakdown_first8 (wait_start, data_ready, mmas_issued, committed)": mma[:8],
           "epilogue_tiles (start, accumulator_ready, done)": epi,
           "ideal_tensor_cycles_per_stage": 512}
    p.close()
    xcb.load_library()
    return out


def only_leg(which, workload, stream):
    """Profiling aid for ncu captures: a few launches of one secondary kernel."""
    if which == "trace":
        import os
        return {"only": "trace", **trace_leg(workload, stream, int(os.environ.get("XC_TRACE_SKIP", "0")))}
    if which == "f32":
        return {"only": "f32", **f32_leg(stream, None, F=32, launches=3, kernel="cuda_cores")}
    if which == "f32tc":
        return {"only": "f32tc", **f32_leg(stream, None, F=128, launches=3, kernel="tc")}
    if which == "fengine":
        return {"only": "fengine", **fengine_leg(stream, workload, launches=3, with_fx=False)}
    if which == "noalloc":
        import torch
        import paper_1107_4264_b200 as xcb
        import xc_workloads as wl
        N, F, T = 128, 32, 1000                             # unpacked block 16.4 MB of the fixed 16.8 MB scratch
        xn = torch.from_numpy(wl.packed_i4(N, F, T, seed=7)).cuda()
        vn = torch.empty((F, N * (N + 1) // 2, 2, 2, 2), dtype=torch.int32, device="cuda")
        ms = _timed(lambda: xcb.correlate_i4_noalloc(xn, vn, stream=stream), stream, 3, warm=3)
        return {"only": "noalloc", "N": N, "F": F, "T": T, "ms_per_call": ms}
    raise ValueError(which)


def fengine_leg(stream, workload, launches=10, with_fx=True):
    """F-engine + corner turn and the FX chain; filled in once the library exports them."""
    import paper_1107_4264_b200 as xcb
    if not hasattr(xcb.Plan, "fengine"):
        return {"unavailable": "this build of the library has no F-engine"}
    return _fx_leg(stream, workload, launches, with_fx)


def extras(stream, clocks, sampler, peaks):
    import torch
    import paper_1107_4264_b200 as xcb
    import xc_workloads as wl
    out = {}
    # ---- S5: fp32-input variant on config 3's values (BASELINE.json configs[2]); ALU-bound ------------------
    out["f32"] = f32_leg(stream, clocks, peaks=peaks, sampler=sampler)
    out["f32_pitch"] = f32_pitch_leg(stream)

    # ---- N = 500 from a block with 128-byte-multiple rows (xc_set_in_pitch; what the F-engine / the host paths produce) ----
    w5 = wl.CONFIGS["cfg5_N500"]
    p5 = xcb.Plan(w5.N, w5.F, w5.T)
    pitch = p5.scratch_pitch
    xp = torch.zeros((w5.T, w5.F, pitch), dtype=torch.int8, device="cuda")
    xp[:, :, :4 * w5.N] = torch.from_numpy(wl.make_input(w5)).cuda().view(w5.T, w5.F, 4 * w5.N)
    p5.set_in_pitch(pitch)
    v5 = p5.new_vis()
    ms = _timed(lambda: p5.correlate(xp, v5, stream=stream), stream, 20)
    i8_burst = peaks["bf16_burst"] * 2.0
    out["N500_pitched"] = {"workload": f"cfg5_N500 values in a block with row pitch {pitch} B (xc_set_in_pitch) instead of 2000 B",
                           "back_to_back_ms": ms, "tops": w5.ops / (ms * 1e-3) / 1e12,
                           "frac_tensor_burst_peak": w5.ops / (ms * 1e-3) / 1e12 / i8_burst}
    # the same N through the host-buffer call: the H2D copy re-pitches, so end to end N = 500 pays no pitch penalty
    xh = torch.from_numpy(wl.make_input(w5)).pin_memory()
    vh = torch.empty(p5.vis_shape(), dtype=torch.int32).pin_memory()
    p5.set_in_pitch(0)
    scr = p5.new_scratch()
    p5.correlate_host(xh, vh, scr, v5, stream=stream)
    t0 = time.perf_counter()
    for _ in range(3):
        p5.correlate_host(xh, vh, scr, v5, stream=stream)
    e = (time.perf_counter() - t0) / 3
    out["N500_pitched"].update({"e2e_ms": 1e3 * e, "e2e_tops": w5.ops / e / 1e12, "e2e_h2d_gbs": w5.in_bytes / e / 1e9})
    p5.close()
    del xp, v5, xh, vh, scr
    torch.cuda.empty_cache()

    # ---- 4-bit samples on config 2's shape ---------------------------------
    w2 = wl.CONFIGS["cfg2"]
    x4h = torch.from_numpy(wl.packed_i4(w2.N, w2.F, w2.T, seed=2002)).pin_memory()
    x4d = x4h.cuda()
    p4 = xcb.Plan(w2.N, w2.F, w2.T)
    v4 = p4.new_vis()
    v4h = torch.empty(p4.vis_shape(), dtype=torch.int32).pin_memory()
    ms4 = _timed(lambda: p4.correlate_i4(x4d, v4, stream=stream), stream, 20)
    p4.correlate_host_i4(x4h, v4h, x4d, v4, stream=stream)
    t0 = time.perf_counter()
    for _ in range(5):
        p4.correlate_host_i4(x4h, v4h, x4d, v4, stream=stream)
    e4 = (time.perf_counter() - t0) / 5
    out["i4"] = {"workload": "config 2's shape with 4-bit complex samples (uniform nibbles), xc_correlate_i4 / xc_correlate_host_i4",
                 "device_ms": ms4, "tops": w2.ops / (ms4 * 1e-3) / 1e12, "launches_per_step": 2,
                 "e2e_ms": 1e3 * e4, "e2e_tops": w2.ops / e4 / 1e12, "h2d_bytes_per_step": w2.in_bytes // 2,
                 "d2h_bytes_per_step": w2.vis_bytes}
    p4.close()
    del x4h, x4d, v4, v4h
    torch.cuda.empty_cache()
    # the no-allocation entry point next to the planned call on a block that fills its fixed 16 MiB scratch (N = 128, F = 32,
    # T = 1000: 16.4 MB unpacked): same two launches, the scratch is a static device array instead of a cudaMalloc'ed workspace
    wn = wl.Workload("i4_noalloc", 128, 32, 1000, "uniform", 0.0, 7)
    xn = torch.from_numpy(wl.packed_i4(wn.N, wn.F, wn.T, seed=7)).cuda()
    pn = xcb.Plan(wn.N, wn.F, wn.T)
    vn = pn.new_vis()
    ms_plan = _timed(lambda: pn.correlate_i4(xn, vn, stream=stream), stream, 50, warm=5)
    ms_na = _timed(lambda: xcb.correlate_i4_noalloc(xn, vn, stream=stream), stream, 50, warm=5)
    out["i4_noalloc"] = {"workload": "N=128, F=32, T=1000, 4-bit samples (unpacked block 16.4 MB of the fixed 16.8 MB scratch)",
                         "xc_correlate_i4_ms": ms_plan, "xc_correlate_i4_noalloc_ms": ms_na,
                         "tops_noalloc": wn.ops / (ms_na * 1e-3) / 1e12, "scratch_bytes": xcb.NOALLOC_SCRATCH_BYTES}
    pn.close()
    del xn, vn
    torch.cuda.empty_cache()

    # ---- S6: two-stream run of config 5: 8 host blocks (the same seeded block 8 times: only the timing matters here;
    # parity of the 8-distinct-block run is tests/test_xc_gpu.py::test_cfg5_two_stream_eight_blocks) -------------------
    w5 = wl.CONFIGS["cfg5_N1024"]
    blk = torch.from_numpy(wl.make_input(w5))
    host = torch.empty((8,) + tuple(blk.shape), dtype=torch.int8).pin_memory()
    for k in range(8):
        host[k].copy_(blk)
    p5 = xcb.Plan(w5.N, w5.F, w5.T)
    dev2 = p5.new_scratch(2)
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
        dev2[:p5.in_bytes].copy_(host[k].view(-1), non_blocking=True)
    torch.cuda.synchronize()
    t_copy = time.perf_counter() - t0
    xk = dev2[:p5.in_bytes].view(w5.T, w5.F, w5.N, 2, 2)
    t_comp = 8e-3 * _timed(lambda: p5.correlate(xk, v5, stream=stream), stream, 5, warm=2)
    out["two_stream"] = {"workload": "cfg5_N1024 x 8 pinned host blocks, xc_correlate_pipelined (Algorithm 1)",
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
    out["integrated"] = {"workload": "cfg5_N1024 x 8 pinned host blocks (16384 samples), xc_integrate: H2D pipeline, "
                                     "X-engine, int64 widening, D2H of the int64 result",
                         "total_ms": 1e3 * tot_i, "tops": 8 * w5.ops / tot_i / 1e12,
                         "h2d_bytes": 8 * w5.in_bytes, "d2h_bytes": 2 * w5.vis_bytes,
                         "pcie_floor_ms": 1e3 * (t_copy + 2 * w5.vis_bytes / (8 * w5.in_bytes / t_copy))}
    del v64, v64h
    p5.close()
    del host, dev2, v5
    torch.cuda.empty_cache()
    out["two_stream_vs_N"] = two_stream_vs_n(stream, s2)

    # ---- T-split of the single-CTA tile (small N, long integration), off / on / what AUTO picks -----------
    out["t_split"] = t_split_leg(stream)

    # ---- small N: what a launch costs with no host in the loop (CUDA-graph replay of back-to-back launches) --------------------
    out["graph_replay"] = graph_replay_leg()

    # ---- F-engine + corner turn, and the FX chain ----------------------------------------------------------
    out["fx"] = fengine_leg(stream, "cfg3")
    return out


def graph_replay_leg(n=50):
    """Config 5's latency-bound sizes (N = 32, 64, 100) and config 1: n xc_correlate launches captured into one CUDA graph (the
    kernels are plain stream work launched with programmatic stream serialization) and replayed -- microseconds per launch with
    the host out of the loop, next to the same n calls issued from Python through the C ABI."""
    import torch
    import paper_1107_4264_b200 as xcb
    import xc_workloads as wl
    res = {}
    for name in ("cfg1", "cfg5_N32", "cfg5_N64", "cfg5_N100"):
        w = wl.CONFIGS[name]
        x = torch.from_numpy(wl.make_input(w)).cuda()
        p = xcb.Plan(w.N, w.F, w.T)
        v = p.new_vis()
        p.correlate(x, v)                                    # plan's device state exists before the capture
        s = torch.cuda.Stream()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            cur = torch.cuda.current_stream()
            for _ in range(n):
                p.correlate(x, v, stream=cur)
        torch.cuda.synchronize()
        for _ in range(3):
            g.replay()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        for _ in range(5):
            g.replay()
        e1.record()
        torch.cuda.synchronize()
        us_graph = e0.elapsed_time(e1) * 1e3 / (5 * n)
        us_calls = _timed(lambda: p.correlate(x, v, stream=s), s, 5 * n) * 1e3
        floor_us = (w.in_bytes + w.vis_bytes) / 6.5e12 * 1e6
        res[name] = {"us_per_launch_graph": us_graph, "us_per_launch_calls": us_calls, "hbm_floor_us": floor_us,
                     "tops_graph": w.ops / (us_graph * 1e-6) / 1e12}
        p.close()
        del g, x, v
    return res


def t_split_leg(stream):
    """The paper's small-N future work: one 128 x 128 tile per channel leaves SMs idle and walks T serially;
    the T-split halves that walk over a cluster of 2.  Two shapes: config 5's N = 32 (T = 2048, where the hand-over costs more
    than it saves and AUTO keeps it off) and a long integration N = 32, F = 32, T = 16384 (where AUTO turns it on)."""
    import torch
    import paper_1107_4264_b200 as xcb
    import xc_workloads as wl
    from bench import kernel_durations
    res = {}
    for name, (N, F, T) in {"cfg5_N32 (F=64, T=2048)": (32, 64, 2048), "long integration (N=32, F=32, T=16384)": (32, 32, 16384)}.items():
        x = torch.from_numpy(wl.gaussian(N, F, T, seed=77, sigma=4.0)).cuda()
        row = {}
        for label, ts in (("off", 1), ("on", 2), ("auto", 0)):
            p = xcb.Plan(N, F, T)
            p.set_option(xcb.OPT_TSPLIT, ts)
            v = p.new_vis()
            km, em, _ = kernel_durations(p, x, v, stream, 10)
            row[label] = {"kernel_us": km * 1e3, "t_split_used": p.t_split}
            p.close()
        res[name] = row
    return res


def _fx_leg(stream, workload, launches, with_fx):
    """F-engine (+ FX chain) on the shape of `workload`: volt int8 [N][2][T*F][2] -> cube -> vis.  Roofline: the F-engine
    moves 4NFT bytes in and 4NFT bytes out (algorithmic; HBM) and needs about 5 F log2 F real operations per spectrum on
    the fp32 CUDA cores (non-FMA: 128 lanes / clk / SM) -- whichever takes longer bounds it."""
    import numpy as np
    import torch
    import paper_1107_4264_b200 as xcb
    import xc_workloads as wl
    from bench import load_peaks
    w = wl.CONFIGS[workload]
    N, F, T = w.N, w.F, w.T
    volt = torch.from_numpy(wl.voltages(N, F, T, seed=w.seed + 500)).cuda()
    scale = wl.fengine_scale(F)
    p = xcb.Plan(N, F, T)
    cube = p.new_cube()
    ms = _timed(lambda: p.fengine(volt, scale, cube, stream=stream), stream, launches)
    peaks = load_peaks()
    alg_bytes = 8.0 * N * F * T
    flops = 5.0 * F * max(np.log2(F), 1.0) * 2 * N * T
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    alu_peak = sms * 128 * 1965e6 / 1e12                     # T non-FMA fp32 operations / s at clocks.max.sm
    t_hbm, t_alu = alg_bytes / (peaks["hbm_gbs"] * 1e9), flops / (alu_peak * 1e12)
    gbs = alg_bytes / (ms * 1e-3) / 1e9
    out = {"workload": f"{workload} shape: N={N}, F={F}-point transforms, T={T} time blocks, int8 complex voltages (Gaussian sigma 16 + 2 tones)",
           "fengine_ms": ms, "bound": "hbm" if t_hbm >= t_alu else "alu", "achieved_gbs": gbs, "hbm_peak_gbs": peaks["hbm_gbs"],
           "frac_hbm": gbs / peaks["hbm_gbs"], "algorithmic_bytes": alg_bytes, "fft_flops_5NlogN": flops,
           "achieved_tflops": flops / (ms * 1e-3) / 1e12, "alu_peak_tops_non_fma": alu_peak,
           "frac_alu": flops / (ms * 1e-3) / 1e12 / alu_peak, "roof_ms": 1e3 * max(t_hbm, t_alu)}
    if with_fx:
        vis = p.new_vis()
        ms_fx = _timed(lambda: p.fx(volt, scale, cube, vis, stream=stream), stream, launches)
        p.set_in_pitch(p.scratch_pitch)
        ms_x = _timed(lambda: p.correlate(cube, vis, stream=stream), stream, launches)
        out.update({"fx_ms": ms_fx, "xengine_alone_ms": ms_x, "fx_tops": w.ops / (ms_fx * 1e-3) / 1e12,
                    "launches_per_fx": 2})
    p.close()
    del volt, cube
    torch.cuda.empty_cache()
    return out
