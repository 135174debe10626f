// bench_probe.cu -- measurement aid, not on the product path: pure-register FFMA2 / FFMA issue-rate probes that give the
// fp32 X-engine (xc_f32.cuh) its practical ceiling.  Built as libbench_probe.so by bench_legs.build_probe()
// on demand; bench.py's f32 leg calls xc_probe_fma() and reports the numbers next to the kernel's own rate, so that the
// "ceiling" quoted in DESIGN.md is something the tracked bench measures in the same run (round 1 quoted an untracked probe).
//
// Every mode runs 2 x 256 threads per SM (the kernel's occupancy) doing 64 packed (or 128 scalar) FMAs per thread and
// iteration on 64 accumulators with no memory traffic, and reports FMA / clk / SM from the SM cycle counter (so the result
// does not depend on where the power management puts the clock) as well as the wall-clock TFLOPS.
//   0  the kernel's own statement sequence (cmac4 on a 2 x 4 station-pair tile), scheduled by ptxas
//   1  the same arithmetic with scalar fmaf
//   2  FFMA2 with one and the same multiplicand pair for all 64 accumulators (upper bound: every operand re-used)
//   3  FFMA2 pair x pair with distinct 64-bit multiplicands (no scalar broadcast)
//   4  the kernel's operands, order pinned: for each of the 4 "a" pairs, all 16 "b" scalars      (a stationary)
//   5  the kernel's operands, order pinned: for each of the 16 "b" scalars, all 4 "a" pairs      (b stationary)
#include <cstdint>
#include <cuda_runtime.h>

namespace {

__device__ __forceinline__ float2 ffma2(float2 a, float2 b, float2 c) {
    unsigned long long ua, ub, uc, ud;
    asm("mov.b64 %0, {%1, %2};" : "=l"(ua) : "f"(a.x), "f"(a.y));
    asm("mov.b64 %0, {%1, %2};" : "=l"(ub) : "f"(b.x), "f"(b.y));
    asm("mov.b64 %0, {%1, %2};" : "=l"(uc) : "f"(c.x), "f"(c.y));
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(ud) : "l"(ua), "l"(ub), "l"(uc));
    float2 d;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(d.x), "=f"(d.y) : "l"(ud));
    return d;
}
// same, but the instruction keeps its place in the statement order (asm volatile)
__device__ __forceinline__ float2 ffma2_pinned(float2 a, float2 b, float2 c) {
    unsigned long long ua, ub, uc, ud;
    asm("mov.b64 %0, {%1, %2};" : "=l"(ua) : "f"(a.x), "f"(a.y));
    asm("mov.b64 %0, {%1, %2};" : "=l"(ub) : "f"(b.x), "f"(b.y));
    asm("mov.b64 %0, {%1, %2};" : "=l"(uc) : "f"(c.x), "f"(c.y));
    asm volatile("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(ud) : "l"(ua), "l"(ub), "l"(uc));
    float2 d;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(d.x), "=f"(d.y) : "l"(ud));
    return d;
}
__device__ __forceinline__ void cmac4(float2 (&acc)[4], const float4& a, const float4& b) {
    const float2 a0 = make_float2(a.x, a.y), a0s = make_float2(a.y, -a.x);
    const float2 a1 = make_float2(a.z, a.w), a1s = make_float2(a.w, -a.z);
    acc[0] = ffma2(a0, make_float2(b.x, b.x), acc[0]); acc[0] = ffma2(a0s, make_float2(b.y, b.y), acc[0]);
    acc[1] = ffma2(a0, make_float2(b.z, b.z), acc[1]); acc[1] = ffma2(a0s, make_float2(b.w, b.w), acc[1]);
    acc[2] = ffma2(a1, make_float2(b.x, b.x), acc[2]); acc[2] = ffma2(a1s, make_float2(b.y, b.y), acc[2]);
    acc[3] = ffma2(a1, make_float2(b.z, b.z), acc[3]); acc[3] = ffma2(a1s, make_float2(b.w, b.w), acc[3]);
}

template <int MODE>
__global__ void __launch_bounds__(256, 2) probe_kernel(const float4* in, float* out, int iters, unsigned long long* stamps) {
    float4 a0 = in[threadIdx.x], a1 = in[threadIdx.x + 256], b0 = in[threadIdx.x + 512], b1 = in[threadIdx.x + 768],
           b2 = in[threadIdx.x + 1024], b3 = in[threadIdx.x + 1280];
    float2 acc[2][4][4];
#pragma unroll
    for (int a = 0; a < 2; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b)
#pragma unroll
            for (int c = 0; c < 4; ++c) acc[a][b][c] = make_float2(0.f, 0.f);
    float sc[64];
    if (MODE == 1) {
#pragma unroll
        for (int k = 0; k < 64; ++k) sc[k] = 0.f;
    }
    unsigned long long c0 = 0, g0 = 0;
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        c0 = clock64();
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g0));
    }
    for (int it = 0; it < iters; ++it) {
        if (MODE == 0) {
            cmac4(acc[0][0], a0, b0); cmac4(acc[0][1], a0, b1); cmac4(acc[0][2], a0, b2); cmac4(acc[0][3], a0, b3);
            cmac4(acc[1][0], a1, b0); cmac4(acc[1][1], a1, b1); cmac4(acc[1][2], a1, b2); cmac4(acc[1][3], a1, b3);
        } else if (MODE == 1) {
            const float av[8] = {a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w};
            const float bv[16] = {b0.x, b0.y, b0.z, b0.w, b1.x, b1.y, b1.z, b1.w, b2.x, b2.y, b2.z, b2.w, b3.x, b3.y, b3.z, b3.w};
#pragma unroll
            for (int i = 0; i < 8; ++i)
#pragma unroll
                for (int j = 0; j < 16; j += 2) sc[i * 8 + j / 2] = fmaf(av[i], bv[j], fmaf(av[i], bv[j + 1], sc[i * 8 + j / 2]));
        } else if (MODE == 2) {
            const float2 xa = make_float2(a0.x, a0.y), yb = make_float2(b0.x, b0.x);
#pragma unroll
            for (int r = 0; r < 2; ++r)
#pragma unroll
                for (int a = 0; a < 2; ++a)
#pragma unroll
                    for (int b = 0; b < 4; ++b)
#pragma unroll
                        for (int c = 0; c < 4; ++c) acc[a][b][c] = ffma2(xa, yb, acc[a][b][c]);
        } else if (MODE == 3) {
            const float2 xa = make_float2(a0.x, a0.y), yb = make_float2(b0.x, b0.y);
            const float2 xc = make_float2(a1.x, a1.y), yd = make_float2(b1.x, b1.y);
#pragma unroll
            for (int a = 0; a < 2; ++a)
#pragma unroll
                for (int b = 0; b < 4; ++b)
#pragma unroll
                    for (int c = 0; c < 4; ++c) {
                        acc[a][b][c] = ffma2(xa, yb, acc[a][b][c]);
                        acc[a][b][c] = ffma2(xc, yd, acc[a][b][c]);
                    }
        } else {
            // the kernel's operands: 4 "a" pairs (a, a rotated) x 16 "b" scalars -> 64 accumulators (acc[ia/2][jb/4][..])
            const float2 ap[4] = {make_float2(a0.x, a0.y), make_float2(a0.z, a0.w), make_float2(a1.x, a1.y), make_float2(a1.z, a1.w)};
            const float2 as[4] = {make_float2(a0.y, -a0.x), make_float2(a0.w, -a0.z), make_float2(a1.y, -a1.x), make_float2(a1.w, -a1.z)};
            const float bv[16] = {b0.x, b0.y, b0.z, b0.w, b1.x, b1.y, b1.z, b1.w, b2.x, b2.y, b2.z, b2.w, b3.x, b3.y, b3.z, b3.w};
            if (MODE == 4) {
#pragma unroll
                for (int ia = 0; ia < 4; ++ia)
#pragma unroll
                    for (int half = 0; half < 2; ++half)
#pragma unroll
                        for (int jb = 0; jb < 8; ++jb) {     // b scalar 2*jb + half: the re (half 0) or im (half 1) part
                            float2& d = acc[ia >> 1][jb >> 1][(ia & 1) * 2 + (jb & 1)];
                            d = ffma2_pinned(half ? as[ia] : ap[ia], make_float2(bv[2 * jb + half], bv[2 * jb + half]), d);
                        }
            } else {
#pragma unroll
                for (int half = 0; half < 2; ++half)
#pragma unroll
                    for (int jb = 0; jb < 8; ++jb)
#pragma unroll
                        for (int ia = 0; ia < 4; ++ia) {
                            float2& d = acc[ia >> 1][jb >> 1][(ia & 1) * 2 + (jb & 1)];
                            d = ffma2_pinned(half ? as[ia] : ap[ia], make_float2(bv[2 * jb + half], bv[2 * jb + half]), d);
                        }
            }
        }
        a0.x += 1e-9f;      // perturb operands so nothing is hoisted out of the loop
        b3.w += 1e-9f;
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        unsigned long long g1;
        const unsigned long long c1 = clock64();
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g1));
        stamps[0] = c1 - c0;
        stamps[1] = g1 - g0;
    }
    float s = 0.f;
#pragma unroll
    for (int a = 0; a < 2; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b)
#pragma unroll
            for (int c = 0; c < 4; ++c) s += acc[a][b][c].x + acc[a][b][c].y;
    if (MODE == 1) {
#pragma unroll
        for (int k = 0; k < 64; ++k) s += sc[k];
    }
    out[blockIdx.x * 256 + threadIdx.x] = s;
}

template <int MODE>
void launch(int grid, const float4* in, float* out, int iters, unsigned long long* stamps, cudaStream_t st) {
    probe_kernel<MODE><<<grid, 256, 0, st>>>(in, out, iters, stamps);
}

}  // namespace

extern "C" {

// Runs probe `mode` (0..5) with `iters` iterations per thread on 2 CTAs of 256 threads per SM.  Results:
//   out4[0] = kernel time in ms (CUDA events), out4[1] = FMA per clock per SM (CTA 0's cycle counter; 128 = the fp32 pipe's
//   peak), out4[2] = SM clock in MHz during the kernel, out4[3] = TFLOPS (2 flops per FMA, wall clock).  Returns 0 or a
//   cudaError_t.  Synchronises the device.
int xc_probe_fma(int mode, int iters, double* out4) {
    if (mode < 0 || mode > 5 || iters < 1 || !out4) return -1;
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return static_cast<int>(e);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int grid = 2 * sms;
    float4* in = nullptr;
    float* out = nullptr;
    unsigned long long* stamps = nullptr;
    if ((e = cudaMalloc(&in, 2048 * sizeof(float4))) != cudaSuccess) return static_cast<int>(e);
    cudaMemset(in, 0, 2048 * sizeof(float4));
    cudaMalloc(&out, static_cast<size_t>(grid) * 256 * sizeof(float));
    cudaMalloc(&stamps, 2 * sizeof(unsigned long long));
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    float ms = 0.f;
    for (int rep = 0; rep < 2; ++rep) {       // the first run warms up
        cudaEventRecord(e0, 0);
        switch (mode) {
            case 0: launch<0>(grid, in, out, iters, stamps, 0); break;
            case 1: launch<1>(grid, in, out, iters, stamps, 0); break;
            case 2: launch<2>(grid, in, out, iters, stamps, 0); break;
            case 3: launch<3>(grid, in, out, iters, stamps, 0); break;
            case 4: launch<4>(grid, in, out, iters, stamps, 0); break;
            default: launch<5>(grid, in, out, iters, stamps, 0); break;
        }
        cudaEventRecord(e1, 0);
        e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) break;
        cudaEventElapsedTime(&ms, e0, e1);
    }
    unsigned long long h[2] = {0, 0};
    if (e == cudaSuccess) e = cudaMemcpy(h, stamps, sizeof h, cudaMemcpyDeviceToHost);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(in);
    cudaFree(out);
    cudaFree(stamps);
    if (e != cudaSuccess) return static_cast<int>(e);
    const double fma_per_thread = 128.0 * iters;                  // 64 FFMA2 = 128 scalar FMA per iteration in every mode
    out4[0] = ms;
    out4[2] = h[1] ? static_cast<double>(h[0]) / static_cast<double>(h[1]) * 1e3 : 0.0;
    // whole-kernel FMA rate over the clock CTA 0 saw (the two CTAs of an SM do not share the pipe evenly -- the older CTA's
    // warps win the arbitration and finish in half the kernel's time -- so CTA 0's own duration is not the SM's)
    out4[1] = out4[2] > 0 ? grid * 256.0 * fma_per_thread / (ms * 1e-3) / sms / (out4[2] * 1e6) : 0.0;
    out4[3] = 2.0 * grid * 256.0 * fma_per_thread / (ms * 1e-3) / 1e12;
    return 0;
}

}  // extern "C"
