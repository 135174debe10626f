// xc_f32.cuh -- the fp32-input X-engine on the CUDA cores.
//
// The paper's own arithmetic (a station pair costs 16 fp32 FMAs per sample) and its
// own tiling idea: a register tile of station pairs per thread, fed
// from a shared-memory tile of input vectors that the whole block loads cooperatively, filled in
// only at the innermost level.  Re-sized for sm_100a: 2 x 4 station pairs per thread (64 fp32
// accumulators; the paper's Fermi kernel 11 used 2 x 2), a 32 x 64 station tile per 256-thread
// block, and a 3-stage cp.async ring in place of the paper's double-buffered texture loads.
// The 16 FMAs of a station pair are issued as 8 packed FFMA2 (fma.rn.f32x2) on (re, im) pairs.
// Only tiles that intersect i <= j are launched.  The paper lets threads above
// the diagonal compute without writing (its software-cache choice); here each warp
// owns a 16 x 16-station block and skips the arithmetic when the whole block is above the diagonal,
// which cuts the paper's wasted work from 32 x 64 to 16 x 16 granularity.
// Measured variants (B200, config 3 values): stages of 8 / 16 / 32 samples x 2-4 stages and 1 vs 2
// blocks per SM -- 16 x 3 x 2 is the fastest.  Round 2 also measured a ring synchronised by per-stage full / empty
// mbarriers (cp.async.mbarrier.arrive.noinc, refill lagging two iterations) in place of the block-wide barrier per stage,
// because ncu attributes 17 % of the warp cycles to that barrier: 11.3-11.8 ms against 10.7 ms -- the waiting only moves
// to the mbarriers (the FMA pipe, not the barrier, is what the warps queue for), so the simple ring stays.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace xc {

#ifndef XC_F32_TI
#define XC_F32_TI 2
#endif
constexpr int F32_TI = XC_F32_TI;            // stations per thread on the i side (x 4 on the j side)
constexpr int F32_LI = 16 / F32_TI;          // lanes of a warp along i; the warp's block is 16 stations tall
constexpr int F32_LJ = 32 / F32_LI;          // lanes along j
constexpr int F32_WBJ = 4 * F32_LJ;          // stations of a warp's block along j
constexpr int F32_SI = 16 * F32_TI;          // stations per tile on the i side
constexpr int F32_SJ = 64;                   // stations per tile on the j side
constexpr int F32_WI = F32_SI / 16;          // warps along i
#ifndef XC_F32_BK
#define XC_F32_BK 16
#endif
#ifndef XC_F32_STAGES
#define XC_F32_STAGES 3
#endif
#ifndef XC_F32_MINB
#define XC_F32_MINB (XC_F32_TI == 2 ? 2 : 1)
#endif
constexpr int F32_BK = XC_F32_BK;       // samples per ring stage
constexpr int F32_STAGES = XC_F32_STAGES;
constexpr int F32_THREADS = 256;
constexpr int F32_STAGE_F4 = F32_BK * (F32_SI + F32_SJ);             // float4 per stage
constexpr int F32_SMEM_BYTES = F32_STAGES * F32_STAGE_F4 * 16;       // 72 KB

struct F32Params {
    int N, F, T;
    int tiles_per_f;
    long long NB;
    const uint32_t* tiles;  // device: bi | (bj << 16), bi in 32-station blocks, bj in 64-station blocks
    const float4* in;       // one float4 per (t, f, station): (p0.re, p0.im, p1.re, p1.im)
    float* vis;
    int accumulate;
};

__device__ __forceinline__ void cp_async16(uint32_t dst_smem, const void* src, int src_bytes) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst_smem), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
    asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory");
}

// One station i (a = both polarisations) against the thread's four stations j: 32 packed FMAs = 64 of the paper's FMAs
// (16 per station pair).  acc[n][pi*2+pj] = (re, im) += a_{pi} * conj(b_{n,pj}); per output the order is
//     re = fma(a.im, b.im, fma(a.re, b.re, re)),  im = fma(-a.re, b.im, fma(a.im, b.re, im)),
// i.e. (re, im) += (a.re, a.im) * b.re, then (re, im) += (a.im, -a.re) * b.im.
// The statement order is pinned (asm volatile) and "a-stationary": eight consecutive FFMA2 share their 64-bit a operand
// and differ in the scalar b and the accumulator.  A pure-register probe of this operand pattern (csrc/xc_probe.cu, bench.py
// extras.f32.fma_issue_probe) measured 66.3 TFLOPS for this order against 58.1 for the order ptxas picks by itself and 61.4
// for the b-stationary one: the instruction reads 5 register words (2 + 1 + 2) per two pipe cycles, and holding the pair
// operand in the re-use latch is what fits the register-file bandwidth.
__device__ __forceinline__ float2 ffma2_pinned(float2 a, float bs, float2 c) {
    unsigned long long ua, ub, uc, ud;
    asm("mov.b64 %0, {%1, %2};" : "=l"(ua) : "f"(a.x), "f"(a.y));
    asm("mov.b64 %0, {%1, %2};" : "=l"(ub) : "f"(bs), "f"(bs));
    asm("mov.b64 %0, {%1, %2};" : "=l"(uc) : "f"(c.x), "f"(c.y));
    asm volatile("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(ud) : "l"(ua), "l"(ub), "l"(uc));
    float2 d;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(d.x), "=f"(d.y) : "l"(ud));
    return d;
}
__device__ __forceinline__ void cmac_row(float2 (&acc)[4][4], const float4& a, const float4& b0, const float4& b1,
                                         const float4& b2, const float4& b3) {
    const float bre[8] = {b0.x, b0.z, b1.x, b1.z, b2.x, b2.z, b3.x, b3.z};      // b_{n,pj}.re, index 2n + pj
    const float bim[8] = {b0.y, b0.w, b1.y, b1.w, b2.y, b2.w, b3.y, b3.w};
#pragma unroll
    for (int pi = 0; pi < 2; ++pi) {
        const float2 ap = pi ? make_float2(a.z, a.w) : make_float2(a.x, a.y);
        const float2 as = pi ? make_float2(a.w, -a.z) : make_float2(a.y, -a.x);
#pragma unroll
        for (int k = 0; k < 8; ++k) acc[k >> 1][pi * 2 + (k & 1)] = ffma2_pinned(ap, bre[k], acc[k >> 1][pi * 2 + (k & 1)]);
#pragma unroll
        for (int k = 0; k < 8; ++k) acc[k >> 1][pi * 2 + (k & 1)] = ffma2_pinned(as, bim[k], acc[k >> 1][pi * 2 + (k & 1)]);
    }
}

__global__ void __launch_bounds__(F32_THREADS, XC_F32_MINB) xc_f32_kernel(const F32Params p) {
    extern __shared__ __align__(16) float4 smem_f4[];
    const int tid = threadIdx.x;
    // Each warp owns a 16 x 16-station block of the tile (2 blocks on the i side x 4 on the j side), its lanes an
    // 8 (i) x 4 (j) grid, each lane 2 x 4 station pairs.  A warp whose whole block lies above the diagonal (every
    // i > j) or beyond N skips the arithmetic -- it still loads and synchronises -- so diagonal tiles cost what
    // they store at 16-station granularity, and the co-resident CTA's warps take the freed issue slots.
    const int warp = tid >> 5, lane = tid & 31;
    const int ti = 16 * (warp % F32_WI) + (lane % F32_LI);       // stations i0 + ti + F32_LI a, a < F32_TI
    const int tj = F32_WBJ * (warp / F32_WI) + (lane / F32_LI);  // stations j0 + tj + F32_LJ n, n = 0..3

    const long long w = blockIdx.x;
    const int f = static_cast<int>(w / p.tiles_per_f);
    const uint32_t tb = __ldg(p.tiles + static_cast<int>(w % p.tiles_per_f));
    const int i0 = static_cast<int>(tb & 0xFFFFu) * F32_SI;
    const int j0 = static_cast<int>(tb >> 16) * F32_SJ;

    const uint32_t smem0 = static_cast<uint32_t>(__cvta_generic_to_shared(smem_f4));
    const int KB = (p.T + F32_BK - 1) / F32_BK;

    // Cooperative load of one stage: F32_BK rows of (32 + 64) float4; zero fill outside [0,T) x [0,N).
    auto load_stage = [&](int kb, int stage) {
        const uint32_t sbase = smem0 + static_cast<uint32_t>(stage * F32_STAGE_F4 * 16);
#pragma unroll
        for (int r = 0; r < F32_STAGE_F4 / F32_THREADS; ++r) {
            const int idx = tid + r * F32_THREADS;
            const int k = idx / (F32_SI + F32_SJ);
            const int c = idx - k * (F32_SI + F32_SJ);
            const int s = (c < F32_SI) ? (i0 + c) : (j0 + c - F32_SI);
            const int t = kb * F32_BK + k;
            const bool ok = (t < p.T) && (s < p.N) && (kb < KB);
            const float4* src = ok ? (p.in + (static_cast<long long>(t) * p.F + f) * p.N + s) : p.in;
            cp_async16(sbase + static_cast<uint32_t>(idx * 16), src, ok ? 16 : 0);
        }
    };

    float2 acc[F32_TI][4][4];
#pragma unroll
    for (int a = 0; a < F32_TI; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b)
#pragma unroll
            for (int c = 0; c < 4; ++c) acc[a][b][c] = make_float2(0.f, 0.f);

#pragma unroll
    for (int s = 0; s < F32_STAGES - 1; ++s) {
        load_stage(s, s);
        cp_async_commit();
    }

    // warp-uniform: does this warp's 16 x 16 block hold any stored pair (i <= j < N)?
    const int wi0 = i0 + 16 * (warp % F32_WI), wj0 = j0 + F32_WBJ * (warp / F32_WI);
    const bool active = (wi0 <= wj0 + F32_WBJ - 1) && (wi0 < p.N) && (wj0 < p.N);

    for (int kb = 0; kb < KB; ++kb) {
        cp_async_wait<F32_STAGES - 2>();
        __syncthreads();
        load_stage(kb + F32_STAGES - 1, (kb + F32_STAGES - 1) % F32_STAGES);
        cp_async_commit();
        if (!active) continue;
        const float4* sA = smem_f4 + (kb % F32_STAGES) * F32_STAGE_F4;
#pragma unroll
        for (int k = 0; k < F32_BK; ++k) {
            const float4* row = sA + k * (F32_SI + F32_SJ);
            const float4 b0 = row[F32_SI + tj], b1 = row[F32_SI + tj + F32_LJ];
            const float4 b2 = row[F32_SI + tj + 2 * F32_LJ], b3 = row[F32_SI + tj + 3 * F32_LJ];
#pragma unroll
            for (int a = 0; a < F32_TI; ++a) cmac_row(acc[a], row[ti + F32_LI * a], b0, b1, b2, b3);
        }
    }
    cp_async_wait<0>();

    float* visf = p.vis + static_cast<long long>(f) * p.NB * 8;
#pragma unroll
    for (int b = 0; b < 4; ++b) {
        const int j = j0 + tj + F32_LJ * b;
#pragma unroll
        for (int a = 0; a < F32_TI; ++a) {
            const int i = i0 + ti + F32_LI * a;
            if (i <= j && j < p.N) {
                float4* dst = reinterpret_cast<float4*>(visf + (static_cast<long long>(j) * (j + 1) / 2 + i) * 8);
                float4 lo = make_float4(acc[a][b][0].x, acc[a][b][0].y, acc[a][b][1].x, acc[a][b][1].y);
                float4 hi = make_float4(acc[a][b][2].x, acc[a][b][2].y, acc[a][b][3].x, acc[a][b][3].y);
                if (p.accumulate) {
                    const float4 o0 = dst[0], o1 = dst[1];
                    lo.x += o0.x; lo.y += o0.y; lo.z += o0.z; lo.w += o0.w;
                    hi.x += o1.x; hi.y += o1.y; hi.z += o1.z; hi.w += o1.w;
                }
                dst[0] = lo;
                dst[1] = hi;
            }
        }
    }
}

}  // namespace xc
