// xc_i8_tc.cuh -- the int8 X-engine on tcgen05 tensor cores (sm_100a).
//
// What it computes (Eq. 4): V_f[(i,pi),(j,pj)] = sum_t x_i,pi conj(x_j,pj), i <= j.
// How: per channel f the input is a real matrix Z[m][t], m = (station, pol, re/im) = 4N rows of
// int8; the real Gram matrix G = Z Z^T is a dense int8 x int8 -> int32 contraction over t, and
//      Re V = G[(i,pi,re),(j,pj,re)] + G[(i,pi,im),(j,pj,im)]
//      Im V = G[(i,pi,im),(j,pj,re)] - G[(i,pi,re),(j,pj,im)]
// (no operand is negated: -128 has no int8 negative, SURVEY 8(c) reading 6).
//
// The paper's multi-level tiling (matrix filled in only at the innermost
// level, outer levels hold input vectors) maps to: TMEM accumulator tile (innermost) <- smem
// operand ring filled by TMA <- L2 (a channel's input, <= 8 MB, is shared by all its tiles).
// The triangular thread-block map becomes a per-channel tile table walked by
// persistent CTAs; only tiles that intersect i <= j are scheduled.
//
// One CTA = 6 warps: warp 0 TMA producer, warp 1 MMA issuer (+ TMEM owner), warps 2-5 epilogue.
// Tile = 128 Gram rows (32 stations, i side) x UMMA_N Gram columns (UMMA_N/4 stations, j side).
// K (= time) advances BK samples per ring stage, 32 per tcgen05.mma.  Time is the slowest input
// index, so both operands are MN-major in shared memory: a TMA box
// [BK t][1 f][128 B of m] lands as BK rows of 128 bytes, which is exactly the SWIZZLE_128B
// MN-major canonical layout (8-row atoms of 1024 B).  Two TMEM accumulators (2 x UMMA_N columns)
// let the epilogue of tile k overlap the MMAs of tile k+1.
#pragma once
#include "xc_ptx.cuh"

namespace xc {

constexpr int TC_BK = 64;          // samples per pipeline stage
constexpr int TC_UMMA_K = 32;      // samples per tcgen05.mma (kind::i8)
constexpr int TC_M = 128;          // Gram rows per tile = 32 stations
constexpr int TC_THREADS = 192;    // 6 warps
constexpr int TC_SMEM_LIMIT = 232448;  // 227 KB

template <int UMMA_N>
struct TcCfg {
    static constexpr int A_BYTES = TC_BK * 128;
    static constexpr int B_BYTES = TC_BK * UMMA_N;
    static constexpr int STAGE_BYTES = A_BYTES + B_BYTES;
    static constexpr int STAGES = (UMMA_N == 256) ? 8 : 12;
    static constexpr int BAR_BYTES = 1024;  // barriers + tmem slot, kept in the first KB
    static constexpr int SMEM_BYTES = BAR_BYTES + STAGES * STAGE_BYTES + 1024;  // + slack for 1024-B alignment
    static constexpr int SJ = UMMA_N / 4;   // stations per tile on the j side
    static_assert(SMEM_BYTES <= TC_SMEM_LIMIT, "smem");
};

struct TcParams {
    int N, F, T;
    int tiles_per_f;          // entries of `tiles` per channel
    long long total_tiles;    // F * tiles_per_f
    long long NB;             // N(N+1)/2
    const uint32_t* tiles;    // device: bi | (bj << 16)
    int32_t* vis;
    int accumulate;
};

// Epilogue for one 32-column chunk (8 stations j) held in v[]: complex combine, mask, store.
// Thread <-> Gram row r = (i, pi, ci): lanes 4s..4s+3 of a warp are one station i.
//   ci = 0 holds G[(i,pi,re), (j,pj,cj)], ci = 1 holds G[(i,pi,im), (j,pj,cj)]; the pair swaps
//   two values so that lane ci=0 ends with (Re,Im) of [pi][pj=0] and lane ci=1 with [pi][pj=1]:
//   every lane then stores 8 contiguous bytes and four lanes one 32-byte record.
template <bool MASKED, bool ACC>
__device__ __forceinline__ void epi_chunk(const uint32_t (&v)[32], int32_t* __restrict__ visf, int i, int jbase, int N,
                                          int lane) {
    const int ci = lane & 1;
    const int slot = (lane & 3) * 2;  // int32 offset inside the 8-int record: pi*4 + pj*2, pj := ci
#pragma unroll
    for (int js = 0; js < 8; ++js) {
        const int a0 = static_cast<int>(v[4 * js + 0]);  // column (j, pj=0, re)
        const int a1 = static_cast<int>(v[4 * js + 1]);  // column (j, pj=0, im)
        const int a2 = static_cast<int>(v[4 * js + 2]);  // column (j, pj=1, re)
        const int a3 = static_cast<int>(v[4 * js + 3]);  // column (j, pj=1, im)
        const int sx = ci ? a0 : a2;
        const int sy = ci ? a1 : a3;
        const int rx = __shfl_xor_sync(0xffffffffu, sx, 1);
        const int ry = __shfl_xor_sync(0xffffffffu, sy, 1);
        // ci=0: Re = G[re,re] + G[im,im] = a0 + ry ; Im = G[im,re] - G[re,im] = rx - a1   (pj = 0)
        // ci=1: Re = G[re,re] + G[im,im] = rx + a3 ; Im = G[im,re] - G[re,im] = a2 - ry   (pj = 1)
        int re = ci ? (rx + a3) : (a0 + ry);
        int im = ci ? (a2 - ry) : (rx - a1);
        const int j = jbase + js;
        if (!MASKED || (i <= j && j < N)) {
            int2* dst = reinterpret_cast<int2*>(visf + ((static_cast<long long>(j) * (j + 1) / 2 + i) * 8 + slot));
            if (ACC) {
                const int2 old = *dst;
                re += old.x;
                im += old.y;
            }
            *dst = make_int2(re, im);
        }
    }
}

template <int UMMA_N>
__global__ void __launch_bounds__(TC_THREADS, 1)
xc_i8_tc_kernel(const __grid_constant__ CUtensorMap tmap, const TcParams p) {
    using Cfg = TcCfg<UMMA_N>;
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    // Barriers first, operand ring after, on a 1024-byte boundary (SWIZZLE_128B atoms).
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem_raw);
    const uint32_t bar0 = smem_u32(bars);
    auto full_bar = [&](int s) { return bar0 + 8u * s; };
    auto empty_bar = [&](int s) { return bar0 + 8u * (Cfg::STAGES + s); };
    auto tfull_bar = [&](int b) { return bar0 + 8u * (2 * Cfg::STAGES + b); };
    auto tempty_bar = [&](int b) { return bar0 + 8u * (2 * Cfg::STAGES + 2 + b); };
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem_raw + 8 * (2 * Cfg::STAGES + 4));
    const uint32_t ring0 = (smem_u32(smem_raw) + Cfg::BAR_BYTES + 1023u) & ~1023u;

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;
    constexpr uint32_t TMEM_COLS = 2 * UMMA_N;  // 512 or 256: a power of two >= 32

    if (warp == 0 && lane == 0) {
        tma_prefetch_desc(&tmap);
        for (int s = 0; s < Cfg::STAGES; ++s) {
            mbar_init(full_bar(s), 1);
            mbar_init(empty_bar(s), 1);
        }
        for (int b = 0; b < 2; ++b) {
            mbar_init(tfull_bar(b), 1);
            mbar_init(tempty_bar(b), 4);  // one arrival per epilogue warp
        }
        fence_barrier_init();
    }
    if (warp == 1) {
        tmem_alloc(smem_u32(tmem_slot), TMEM_COLS);
        tmem_relinquish();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    const int KB = (p.T + TC_BK - 1) / TC_BK;

    if (warp == 0) {
        // ===== TMA producer (one lane) =====
        if (lane == 0) {
            int stage = 0;
            uint32_t phase = 0;
            for (long long w = blockIdx.x; w < p.total_tiles; w += gridDim.x) {
                const int f = static_cast<int>(w / p.tiles_per_f);
                const uint32_t tb = __ldg(p.tiles + static_cast<int>(w % p.tiles_per_f));
                const int m_a = static_cast<int>(tb & 0xFFFFu) * TC_M;
                const int m_b = static_cast<int>(tb >> 16) * UMMA_N;
                for (int kb = 0; kb < KB; ++kb) {
                    mbar_wait(empty_bar(stage), phase ^ 1u);
                    const uint32_t sa = ring0 + stage * Cfg::STAGE_BYTES;
                    const uint32_t sb = sa + Cfg::A_BYTES;
                    mbar_arrive_expect_tx(full_bar(stage), Cfg::STAGE_BYTES);
                    const int t0 = kb * TC_BK;
                    tma_load_3d(sa, &tmap, full_bar(stage), m_a, f, t0);
#pragma unroll
                    for (int h = 0; h < UMMA_N / 128; ++h)
                        tma_load_3d(sb + h * (TC_BK * 128), &tmap, full_bar(stage), m_b + 128 * h, f, t0);
                    if (++stage == Cfg::STAGES) {
                        stage = 0;
                        phase ^= 1u;
                    }
                }
            }
        }
    } else if (warp == 1) {
        // ===== MMA issuer (one lane) =====
        if (lane == 0) {
            constexpr uint32_t idesc = make_idesc_i8_mn(TC_M, UMMA_N);
            int stage = 0;
            uint32_t phase = 0;
            int buf = 0;
            uint32_t tphase = 0u;  // bit b = phase of accumulator b
            for (long long w = blockIdx.x; w < p.total_tiles; w += gridDim.x) {
                mbar_wait(tempty_bar(buf), ((tphase >> buf) & 1u) ^ 1u);  // epilogue has drained this accumulator
                tc_fence_after();
                const uint32_t d_tmem = tmem_base + static_cast<uint32_t>(buf * UMMA_N);
                for (int kb = 0; kb < KB; ++kb) {
                    mbar_wait(full_bar(stage), phase);
                    tc_fence_after();
                    const uint32_t sa = ring0 + stage * Cfg::STAGE_BYTES;
                    const uint32_t sb = sa + Cfg::A_BYTES;
                    const uint64_t adesc = make_smem_desc_mn_sw128(sa, TC_BK * 128, 1024);
                    const uint64_t bdesc = make_smem_desc_mn_sw128(sb, TC_BK * 128, 1024);
                    const int rows = min(TC_BK, p.T - kb * TC_BK);           // valid samples in this stage
                    const int nk = (rows + TC_UMMA_K - 1) / TC_UMMA_K;       // rows beyond T are TMA zero fill
#pragma unroll
                    for (int ks = 0; ks < TC_BK / TC_UMMA_K; ++ks) {
                        if (ks < nk) {
                            // K advance: 32 samples = 4 swizzle atoms = 4096 B -> +256 in the address field
                            umma_i8(d_tmem, adesc + static_cast<uint64_t>(ks * 256), bdesc + static_cast<uint64_t>(ks * 256),
                                    idesc, (kb | ks) ? 1u : 0u);
                        }
                    }
                    umma_commit(empty_bar(stage));  // frees the ring slot when these MMAs retire
                    if (++stage == Cfg::STAGES) {
                        stage = 0;
                        phase ^= 1u;
                    }
                }
                umma_commit(tfull_bar(buf));  // accumulator complete -> epilogue
                tphase ^= 1u << buf;
                buf ^= 1;
            }
        }
    } else {
        // ===== epilogue: warps 2..5, TMEM lane quarter = warp % 4 =====
        const int q = warp & 3;
        int buf = 0;
        uint32_t tphase = 0u;
        for (long long w = blockIdx.x; w < p.total_tiles; w += gridDim.x) {
            const int f = static_cast<int>(w / p.tiles_per_f);
            const uint32_t tb = __ldg(p.tiles + static_cast<int>(w % p.tiles_per_f));
            const int i0 = static_cast<int>(tb & 0xFFFFu) * 32 + 8 * q;  // first station of this warp's rows
            const int j0 = static_cast<int>(tb >> 16) * Cfg::SJ;
            const int i = i0 + (lane >> 2);
            int32_t* visf = p.vis + static_cast<long long>(f) * p.NB * 8;

            mbar_wait(tfull_bar(buf), (tphase >> buf) & 1u);
            tc_fence_after();
            const uint32_t taddr0 = tmem_base + (static_cast<uint32_t>(32 * q) << 16) + static_cast<uint32_t>(buf * UMMA_N);
#pragma unroll 1
            for (int cc = 0; cc < UMMA_N / 32; ++cc) {
                const int jbase = j0 + 8 * cc;
                if (jbase >= p.N || jbase + 7 < i0) continue;  // warp-uniform: nothing of this chunk is stored
                uint32_t v[32];
                tmem_ld_32x32(taddr0 + static_cast<uint32_t>(32 * cc), v);
                tmem_ld_wait();
                const bool full = (i0 + 7 <= jbase) && (jbase + 7 < p.N);  // warp-uniform: no masking needed
                if (p.accumulate) {
                    if (full) epi_chunk<false, true>(v, visf, i, jbase, p.N, lane);
                    else epi_chunk<true, true>(v, visf, i, jbase, p.N, lane);
                } else {
                    if (full) epi_chunk<false, false>(v, visf, i, jbase, p.N, lane);
                    else epi_chunk<true, false>(v, visf, i, jbase, p.N, lane);
                }
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(tempty_bar(buf));
            tphase ^= 1u << buf;
            buf ^= 1;
        }
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        __syncwarp();
        tc_fence_after();
        tmem_dealloc(tmem_base, TMEM_COLS);
    }
}

}  // namespace xc
