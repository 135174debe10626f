// xc_f32_tc.cuh -- the fp32-input X-engine on tcgen05 tensor cores: every product from three TF32 MMAs.
//
// What it computes: the same visibilities as xc_f32.cuh (Eq. 4, float samples), i.e. the real Gram matrix
// G = Z Z^T of the 4N rows m = (station, pol, re/im) over time, combined into complex entries in the epilogue exactly as
// in xc_i8_tc.cuh.  x x^H is a dense contraction, so it belongs on the tensor cores; they have no fp32 input type, so every
// sample is split into two TF32 numbers
//      a = hi + lo,   hi = rna_tf32(a) (11 significant bits),   lo = a - hi (exact in fp32, |lo| <= 2^-11 |a|)
// and a b is taken as  lo_a hi_b + hi_a lo_b + hi_a hi_b  (three kind::tf32 MMAs into one fp32 TMEM accumulator, small
// terms first).  What is dropped is lo_a lo_b (<= 2^-22 |a b|) and the bits of lo beyond TF32's 11 (<= 2^-21 |a b|, either
// sign): the same order as the fp32 rounding of the products themselves, far inside north_star's 1e-5 sqrt(V_ii V_jj).
// Integer-valued samples below 2^11 have lo = 0 and exact products: the result then equals the int8 path's bit for bit
// (sums below 2^24), which the tests use.
//
// Accumulation.  The tensor core adds into its fp32 accumulator by truncation, not to nearest: a sum of T like-signed
// terms (every autocorrelation) comes out low by ~1e-8 T relative (measured: 9e-6 at T = 1000, i.e. the whole of
// north_star's 1e-5 budget).  One TMEM accumulator therefore only sums FT_CHUNK_STAGES x 32 = 128 samples (bias <= ~1.3e-6
// whatever T is); the epilogue warps add the chunks in registers with round-to-nearest fp32 adds while the tensor core
// already fills the other accumulator with the next chunk.
//
// Pipeline per CTA of a pair (cta_group::2, 256 x 256 Gram tile = 64 x 64 stations, as in xc_i8_tc.cuh):
//   warp 0      TMA producer: per 32-sample stage 4 + 4 boxes [32 t][32 floats] (A rows, this CTA's half of the B rows;
//               diagonal tiles load B only), 128-byte swizzle with 32-byte atoms, MN-major -- time is the slowest input index
//   warps 2-7   split: read the stage's raw samples, write hi in their place and lo into the stage's second half (the
//               split is elementwise, so it does not care about the swizzle), fence.proxy.async, then arrive on the leader's
//               barrier with CTA-scope release (as CUTLASS's ClusterBarrier::arrive does): the bytes are only ever read by
//               this CTA's own SM on behalf of the pair's MMA.  A cluster-scope release compiles to MEMBAR.ALL.GPU and cost
//               a quarter of the throughput (0.96 ms against 0.58 ms on config 3's shape, F = 128)
//   warp 1      MMA issuer (leader CTA): per 8-sample K step three tcgen05.mma.kind::tf32 M = 256, N = 256
//   warps 8-15  epilogue: per 128-sample chunk tcgen05.ld + add into 128 running sums per thread; per tile lane-pair swap,
//               float combine, 16-byte streaming stores (same packing as int8)
// Shared memory per stage: 32 KB raw/hi + 32 KB lo; three stages.  TMEM: two 256-column fp32 accumulators.
// Registers: the epilogue threads hold 128 running sums each, so the two warpgroups of warps 0-7 drop to 72 registers per thread
// and the two epilogue warpgroups rise to 184 (setmaxnreg; with two split warps and 384 threads of 168 registers the split was
// the bottleneck: 0.574 against 0.504 ms on config 3's shape, F = 128).
#pragma once
#include "xc_i8_tc.cuh"

namespace xc {

#ifndef XC_FT_BK
#define XC_FT_BK 32
#endif
constexpr int FT_BK = XC_FT_BK;                            // samples per ring stage (K = 8 steps of three MMAs each)
constexpr int FT_UMMA_K = 8;                               // samples per tcgen05.mma (kind::tf32)
constexpr int FT_BOX_BYTES = FT_BK * 128;                  // one TMA box: FT_BK rows of 32 floats
constexpr int FT_OP_BYTES = 4 * FT_BOX_BYTES;              // 128 Gram rows = 4 boxes = 4 MN atoms of 32 floats
constexpr int FT_RAW_BYTES = 2 * FT_OP_BYTES;              // A rows + this CTA's half of the B rows
constexpr int FT_STAGE_BYTES = 2 * FT_RAW_BYTES;           // hi parts (in place of the raw samples) + lo parts
constexpr int FT_STAGES = 196608 / FT_STAGE_BYTES;          // 192 KB of ring
#ifndef XC_FT_CHUNK
#define XC_FT_CHUNK (128 / XC_FT_BK)
#endif
#ifndef XC_FT_CONV_WARPS
#define XC_FT_CONV_WARPS 6
#endif
constexpr int FT_CHUNK_STAGES = XC_FT_CHUNK;               // stages (of 32 samples) summed in one TMEM accumulator, see below
constexpr int FT_CONV_WARPS = XC_FT_CONV_WARPS;
constexpr int FT_EPI_WARPS = 8;
constexpr int FT_THREADS = 64 + 32 * (FT_CONV_WARPS + FT_EPI_WARPS);   // 512 with 6 split warps: 128 registers per thread at launch, re-divided with setmaxnreg
constexpr int FT_BAR_BYTES = 1024;
constexpr int FT_SMEM_BYTES = FT_BAR_BYTES + FT_STAGES * FT_STAGE_BYTES + 1024;   // + slack for 1024-byte alignment
constexpr int FT_INLINE_TILES = 48;
static_assert(FT_SMEM_BYTES <= TC_SMEM_LIMIT, "smem");
static_assert((2 + FT_CONV_WARPS) % 4 == 0, "the epilogue warps must start on a multiple of 4 (TMEM lane quarter = warp % 4)");

struct F32TcParams {
    int N, F, T;
    int tiles_per_f;          // entries of the tile table per channel
    int total_tiles;          // F * tiles_per_f
    long long NB;             // N(N+1)/2
    const uint32_t* tiles;    // device: bi | (bj << 16) in 64-station blocks (used if tiles_per_f > FT_INLINE_TILES)
    float* vis;
    int accumulate;
    unsigned long long* stamps;   // as TcParams::stamps, or null
    uint32_t tiles_inline[FT_INLINE_TILES];
};

__device__ __forceinline__ uint32_t ft_tile_at(const F32TcParams& p, int k) {
    return p.tiles_per_f <= FT_INLINE_TILES ? p.tiles_inline[k] : __ldg(p.tiles + k);
}

// Instruction descriptor for kind::tf32: D = F32, A = B = TF32, both MN-major, dense.
//   [4,6) c_format = 1 (F32)   [7,10) a_format = 2 (TF32)   [10,13) b_format = 2 (TF32)
//   [15] a_major = 1 (MN)      [16] b_major = 1 (MN)        [17,23) N >> 3   [24,29) M >> 4
__host__ __device__ constexpr uint32_t make_idesc_tf32_mn(int M, int N) {
    return (1u << 4) | (2u << 7) | (2u << 10) | (1u << 15) | (1u << 16) | (static_cast<uint32_t>(N >> 3) << 17) |
           (static_cast<uint32_t>(M >> 4) << 24);
}
// D[tmem] (+)= A[smem desc] * B[smem desc]^T, tf32 x tf32 -> fp32, CTA pair, issued by one thread of the leader.
__device__ __forceinline__ void umma_tf32_2cta(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc,
                                               uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::2.kind::tf32 [%0], %1, %2, %3, p;\n\t}"
        ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate)
        : "memory");
}
// Shared-memory descriptor for an MN-major 32-bit operand: the only swizzle the tensor core accepts there is "128 B with
// 32-byte atomicity" (layout type 1; TMA: CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B): atoms of 4 k-rows x 128 contiguous bytes of
// mn (512 B), inside which the four 32-byte chunks of a row are permuted by the row index mod 4.  LBO = distance between
// atoms along MN, SBO = distance between atoms along K (field layout as make_smem_desc_mn_sw128).
__device__ __forceinline__ uint64_t make_smem_desc_mn_sw128_32b(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
    uint64_t d = 0;
    d |= static_cast<uint64_t>((saddr & 0x3FFFFu) >> 4);
    d |= static_cast<uint64_t>((lbo_bytes >> 4) & 0x3FFFu) << 16;
    d |= static_cast<uint64_t>((sbo_bytes >> 4) & 0x3FFFu) << 32;
    d |= 1ull << 46;
    d |= 1ull << 61;
    return d;
}
// Nearest TF32 (10 mantissa bits), ties away from zero -- cvt.rna.tf32.f32 for finite values, in two integer instructions on
// the full-rate ALU instead of the conversion unit (a value that rounds up into the next binade or to infinity does so here too).
__device__ __forceinline__ float ft_rna_tf32(float a) {
    return __uint_as_float((__float_as_uint(a) + 0x1000u) & 0xFFFFE000u);
}
__device__ __forceinline__ float4 ft_ld_shared_f4(uint32_t addr) {
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ void ft_st_shared_f4(uint32_t addr, float4 v) {
    asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}

// Epilogue for one 32-column chunk: xc_i8_tc.cuh's epi_chunk with float arithmetic (same lane roles, same packing).
template <bool MASKED, bool ACC>
__device__ __forceinline__ void ft_epi_chunk(const float (&v)[32], float* __restrict__ visf, int i, int jbase, int N, int lane) {
    const int ci = lane & 1;
    const int slot = ((lane >> 1) & 1) * 4;
#pragma unroll
    for (int jp = 0; jp < 4; ++jp) {
        float own[4], got[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const float e = v[8 * jp + k];
            const float o = v[8 * jp + 4 + k];
            own[k] = ci ? o : e;
            got[k] = __shfl_xor_sync(0xffffffffu, ci ? e : o, 1);
        }
        const float R0 = ci ? got[0] : own[0], R1 = ci ? got[1] : own[1], R2 = ci ? got[2] : own[2], R3 = ci ? got[3] : own[3];
        const float I0 = ci ? own[0] : got[0], I1 = ci ? own[1] : got[1], I2 = ci ? own[2] : got[2], I3 = ci ? own[3] : got[3];
        float4 out;
        out.x = R0 + I1;   // Re [pi][0] = G[re,re] + G[im,im]
        out.y = I0 - R1;   // Im [pi][0] = G[im,re] - G[re,im]
        out.z = R2 + I3;   // Re [pi][1]
        out.w = I2 - R3;   // Im [pi][1]
        const int j = jbase + 2 * jp + ci;
        if (!MASKED || (i <= j && j < N)) {
            float4* dst = reinterpret_cast<float4*>(visf + (static_cast<long long>(j) * (j + 1) / 2 + i) * 8 + slot);
            if (ACC) {
                const float4 old = __ldcs(dst);
                out.x += old.x;
                out.y += old.y;
                out.z += old.z;
                out.w += old.w;
            }
            __stcs(dst, out);
        }
    }
}

__global__ void __launch_bounds__(FT_THREADS, 1)
xc_f32_tc_kernel(const __grid_constant__ CUtensorMap tmap, const __grid_constant__ F32TcParams p) {
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    const uint32_t bar0 = smem_u32(smem_raw);
    auto full_bar = [&](uint32_t s) { return bar0 + 8u * s; };                          // local: this CTA's TMA bytes
    auto conv_bar = [&](uint32_t s) { return bar0 + 8u * (FT_STAGES + s); };            // leader: both CTAs' stages are split
    auto empty_bar = [&](uint32_t s) { return bar0 + 8u * (2 * FT_STAGES + s); };       // both: the MMAs have read the stage
    auto tfull_bar = [&](uint32_t b) { return bar0 + 8u * (3 * FT_STAGES + b); };
    auto tempty_bar = [&](uint32_t b) { return bar0 + 8u * (3 * FT_STAGES + 2 + b); };
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem_raw + 8 * (3 * FT_STAGES + 4));
    const uint32_t ring0 = (bar0 + FT_BAR_BYTES + 1023u) & ~1023u;

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;
    const uint32_t rank = cluster_ctarank();                 // 0 = leader of the pair
    const int unit = static_cast<int>(blockIdx.x) / 2, nunits = static_cast<int>(gridDim.x) / 2;
    constexpr uint32_t TMEM_COLS = 512;

    if (p.stamps && threadIdx.x == FT_THREADS - 32) {
        const unsigned long long c = static_cast<unsigned long long>(clock64());
        const unsigned long long gt = globaltimer_ns();
        atomicMin(p.stamps + 0, gt);
        if (blockIdx.x == 0) {
            p.stamps[2] = c;
            p.stamps[3] = gt;
        }
    }
    if (warp == 0 && lane == 0) {
        tma_prefetch_desc(&tmap);
        for (int s = 0; s < FT_STAGES; ++s) {
            mbar_init(full_bar(s), 1);                       // producer's arrive.expect_tx (+ this CTA's TMA bytes)
            mbar_init(conv_bar(s), 2 * FT_CONV_WARPS);       // (on the leader) one arrival per split warp of the pair
            mbar_init(empty_bar(s), 1);                      // tcgen05.commit, multicast to both CTAs
        }
        for (int b = 0; b < 2; ++b) {
            mbar_init(tfull_bar(b), 1);
            mbar_init(tempty_bar(b), 2 * FT_EPI_WARPS);
        }
        fence_barrier_init();
    }
    if (warp == 1) {
        tmem_alloc<2>(smem_u32(tmem_slot), TMEM_COLS);
        tmem_relinquish<2>();
    }
    tc_fence_before();
    cluster_sync_all();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;
    pdl_grid_dependency_wait();
    pdl_launch_dependents();

    const int KB = (p.T + FT_BK - 1) / FT_BK;

    if (warp < 2 + FT_CONV_WARPS) {
#if XC_FT_CONV_WARPS == 6
        // 16 warps = four warpgroups of 128 registers per thread at launch: the two groups that hold the producer, the issuer
        // and the split warps hand registers to the two epilogue groups (128 running sums per thread): 256 x 72 + 256 x 184 = 64 K
        asm volatile("setmaxnreg.dec.sync.aligned.u32 72;" ::: "memory");
#endif
        if (warp == 0) {
            // ===== TMA producer =====
            const uint32_t elected = elect_one();
            uint32_t stage = 0, phase = 0;
            int w_next = walk(0, unit, nunits, p.total_tiles);
            uint32_t tb_next = (w_next >= 0) ? ft_tile_at(p, w_next % p.tiles_per_f) : 0u;
            for (int n = 0; w_next >= 0; ++n) {
                const int f = w_next / p.tiles_per_f;
                const uint32_t tb = __shfl_sync(0xffffffffu, tb_next, 0);
                w_next = walk(n + 1, unit, nunits, p.total_tiles);
                if (w_next >= 0) tb_next = ft_tile_at(p, w_next % p.tiles_per_f);
                const int m_a = static_cast<int>(tb & 0xFFFFu) * 256 + 128 * static_cast<int>(rank);   // first Gram row (float) of A
                const int m_b = static_cast<int>(tb >> 16) * 256 + 128 * static_cast<int>(rank);
                const bool a_in_b = (m_a == m_b);     // diagonal tile: this CTA's A rows are its B rows
                for (int kb = 0; kb < KB; ++kb) {
                    mbar_wait(empty_bar(stage), phase ^ 1u);
                    if (elected) {
                        const uint32_t sa = ring0 + stage * FT_STAGE_BYTES;
                        const uint32_t sb = sa + FT_OP_BYTES;
                        const int t0 = kb * FT_BK;
                        mbar_arrive_expect_tx(full_bar(stage), a_in_b ? FT_OP_BYTES : FT_RAW_BYTES);
                        if (!a_in_b) {
#pragma unroll
                            for (int g = 0; g < 4; ++g) tma_load_3d(sa + g * FT_BOX_BYTES, &tmap, full_bar(stage), m_a + 32 * g, f, t0);
                        }
#pragma unroll
                        for (int g = 0; g < 4; ++g) tma_load_3d(sb + g * FT_BOX_BYTES, &tmap, full_bar(stage), m_b + 32 * g, f, t0);
                    }
                    __syncwarp();
                    if (++stage == FT_STAGES) {
                        stage = 0;
                        phase ^= 1u;
                    }
                }
            }
        } else if (warp == 1) {
            // ===== MMA issuer: leader CTA only =====
            if (rank == 0) {
                const uint32_t elected = elect_one();
                constexpr uint32_t idesc = make_idesc_tf32_mn(256, 256);
                uint32_t stage = 0, phase = 0, buf = 0, tphase = 0;
                int w_next = walk(0, unit, nunits, p.total_tiles);
                uint32_t tb_next = (w_next >= 0) ? ft_tile_at(p, w_next % p.tiles_per_f) : 0u;
                for (int n = 0; w_next >= 0; ++n) {
                    const uint32_t tb = __shfl_sync(0xffffffffu, tb_next, 0);
                    w_next = walk(n + 1, unit, nunits, p.total_tiles);
                    if (w_next >= 0) tb_next = ft_tile_at(p, w_next % p.tiles_per_f);
                    const bool a_in_b = ((tb & 0xFFFFu) == (tb >> 16));
                    const uint32_t a_off = a_in_b ? static_cast<uint32_t>(FT_OP_BYTES) : 0u;
                    for (int kb = 0; kb < KB; ++kb) {
                        const int kc = kb % FT_CHUNK_STAGES;                     // stage inside the chunk
                        if (kc == 0) {
                            mbar_wait(tempty_bar(buf), ((tphase >> buf) & 1u) ^ 1u);   // the epilogues have drained this accumulator
                            tc_fence_after();
                        }
                        const uint32_t d_tmem = tmem_base + buf * 256u;
                        mbar_wait_acquire_cluster(conv_bar(stage), phase);     // both CTAs' halves of the stage are split
                        tc_fence_after();
                        const bool chunk_end = (kc == FT_CHUNK_STAGES - 1) || (kb == KB - 1);
                        if (elected) {
                            const uint32_t sa = ring0 + stage * FT_STAGE_BYTES;
                            // MN-major, 128-byte swizzle with 32-byte atoms: atoms of 4 samples x 32 floats; LBO = one box between
                            // MN atoms, SBO = 512 B between the two atoms of an 8-sample K step
                            const uint64_t ahi = make_smem_desc_mn_sw128_32b(sa + a_off, FT_BOX_BYTES, 512);
                            const uint64_t alo = make_smem_desc_mn_sw128_32b(sa + FT_RAW_BYTES + a_off, FT_BOX_BYTES, 512);
                            const uint64_t bhi = make_smem_desc_mn_sw128_32b(sa + FT_OP_BYTES, FT_BOX_BYTES, 512);
                            const uint64_t blo = make_smem_desc_mn_sw128_32b(sa + FT_RAW_BYTES + FT_OP_BYTES, FT_BOX_BYTES, 512);
                            const int rows = min(FT_BK, p.T - kb * FT_BK);
                            const int nk = (rows + FT_UMMA_K - 1) / FT_UMMA_K;       // rows beyond T are TMA zero fill
#pragma unroll
                            for (int ks = 0; ks < FT_BK / FT_UMMA_K; ++ks) {
                                if (ks < nk) {
                                    const uint64_t adv = static_cast<uint64_t>(ks * 64);   // 8 samples = two atoms = 1024 B
                                    umma_tf32_2cta(d_tmem, alo + adv, bhi + adv, idesc, (kc | ks) ? 1u : 0u);
                                    umma_tf32_2cta(d_tmem, ahi + adv, blo + adv, idesc, 1u);
                                    umma_tf32_2cta(d_tmem, ahi + adv, bhi + adv, idesc, 1u);
                                }
                            }
                            umma_commit<2>(empty_bar(stage));
                            if (chunk_end) umma_commit<2>(tfull_bar(buf));      // chunk complete -> epilogues
                        }
                        __syncwarp();
                        if (chunk_end) {
                            tphase ^= 1u << buf;
                            buf ^= 1u;
                        }
                        if (++stage == FT_STAGES) {
                            stage = 0;
                            phase ^= 1u;
                        }
                    }
                }
            }
        } else {
            // ===== split warps: raw fp32 -> hi (in place) + lo =====
            const uint32_t tid_c = static_cast<uint32_t>((warp - 2) * 32 + lane);
            const uint32_t lead_conv0 = mapa_u32(conv_bar(0), 0);
            uint32_t stage = 0, phase = 0;
            int w_next = walk(0, unit, nunits, p.total_tiles);
            uint32_t tb_next = (w_next >= 0) ? ft_tile_at(p, w_next % p.tiles_per_f) : 0u;
            for (int n = 0; w_next >= 0; ++n) {
                const uint32_t tb = tb_next;
                w_next = walk(n + 1, unit, nunits, p.total_tiles);
                if (w_next >= 0) tb_next = ft_tile_at(p, w_next % p.tiles_per_f);
                const bool a_in_b = ((tb & 0xFFFFu) == (tb >> 16));
                const uint32_t first = a_in_b ? static_cast<uint32_t>(FT_OP_BYTES) : 0u;     // diagonal tiles hold B rows only
                for (int kb = 0; kb < KB; ++kb) {
                    mbar_wait(full_bar(stage), phase);
                    const uint32_t base = ring0 + stage * FT_STAGE_BYTES;
#pragma unroll 4
                    for (uint32_t off = first + tid_c * 16u; off < static_cast<uint32_t>(FT_RAW_BYTES); off += FT_CONV_WARPS * 32u * 16u) {
                        const float4 a = ft_ld_shared_f4(base + off);
                        float4 hi, lo;
                        hi.x = ft_rna_tf32(a.x); hi.y = ft_rna_tf32(a.y); hi.z = ft_rna_tf32(a.z); hi.w = ft_rna_tf32(a.w);
                        lo.x = a.x - hi.x; lo.y = a.y - hi.y; lo.z = a.z - hi.z; lo.w = a.w - hi.w;
                        ft_st_shared_f4(base + off, hi);
                        ft_st_shared_f4(base + FT_RAW_BYTES + off, lo);
                    }
                    fence_proxy_async_smem();          // the tensor core reads these bytes through the async proxy
                    __syncwarp();
#ifdef XC_FT_RELEASE_CLUSTER
                    // canary build (-DXC_FT_RELEASE_CLUSTER): the arrive that the PTX memory model formally pairs with the
                    // leader's cluster-scope acquire; 1.65x slower, run once per round against test_f32_*
                    if (lane == 0) mbar_arrive_release_cluster(lead_conv0 + 8u * stage);
#else
                    if (lane == 0) mbar_arrive_remote_release_cta(lead_conv0 + 8u * stage);
#endif
                    if (++stage == FT_STAGES) {
                        stage = 0;
                        phase ^= 1u;
                    }
                }
            }
        }
    } else {
#if XC_FT_CONV_WARPS == 6
        asm volatile("setmaxnreg.inc.sync.aligned.u32 184;" ::: "memory");
#endif
        // ===== epilogue: the last 8 warps; TMEM lane quarter = warp % 4, column half = (warp - first) / 4 =====
        const int q = warp & 3;
        const int half = (warp - 2 - FT_CONV_WARPS) >> 2;
        constexpr int CHUNKS = 4;                       // 32-column chunks per warp (128 of the 256 columns)
        uint32_t buf = 0, tphase = 0;
        const uint32_t lead_tempty0 = mapa_u32(tempty_bar(0), 0);
        int w_next = walk(0, unit, nunits, p.total_tiles);
        uint32_t tb_next = (w_next >= 0) ? ft_tile_at(p, w_next % p.tiles_per_f) : 0u;
        for (int n = 0; w_next >= 0; ++n) {
            const int f = w_next / p.tiles_per_f;
            const uint32_t tb = tb_next;
            w_next = walk(n + 1, unit, nunits, p.total_tiles);
            if (w_next >= 0) tb_next = ft_tile_at(p, w_next % p.tiles_per_f);
            const int i0 = static_cast<int>(tb & 0xFFFFu) * 64 + 32 * static_cast<int>(rank) + 8 * q;
            const int col0 = 32 * CHUNKS * half;
            const int j0 = static_cast<int>(tb >> 16) * 64 + col0 / 4;
            const int i = i0 + (lane >> 2);
            float* visf = p.vis + static_cast<long long>(f) * p.NB * 8;

            // warp-uniform: which of this warp's four 32-column chunks hold anything that is stored
            bool live[CHUNKS];
#pragma unroll
            for (int cc = 0; cc < CHUNKS; ++cc) live[cc] = !(j0 + 8 * cc >= p.N || j0 + 8 * cc + 7 < i0);
            float acc[CHUNKS][32];                  // running sums over the tile's 128-sample chunks
            const int nchunks = (KB + FT_CHUNK_STAGES - 1) / FT_CHUNK_STAGES;
            for (int c = 0; c < nchunks; ++c) {
                mbar_wait(tfull_bar(buf), (tphase >> buf) & 1u);
                tc_fence_after();
                const uint32_t taddr0 = tmem_base + (static_cast<uint32_t>(32 * q) << 16) + buf * 256u + col0;
#pragma unroll
                for (int cc = 0; cc < CHUNKS; ++cc) {
                    if (!live[cc]) continue;
                    uint32_t v[32];
                    tmem_ld_32x32(taddr0 + static_cast<uint32_t>(32 * cc), v);
                    tmem_ld_wait();
                    if (c == 0) {
#pragma unroll
                        for (int k = 0; k < 32; ++k) acc[cc][k] = __uint_as_float(v[k]);
                    } else {
#pragma unroll
                        for (int k = 0; k < 32; ++k) acc[cc][k] += __uint_as_float(v[k]);    // fp32 add, round to nearest
                    }
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive_cluster(lead_tempty0 + 8u * buf);
                tphase ^= 1u << buf;
                buf ^= 1u;
            }
#pragma unroll
            for (int cc = 0; cc < CHUNKS; ++cc) {
                if (!live[cc]) continue;
                const int jbase = j0 + 8 * cc;
                const bool full = (i0 + 7 <= jbase) && (jbase + 7 < p.N);
                if (p.accumulate) {
                    if (full) ft_epi_chunk<false, true>(acc[cc], visf, i, jbase, p.N, lane);
                    else ft_epi_chunk<true, true>(acc[cc], visf, i, jbase, p.N, lane);
                } else {
                    if (full) ft_epi_chunk<false, false>(acc[cc], visf, i, jbase, p.N, lane);
                    else ft_epi_chunk<true, false>(acc[cc], visf, i, jbase, p.N, lane);
                }
            }
        }
    }

    // Teardown: nobody leaves (or frees TMEM) while a peer may still signal into this CTA.
    tc_fence_before();
    cluster_sync_relaxed();
    if (warp == 1) {
        __syncwarp();
        tc_fence_after();
        tmem_dealloc<2>(tmem_base, TMEM_COLS);
    }
    if (p.stamps && threadIdx.x == FT_THREADS - 32) {
        const unsigned long long c = static_cast<unsigned long long>(clock64());
        const unsigned long long gt = globaltimer_ns();
        atomicMax(p.stamps + 1, gt);
        if (blockIdx.x == 0) {
            p.stamps[4] = c;
            p.stamps[5] = gt;
        }
    }
}

}  // namespace xc
