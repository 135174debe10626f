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
// persistent CTAs (or CTA pairs); only tiles that intersect i <= j are scheduled.
//
// One CTA = 10 warps: warp 0 TMA producer, warp 1 MMA issuer (+ TMEM owner), warps 2-9 epilogue.
// CG = 1: tile = 128 Gram rows (32 stations, i side) x UMMA_N Gram columns, one CTA.
// CG = 2: tile = 256 Gram rows (64 stations) x 256 columns (64 stations) on a CTA pair
//         (tcgen05 cta_group::2): each CTA holds its own 128 A rows and half of B, so every
//         operand byte is fetched from L2 and written to shared memory once per pair.
// K (= time) advances BK samples per ring stage, 32 per tcgen05.mma.  Time is the slowest input
// index, so both operands are MN-major in shared memory: a TMA box
// [BK t][1 f][128 B of m] lands as BK rows of 128 bytes, which is exactly the SWIZZLE_128B
// MN-major canonical layout (8-row atoms of 1024 B).  Two TMEM accumulators (2 x UMMA_N columns)
// let the epilogue of tile k overlap the MMAs of tile k+1.  On tiles that touch the diagonal the
// A rows are a sub-block of the B rows: they are loaded once and both descriptors point at them.
//
// Producer and MMA loops run warp-uniformly (all 32 lanes walk the loop, one elected lane issues)
// so that addresses, coordinates and descriptors stay in uniform registers: a single-lane branch
// costs ~80 cycles per TMA / MMA issue in register->uniform-register waterfalls, which at 128
// tensor cycles per MMA starves the pipe (measured).
#pragma once
#include "xc_ptx.cuh"

namespace xc {

constexpr int TC_UMMA_K = 32;      // samples per tcgen05.mma (kind::i8)
constexpr int TC_EPI_WARPS = 8;     // 2 per TMEM lane quarter, each owning half of the tile's columns
constexpr int TC_THREADS = 64 + 32 * TC_EPI_WARPS;   // + TMA producer warp + MMA issuer warp
constexpr int TC_SMEM_LIMIT = 232448;  // 227 KB

template <int UMMA_N, int CG, bool STAGED, int BK_ = 128, bool DIAG_ = false>
struct TcCfg {
    // DIAG: every tile of the launch sits on the diagonal (its A rows are one of its own B boxes), so the ring
    // holds no separate A box -- the single-CTA 128x256 tile then has the same 32 KB stages as the CTA-pair tile.
    static constexpr bool DIAG = DIAG_;
    static constexpr int M = 128 * CG;                    // Gram rows per tile
    static constexpr int B_BOXES = UMMA_N / 128 / CG;     // 128-row B boxes held by one CTA
    // Samples per pipeline stage.  Every stage costs the producer and the MMA issuer some hundred cycles of
    // barrier round trips and instruction issue (measured), so a stage must hold clearly more than that in
    // tensor work (128 cycles per 32 samples).  192-sample stages (4 of them) measured slower than 128 x 7.
    static constexpr int BK = BK_;
    static constexpr int BOX_BYTES = BK * 128;            // one TMA box: BK rows of 128 bytes
    static constexpr int A_BYTES = DIAG_ ? 0 : BOX_BYTES;
    static constexpr int B_BYTES = B_BOXES * BOX_BYTES;
    static constexpr int STAGE_BYTES = A_BYTES + B_BYTES;
    static constexpr int SI = 32 * CG;                    // stations per tile on the i side
    static constexpr int SJ = UMMA_N / 4;                 // stations per tile on the j side
    // STAGED: the epilogue packs the tile's visibilities into shared memory ([SJ rows j][32 stations i][32 B]) and
    // the TMA store engine writes each row's contiguous run to global memory (bulk copy / bulk reduce-add).
    static constexpr int OUT_BYTES = STAGED ? SJ * 1024 : 0;
    static constexpr int STAGES = (229376 - OUT_BYTES) / STAGE_BYTES;   // 224 KB for ring + staging tile
    static constexpr int BAR_BYTES = 1024;                // barriers + tmem slot, kept in the first KB
    static constexpr int SMEM_BYTES = BAR_BYTES + STAGES * STAGE_BYTES + OUT_BYTES + 1024;  // + slack for 1024-B alignment
    static_assert(B_BOXES >= 1, "a CTA holds at least one 128-row B box");
    static_assert(!DIAG_ || (CG == 1 && UMMA_N == 256 && !STAGED), "DIAG is the single-CTA 128x256 direct-store variant");
    static_assert(SMEM_BYTES <= TC_SMEM_LIMIT, "smem");
    static_assert(STAGES >= 2, "ring too shallow");
};

struct TcParams {
    int N, F, T;
    int tiles_per_f;          // entries of `tiles` per channel (a multiple of 1 << group_shift)
    int total_tiles;          // F * tiles_per_f
    int group_shift;          // a persistent CTA takes 2^group_shift consecutive table entries at a time (walk())
    long long NB;             // N(N+1)/2
    const uint32_t* tiles;    // device: bi | (bj << 16), in units of (SI, SJ) stations; TC_TILE_EMPTY = padding entry
    int32_t* vis;
    int accumulate;
    int debug_skip;           // profiling only (XC_OPT_DEBUG_SKIP): 1 = no TMA after the first ring fill,
                              // 2 = no MMA, 4 = no global stores; results are then meaningless
    long long* trace;         // profiling only: CTA 0 writes clock64() stamps here (see TC_TRACE_*), or null
};
constexpr uint32_t TC_TILE_EMPTY = 0xFFFFFFFFu;
constexpr int TC_TRACE_ITERS = 256;

// The persistent walk (S1): work unit `unit` of `nunits` takes groups unit, unit + nunits, ... of 2^gs consecutive
// entries of the (channel-major) tile list; n counts the entries this unit has taken so far.  Returns the global
// entry index, or -1 past the end.  Groups keep the two unequal sub-tiles of one diagonal block on one CTA.
__device__ __forceinline__ int walk(int n, int unit, int nunits, int gs, int total) {
    const long long w = ((static_cast<long long>(unit) + static_cast<long long>(n >> gs) * nunits) << gs) + (n & ((1 << gs) - 1));
    return w < total ? static_cast<int>(w) : -1;
}   // k-blocks traced; layout: [3 roles][TC_TRACE_ITERS][4] long long + 4 clock words

// Epilogue for one 32-column chunk (8 stations j) held in v[]: complex combine, mask, store.
// Thread <-> Gram row r = (i, pi, ci): lanes 4s..4s+3 of a warp are one station i; ci = 0 holds
// G[(i,pi,re), (j,pj,cj)] and ci = 1 holds G[(i,pi,im), (j,pj,cj)] for the chunk's columns (j,pj,cj).
// Stations j are taken two at a time: the ci = 0 lane finishes the even one, the ci = 1 lane the odd
// one, after swapping the four values the other needs (4 shuffles per station pair).  Each lane then
// owns [pi][pj=0,1][re,im] of its (i, j) = 16 contiguous bytes, two lanes one 32-byte record, and a
// warp store instruction writes two 256-byte runs (8 consecutive i for each of the two j).
template <bool MASKED, bool ACC, bool NOSTORE = false, bool WRAP = false>
__device__ __forceinline__ void epi_chunk(const uint32_t (&v)[32], int32_t* __restrict__ visf, int i, int jbase, int N,
                                          int lane) {
    const int ci = lane & 1;
    const int slot = ((lane >> 1) & 1) * 4;  // int32 offset of [pi] inside the 8-int record
#pragma unroll
    for (int jp = 0; jp < 4; ++jp) {
        int own[4], got[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const int e = static_cast<int>(v[8 * jp + k]);      // even station of the pair, column (pj, cj) = k
            const int o = static_cast<int>(v[8 * jp + 4 + k]);  // odd station of the pair
            own[k] = ci ? o : e;
            got[k] = __shfl_xor_sync(0xffffffffu, ci ? e : o, 1);
        }
        // R[k] = G[(i,pi,re),(j,k)], I[k] = G[(i,pi,im),(j,k)] for this lane's station j; k = 2*pj + cj
        const int R0 = ci ? got[0] : own[0], R1 = ci ? got[1] : own[1], R2 = ci ? got[2] : own[2], R3 = ci ? got[3] : own[3];
        const int I0 = ci ? own[0] : got[0], I1 = ci ? own[1] : got[1], I2 = ci ? own[2] : got[2], I3 = ci ? own[3] : got[3];
        int4 out;
        out.x = R0 + I1;   // Re [pi][0] = G[re,re] + G[im,im]
        out.y = I0 - R1;   // Im [pi][0] = G[im,re] - G[re,im]
        out.z = R2 + I3;   // Re [pi][1]
        out.w = I2 - R3;   // Im [pi][1]
        const int j = jbase + 2 * jp + ci;
        if ((!MASKED || (i <= j && j < N)) && !NOSTORE) {
            long long off = (static_cast<long long>(j) * (j + 1) / 2 + i) * 8 + slot;
            if (WRAP) off &= (1 << 21) - 1;   // profiling: keep all stores inside an 8 MB window (L2 resident)
            int4* dst = reinterpret_cast<int4*>(visf + off);
            if (ACC) {
                const int4 old = __ldcs(dst);
                out.x += old.x;
                out.y += old.y;
                out.z += old.z;
                out.w += old.w;
            }
            __stcs(dst, out);   // streaming: written once, never re-read by this kernel
        }
    }
}

// Same combine, but the 16 bytes go to the packed staging tile in shared memory (row pitch 1024 B per j).
__device__ __forceinline__ void epi_chunk_smem(const uint32_t (&v)[32], uint32_t dst, int lane) {
    const int ci = lane & 1;
#pragma unroll
    for (int jp = 0; jp < 4; ++jp) {
        int own[4], got[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const int e = static_cast<int>(v[8 * jp + k]);
            const int o = static_cast<int>(v[8 * jp + 4 + k]);
            own[k] = ci ? o : e;
            got[k] = __shfl_xor_sync(0xffffffffu, ci ? e : o, 1);
        }
        const int R0 = ci ? got[0] : own[0], R1 = ci ? got[1] : own[1], R2 = ci ? got[2] : own[2], R3 = ci ? got[3] : own[3];
        const int I0 = ci ? own[0] : got[0], I1 = ci ? own[1] : got[1], I2 = ci ? own[2] : got[2], I3 = ci ? own[3] : got[3];
        st_shared_v4(dst + static_cast<uint32_t>((2 * jp + ci) * 1024), make_int4(R0 + I1, I0 - R1, R2 + I3, I2 - R3));
    }
}

// The whole life of one persistent CTA (CG = 1) or of one CTA of a pair (CG = 2): work unit `unit` of `nunits`
// walks the tile list of p.  `tmap` is the kernel's __grid_constant__ tensor map.
template <int UMMA_N, int CG, bool STAGED, bool TRACE, int BK_, bool DIAG>
__device__ __forceinline__ void tc_body(const CUtensorMap& tmap, const TcParams& p, const int unit, const int nunits) {
    using Cfg = TcCfg<UMMA_N, CG, STAGED, BK_, DIAG>;
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    // Barriers first, operand ring after, on a 1024-byte boundary (SWIZZLE_128B atoms).
    const uint32_t bar0 = smem_u32(smem_raw);
    auto full_bar = [&](uint32_t s) { return bar0 + 8u * s; };
    auto empty_bar = [&](uint32_t s) { return bar0 + 8u * (Cfg::STAGES + s); };
    auto tfull_bar = [&](uint32_t b) { return bar0 + 8u * (2 * Cfg::STAGES + b); };
    auto tempty_bar = [&](uint32_t b) { return bar0 + 8u * (2 * Cfg::STAGES + 2 + b); };
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem_raw + 8 * (2 * Cfg::STAGES + 4));
    const uint32_t ring0 = (bar0 + Cfg::BAR_BYTES + 1023u) & ~1023u;
    const uint32_t out0 = ring0 + Cfg::STAGES * Cfg::STAGE_BYTES;    // STAGED: packed output tile

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;
    const uint32_t rank = (CG == 2) ? cluster_ctarank() : 0u;         // 0 = leader of the CTA pair
    constexpr uint32_t TMEM_COLS = 2 * UMMA_N;                         // 512 or 256: a power of two >= 32

    if (warp == 0 && lane == 0) {
        tma_prefetch_desc(&tmap);
        for (int s = 0; s < Cfg::STAGES; ++s) {
            mbar_init(full_bar(s), 1);     // producer's arrive.expect_tx (+ TMA bytes of the whole pair)
            mbar_init(empty_bar(s), 1);    // tcgen05.commit (multicast to both CTAs when CG = 2)
        }
        for (int b = 0; b < 2; ++b) {
            mbar_init(tfull_bar(b), 1);            // tcgen05.commit
            mbar_init(tempty_bar(b), TC_EPI_WARPS * CG);   // one arrival per epilogue warp of the pair (on the leader)
        }
        fence_barrier_init();
    }
    if (warp == 1) {
        tmem_alloc<CG>(smem_u32(tmem_slot), TMEM_COLS);
        tmem_relinquish<CG>();
    }
    tc_fence_before();
    if (CG == 2) cluster_sync_all(); else __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;
    // Programmatic dependent launch: everything above (barrier init, TMEM allocation, descriptor prefetch) touched no
    // global memory and may overlap the tail of the previous kernel in the stream; from here on this kernel reads the
    // input / tile table and writes vis, so it first waits for that kernel to complete.  The next launch may in turn
    // begin its own prologue while this grid drains.
    pdl_grid_dependency_wait();
    pdl_launch_dependents();

    const int KB = (p.T + Cfg::BK - 1) / Cfg::BK;
    // profiling only: CTA 0 records (SM cycle counter, global nanosecond timer) at start and end, from which the
    // caller derives the SM clock the kernel really ran at (trace[3 * TC_TRACE_ITERS * 4 + 0..3])
    if (p.trace && blockIdx.x == 0 && threadIdx.x == 0) {
        unsigned long long gt;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(gt));
        p.trace[3 * TC_TRACE_ITERS * 4 + 0] = clock64();
        p.trace[3 * TC_TRACE_ITERS * 4 + 1] = static_cast<long long>(gt);
    }

    if (warp == 0) {
        // ===== TMA producer: the whole warp walks the loop, one elected lane issues =====
        const uint32_t elected = elect_one();
        uint32_t stage = 0, phase = 0;
        int it = 0;
        int w_next = walk(0, unit, nunits, p.group_shift, p.total_tiles);
        uint32_t tb_next = (w_next >= 0) ? __ldg(p.tiles + w_next % p.tiles_per_f) : 0u;
        for (int n = 0; w_next >= 0; ++n) {
            const int f = w_next / p.tiles_per_f;
            const uint32_t tb = __shfl_sync(0xffffffffu, tb_next, 0);
            // the next tile's table entry is fetched now so that its latency hides behind this tile's k loop
            w_next = walk(n + 1, unit, nunits, p.group_shift, p.total_tiles);
            if (w_next >= 0) tb_next = __ldg(p.tiles + w_next % p.tiles_per_f);
            if (tb == TC_TILE_EMPTY) continue;
            const int m_a = static_cast<int>(tb & 0xFFFFu) * Cfg::M + 128 * static_cast<int>(rank);
            const int m_b = static_cast<int>(tb >> 16) * UMMA_N + Cfg::B_BOXES * 128 * static_cast<int>(rank);
            const bool a_in_b = DIAG || ((m_a >= m_b) && (m_a < m_b + Cfg::B_BOXES * 128));   // diagonal: A rows are B rows
            // DIAG: a row block that lies in the tile's second column box needs nothing of the first one (every pair
            // there has i > j): only box 1 is loaded and the MMA shrinks to N = 128
            // Such a tile keeps 32 KB / 512 tensor cycles per stage by putting TWO time slices of box 1 into the stage's
            // two box slots (256 samples per stage): a 128-sample stage of N = 128 MMAs would hold only 256 tensor cycles,
            // less than the barrier round trip of a stage.
            // The same holds for the diagonal tile of the single-CTA 128x128 variant (A rows = B rows = one box).
            constexpr bool SOLO128 = (CG == 1 && UMMA_N == 128 && !STAGED);
            const int h0 = ((DIAG && m_a >= m_b + 128) || (SOLO128 && a_in_b)) ? 1 : 0;
            const int m_ts = DIAG ? m_b + 128 : m_b;       // rows of the one box a two-slice tile loads
            const uint32_t my_bytes = a_in_b ? static_cast<uint32_t>(Cfg::B_BYTES) : Cfg::STAGE_BYTES;
            const int KBt = h0 ? (p.T + 2 * Cfg::BK - 1) / (2 * Cfg::BK) : KB;
            for (int kb = 0; kb < KBt; ++kb) {
                const bool tr = TRACE && p.trace && blockIdx.x == 0 && it < TC_TRACE_ITERS && elected;
                if (tr) p.trace[(0 * TC_TRACE_ITERS + it) * 4 + 0] = clock64();
                mbar_wait(empty_bar(stage), phase ^ 1u);
                if (tr) p.trace[(0 * TC_TRACE_ITERS + it) * 4 + 1] = clock64();
                if (elected) {
                    const uint32_t sa = ring0 + stage * Cfg::STAGE_BYTES;
                    const uint32_t sb = sa + Cfg::A_BYTES;
                    const int t0 = kb * Cfg::BK * (1 + h0);
                    if ((p.debug_skip & 1) && (n != 0 || kb >= Cfg::STAGES)) {
                        if (rank == 0) mbar_arrive(full_bar(stage));
                    } else if ((DIAG || SOLO128) && h0) {
                        const bool two = t0 + Cfg::BK < p.T;     // the second time slice exists
                        mbar_arrive_expect_tx(full_bar(stage), two ? 2 * Cfg::BOX_BYTES : Cfg::BOX_BYTES);
                        tma_load_3d(sa, &tmap, full_bar(stage), m_ts, f, t0);
                        if (two) tma_load_3d(sa + Cfg::BOX_BYTES, &tmap, full_bar(stage), m_ts, f, t0 + Cfg::BK);
                    } else if (CG == 1) {
                        mbar_arrive_expect_tx(full_bar(stage), my_bytes);
                        if (!a_in_b) tma_load_3d(sa, &tmap, full_bar(stage), m_a, f, t0);
#pragma unroll
                        for (int h = 0; h < Cfg::B_BOXES; ++h)
                            tma_load_3d(sb + h * Cfg::BOX_BYTES, &tmap, full_bar(stage), m_b + 128 * h, f, t0);
                    } else {
                        // both CTAs' bytes are counted on the LEADER's barrier (a_in_b is the same in both)
                        const uint32_t lead_full = mapa_u32(full_bar(stage), 0);
                        if (rank == 0) mbar_arrive_expect_tx(full_bar(stage), 2 * my_bytes);
                        if (!a_in_b) tma_load_3d_2sm(sa, &tmap, lead_full, m_a, f, t0);
#pragma unroll
                        for (int h = 0; h < Cfg::B_BOXES; ++h)
                            tma_load_3d_2sm(sb + h * Cfg::BOX_BYTES, &tmap, lead_full, m_b + 128 * h, f, t0);
                    }
                }
                __syncwarp();
                if (tr) p.trace[(0 * TC_TRACE_ITERS + it) * 4 + 2] = clock64();
                ++it;
                if (++stage == Cfg::STAGES) {
                    stage = 0;
                    phase ^= 1u;
                }
            }
        }
    } else if (warp == 1) {
        // ===== MMA issuer: leader CTA only; warp-uniform loop, one elected lane issues =====
        if (rank == 0) {
            const uint32_t elected = elect_one();
            constexpr uint32_t idesc = make_idesc_i8_mn(Cfg::M, UMMA_N);
            uint32_t stage = 0, phase = 0, buf = 0, tphase = 0;   // tphase bit b = phase of accumulator b
            int it = 0;
            int w_next = walk(0, unit, nunits, p.group_shift, p.total_tiles);
            uint32_t tb_next = (w_next >= 0) ? __ldg(p.tiles + w_next % p.tiles_per_f) : 0u;
            for (int n = 0; w_next >= 0; ++n) {
                const uint32_t tb = __shfl_sync(0xffffffffu, tb_next, 0);
                w_next = walk(n + 1, unit, nunits, p.group_shift, p.total_tiles);
                if (w_next >= 0) tb_next = __ldg(p.tiles + w_next % p.tiles_per_f);
                if (tb == TC_TILE_EMPTY) continue;
                const int m_a = static_cast<int>(tb & 0xFFFFu) * Cfg::M;
                const int m_b = static_cast<int>(tb >> 16) * UMMA_N;
                const bool a_in_b = DIAG || ((m_a >= m_b) && (m_a < m_b + Cfg::B_BOXES * 128));
                // byte offset of the A operand inside a stage: its own box, or the B box holding the same rows
                // DIAG, row block in the second column box: N = 128 MMAs on box 1 (A = B = that box; the stage's two slots
                // hold two consecutive time slices of it) into the accumulator's upper 128 columns
                constexpr bool SOLO128 = (CG == 1 && UMMA_N == 128 && !STAGED);
                const uint32_t h0 = ((DIAG && m_a >= m_b + 128) || (SOLO128 && a_in_b)) ? 1u : 0u;
                const uint32_t a_off = h0 ? 0u : (a_in_b ? static_cast<uint32_t>(Cfg::A_BYTES + ((m_a - m_b) >> 7) * Cfg::BOX_BYTES) : 0u);
                const uint32_t idesc_t = h0 ? make_idesc_i8_mn(Cfg::M, 128) : idesc;
                const int BKt = Cfg::BK * (1 + static_cast<int>(h0));           // samples per stage of this tile
                const int KBt = (p.T + BKt - 1) / BKt;
                mbar_wait(tempty_bar(buf), ((tphase >> buf) & 1u) ^ 1u);  // epilogues have drained this accumulator
                tc_fence_after();
                const uint32_t d_tmem = tmem_base + buf * UMMA_N + (DIAG ? h0 * 128u : 0u);
                for (int kb = 0; kb < KBt; ++kb) {
                    const bool tr = TRACE && p.trace && blockIdx.x == 0 && it < TC_TRACE_ITERS && elected;
                    if (tr) p.trace[(1 * TC_TRACE_ITERS + it) * 4 + 0] = clock64();
                    mbar_wait(full_bar(stage), phase);
                    tc_fence_after();
                    if (tr) p.trace[(1 * TC_TRACE_ITERS + it) * 4 + 1] = clock64();
                    if (elected) {
                        const uint32_t sa = ring0 + stage * Cfg::STAGE_BYTES;
                        const uint64_t adesc = make_smem_desc_mn_sw128(sa + a_off, Cfg::BOX_BYTES, 1024);
                        const uint64_t bdesc = make_smem_desc_mn_sw128(sa + (h0 ? 0u : static_cast<uint32_t>(Cfg::A_BYTES)), Cfg::BOX_BYTES, 1024);
                        const int rows = min(BKt, p.T - kb * BKt);                // valid samples in this stage
                        const int nk = (rows + TC_UMMA_K - 1) / TC_UMMA_K;       // rows beyond T are TMA zero fill
#pragma unroll
                        for (int ks = 0; ks < ((DIAG || SOLO128) ? 2 : 1) * Cfg::BK / TC_UMMA_K; ++ks) {
                            if (ks < nk && !(p.debug_skip & 2)) {
                                // K advance: 32 samples = 4 swizzle atoms = 4096 B -> +256 in the address field
                                umma_i8<CG>(d_tmem, adesc + static_cast<uint64_t>(ks * 256),
                                            bdesc + static_cast<uint64_t>(ks * 256), idesc_t, (kb | ks) ? 1u : 0u);
                            }
                        }
                        if (tr) p.trace[(1 * TC_TRACE_ITERS + it) * 4 + 2] = clock64();
                        umma_commit<CG>(empty_bar(stage));  // frees the ring slot (in both CTAs) when these MMAs retire
                        if (kb == KBt - 1) umma_commit<CG>(tfull_bar(buf));  // accumulator complete -> epilogues
                    }
                    __syncwarp();
                    if (tr) p.trace[(1 * TC_TRACE_ITERS + it) * 4 + 3] = clock64();
                    ++it;
                    if (++stage == Cfg::STAGES) {
                        stage = 0;
                        phase ^= 1u;
                    }
                }
                tphase ^= 1u << buf;
                buf ^= 1u;
            }
        }
    } else {
        // ===== epilogue: warps 2..9; TMEM lane quarter = warp % 4, column half = (warp - 2) / 4 =====
        const int q = warp & 3;
        const int half = (warp - 2) >> 2;
        constexpr int CHUNKS = UMMA_N / 32 / 2;   // 32-column chunks per warp
        uint32_t buf = 0, tphase = 0;
        int it = 0;
        const uint32_t lead_tempty0 = (CG == 2) ? mapa_u32(tempty_bar(0), 0) : tempty_bar(0);
        int w_next = walk(0, unit, nunits, p.group_shift, p.total_tiles);
        uint32_t tb_next = (w_next >= 0) ? __ldg(p.tiles + w_next % p.tiles_per_f) : 0u;
        for (int n = 0; w_next >= 0; ++n) {
            const bool tr = TRACE && p.trace && blockIdx.x == 0 && it < TC_TRACE_ITERS && warp == 2 && lane == 0;
            if (tr) p.trace[(2 * TC_TRACE_ITERS + it) * 4 + 0] = clock64();
            const int f = w_next / p.tiles_per_f;
            const uint32_t tb = tb_next;
            w_next = walk(n + 1, unit, nunits, p.group_shift, p.total_tiles);
            if (w_next >= 0) tb_next = __ldg(p.tiles + w_next % p.tiles_per_f);
            if (tb == TC_TILE_EMPTY) continue;
            const int i0 = static_cast<int>(tb & 0xFFFFu) * Cfg::SI + 32 * static_cast<int>(rank) + 8 * q;
            // DIAG tile whose row block sits in the second column box: only accumulator columns 128..255 exist, and
            // all eight warps share them (two 32-column chunks each instead of four)
            const bool h0 = DIAG && (static_cast<int>(tb & 0xFFFFu) * Cfg::SI >= static_cast<int>(tb >> 16) * Cfg::SJ + 32);
            const int nchunks = h0 ? CHUNKS / 2 : CHUNKS;
            const int col0 = h0 ? 128 + 32 * nchunks * half : 32 * CHUNKS * half;    // first accumulator column of this warp
            const int j0 = static_cast<int>(tb >> 16) * Cfg::SJ + col0 / 4;           // first station of this warp's columns
            const int i = i0 + (lane >> 2);                     // i0 = first station of this warp's rows
            int32_t* visf = p.vis + static_cast<long long>(f) * p.NB * 8;

            mbar_wait(tfull_bar(buf), (tphase >> buf) & 1u);
            tc_fence_after();
            if (tr) p.trace[(2 * TC_TRACE_ITERS + it) * 4 + 1] = clock64();
            const uint32_t taddr0 = tmem_base + (static_cast<uint32_t>(32 * q) << 16) + buf * UMMA_N + col0;
            if (STAGED) {
                // the previous tile's bulk stores must have finished reading the staging buffer
                if (warp < 4) bulk_wait_read0();            // warps 2-3 issue the bulk stores
                named_bar_sync(1, 32 * TC_EPI_WARPS);
            }
#pragma unroll 1
            for (int cc = 0; cc < nchunks; ++cc) {
                const int jbase = j0 + 8 * cc;
                if (jbase >= p.N || jbase + 7 < i0) continue;  // warp-uniform: nothing of this chunk is stored
                uint32_t v[32];
                tmem_ld_32x32(taddr0 + static_cast<uint32_t>(32 * cc), v);
                tmem_ld_wait();
                const bool full = (i0 + 7 <= jbase) && (jbase + 7 < p.N);  // warp-uniform: no masking needed
                if (STAGED) {
                    // row (j - tile's first j) of the staging buffer, 32 bytes per station i of this CTA, 16 per pol_i
                    const uint32_t dst = out0 + static_cast<uint32_t>((8 * (CHUNKS * half + cc)) * 1024 +
                                                                       (8 * q + (lane >> 2)) * 32 + ((lane >> 1) & 1) * 16);
                    epi_chunk_smem(v, dst, lane);
                } else if (p.debug_skip & 4) {
                    epi_chunk<true, false, true>(v, visf, i, jbase, p.N, lane);
                } else if (p.debug_skip & 8) {
                    epi_chunk<true, false, false, true>(v, p.vis, i, jbase, p.N, lane);
                } else if (p.accumulate) {
                    if (full) epi_chunk<false, true>(v, visf, i, jbase, p.N, lane);
                    else epi_chunk<true, true>(v, visf, i, jbase, p.N, lane);
                } else {
                    if (full) epi_chunk<false, false>(v, visf, i, jbase, p.N, lane);
                    else epi_chunk<true, false>(v, visf, i, jbase, p.N, lane);
                }
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) {
                if (CG == 2) mbar_arrive_cluster(lead_tempty0 + 8u * buf);
                else mbar_arrive(tempty_bar(buf));
            }
            if (STAGED) {
                fence_proxy_async();                         // my st.shared -> visible to the bulk-copy engine
                named_bar_sync(1, 32 * TC_EPI_WARPS);        // the whole tile is packed
                const int e = static_cast<int>(threadIdx.x) - 64;   // epilogue thread index; thread e stores row e
                if (e < Cfg::SJ && !(p.debug_skip & 4)) {
                    const int ic = i0 - 8 * q;                       // first station of this CTA's 32 rows
                    const int j = static_cast<int>(tb >> 16) * Cfg::SJ + e;
                    const int last = min(min(ic + 31, j), p.N - 1);  // stored pairs of row j: ic <= i <= last (a prefix)
                    if (j < p.N && last >= ic) {
                        int32_t* g = visf + (static_cast<long long>(j) * (j + 1) / 2 + ic) * 8;
                        const uint32_t bytes = static_cast<uint32_t>(last - ic + 1) * 32u;
                        if (p.accumulate) bulk_reduce_add_s32(g, out0 + e * 1024, bytes);
                        else bulk_store(g, out0 + e * 1024, bytes);
                    }
                    bulk_commit();
                }
            }
            if (tr) p.trace[(2 * TC_TRACE_ITERS + it) * 4 + 2] = clock64();
            ++it;
            tphase ^= 1u << buf;
            buf ^= 1u;
        }
    }

    if (p.trace && blockIdx.x == 0 && threadIdx.x == 64) {   // an epilogue thread: it finishes last
        unsigned long long gt;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(gt));
        p.trace[3 * TC_TRACE_ITERS * 4 + 2] = clock64();
        p.trace[3 * TC_TRACE_ITERS * 4 + 3] = static_cast<long long>(gt);
    }
    if (STAGED && warp >= 2 && warp < 4) bulk_wait0();   // the CTA's shared memory must outlive its bulk stores
    // Teardown: nobody leaves (or frees TMEM) while the peer may still signal into this CTA.
    tc_fence_before();
    if (CG == 2) cluster_sync_all(); else __syncthreads();
    if (warp == 1) {
        __syncwarp();
        tc_fence_after();
        tmem_dealloc<CG>(tmem_base, TMEM_COLS);
    }
}

// One tile shape per launch: every CTA (CG = 1) or CTA pair (CG = 2, cluster of 2) is one work unit.
template <int UMMA_N, int CG, bool STAGED, bool TRACE = false, int BK_ = 128, bool DIAG = false>
__global__ void __launch_bounds__(TC_THREADS, 1)
xc_i8_tc_kernel(const __grid_constant__ CUtensorMap tmap, const TcParams p) {
    tc_body<UMMA_N, CG, STAGED, TRACE, BK_, DIAG>(tmap, p, static_cast<int>(blockIdx.x) / CG, static_cast<int>(gridDim.x) / CG);
}

// XC_TILE_MIXED: ONE launch in clusters of 2 in which the first n_solo_clusters clusters are two independent
// single-CTA workers on the diagonal 64-station blocks (pd: DIAG sub-tiles, tcgen05 cta_group::1 only) and the other
// clusters are CTA pairs on the off-diagonal 256x256 tiles (po: cta_group::2 only).  A given CTA executes
// tcgen05 instructions of one cta_group only, for its whole life.  Both kinds of worker walk the channels in the
// same order at a rate balanced by the host, so a channel's input is fetched from HBM once and shared through L2
// (two separate launches would each read the whole input from HBM: measured).
__global__ void __launch_bounds__(TC_THREADS, 1)
xc_i8_tc_mixed_kernel(const __grid_constant__ CUtensorMap tmap, const TcParams pd, const TcParams po, const int n_solo_clusters) {
    const int cluster = static_cast<int>(blockIdx.x >> 1);
    if (cluster < n_solo_clusters)
        tc_body<256, 1, false, false, 128, true>(tmap, pd, static_cast<int>(blockIdx.x), 2 * n_solo_clusters);
    else
        tc_body<256, 2, false, false, 128, false>(tmap, po, cluster - n_solo_clusters,
                                                  static_cast<int>(gridDim.x >> 1) - n_solo_clusters);
}

}  // namespace xc
