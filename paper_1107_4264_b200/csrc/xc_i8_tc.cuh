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
// Two tile shapes are built (every other shape tried in round 1 measured slower):
//   CG = 2: 256 Gram rows (64 stations) x 256 columns (64 stations) on a CTA pair (tcgen05
//           cta_group::2): each CTA holds its own 128 A rows and 128 of the 256 B rows, so every
//           operand byte is fetched from L2 and written to shared memory once per pair.
//   CG = 1: 128 x 128 (32 x 32 stations) on one CTA, for small N.  With TS = 2 the T samples of one
//           tile are split over the two CTAs of a cluster ("T-split"; the paper's
//           small-N future work): rank 1 hands its int32 partial accumulators to
//           rank 0 through distributed shared memory, rank 0 adds them to its own and stores --
//           integer addition, so the result stays bit-exact and independent of the split.
// K (= time) advances BK samples per ring stage, 32 per tcgen05.mma.  Time is the slowest input
// index, so both operands are MN-major in shared memory: a TMA box
// [BK t][1 f][128 B of m] lands as BK rows of 128 bytes, which is exactly the SWIZZLE_128B
// MN-major canonical layout (8-row atoms of 1024 B).  Two TMEM accumulators (2 x UMMA_N columns)
// let the epilogue of tile k overlap the MMAs of tile k+1.  On tiles that touch the diagonal the
// A rows are the CTA's B rows: they are loaded once and both descriptors point at them.
//
// Producer and MMA loops run warp-uniformly (all 32 lanes walk the loop, one elected lane issues)
// so that addresses, coordinates and descriptors stay in uniform registers: a single-lane branch
// costs ~80 cycles per TMA / MMA issue in register->uniform-register waterfalls, which at 128
// tensor cycles per MMA starves the pipe (measured).
//
// Profiling hooks (per-iteration clock stamps, switches that drop loads / MMAs / stores) exist only in
// builds with -DXC_PROFILE (python -m paper_1107_4264_b200.build --profile -> libxc_profile.so).
#pragma once
#include "xc_ptx.cuh"

namespace xc {

constexpr int TC_UMMA_K = 32;      // samples per tcgen05.mma (kind::i8)
constexpr int TC_EPI_WARPS = 8;     // 2 per TMEM lane quarter, each owning half of the tile's columns
constexpr int TC_THREADS = 64 + 32 * TC_EPI_WARPS;   // + TMA producer warp + MMA issuer warp
constexpr int TC_SMEM_LIMIT = 232448;  // 227 KB
constexpr int TC_INLINE_TILES = 48;    // tile tables up to this size travel in the kernel parameters

template <int UMMA_N, int CG, int BK_, int TS_>
struct TcCfg {
    static_assert((CG == 2 && UMMA_N == 256 && TS_ == 1) || (CG == 1 && UMMA_N == 128 && (TS_ == 1 || TS_ == 2)),
                  "built shapes: CTA-pair 256x256, single-CTA 128x128 (optionally T-split over a cluster of 2)");
    static constexpr int TS = TS_;                        // CTAs that share one tile's time axis (cluster size if CG == 1)
    static constexpr int M = 128 * CG;                    // Gram rows per tile
    // Samples per pipeline stage.  Every stage costs the producer and the MMA issuer some hundred cycles of
    // barrier round trips and instruction issue (measured), so a stage must hold clearly more than that in
    // tensor work: 512 tensor cycles = 128 samples of the pair tile = 256 samples of the 128 x 128 tile.
    static constexpr int BK = BK_;
    static constexpr int BOX_BYTES = BK * 128;            // one TMA box: BK rows of 128 bytes
    static constexpr int STAGE_BYTES = 2 * BOX_BYTES;     // A box + this CTA's B box
    static constexpr int SI = 32 * CG;                    // stations per tile on the i side
    static constexpr int SJ = UMMA_N / 4;                 // stations per tile on the j side
    static constexpr int RED_BYTES = (TS - 1) * 128 * UMMA_N * 4;       // T-split: partial accumulators of the other rank
    static constexpr int STAGES = (229376 - RED_BYTES) / STAGE_BYTES;   // 224 KB for ring + reduction buffer
    static constexpr int BAR_BYTES = 1024;                // barriers + tmem slot, kept in the first KB
    static constexpr int SMEM_BYTES = BAR_BYTES + STAGES * STAGE_BYTES + RED_BYTES + 1024;  // + slack for 1024-B alignment
    static_assert(SMEM_BYTES <= TC_SMEM_LIMIT, "smem");
    static_assert(STAGES >= 2, "ring too shallow");
};

struct TcParams {
    int N, F, T;
    int tiles_per_f;          // entries of the tile table (the largest per-channel count of any alignment class)
    int total_tiles;          // sum over the F channels of their tile counts
    // Origin shift: when the rows of the block are not 128 bytes apart, channel f's rows start `shift` bytes
    // past a 128-byte line; its tile grid is then moved `shift` bytes (shift / 4 stations) to the left, so that every box row
    // is one whole L2 line (coordinates below 0 are TMA zero fill, masked in the epilogue).  The shift depends on
    // f mod per_n only; class c has per_cum[c + 1] - per_cum[c] tiles (a prefix of the table).
    int per_n;                // channels per alignment period: 1, 2, 4 or 8
    int per_total;            // tiles of one period = per_cum[per_n]
    uint32_t per_cum[9];
    uint8_t per_shift[8];     // bytes, multiples of 16, < 128
    int t_split;              // T-split: samples per rank (a multiple of 32); T when TS == 1
    long long NB;             // N(N+1)/2
    const uint32_t* tiles;    // device: bi | (bj << 16), in units of (SI, SJ) stations (used if tiles_per_f > TC_INLINE_TILES)
    int32_t* vis;
    int accumulate;
    // xc_set_timing_buffer: [0] min over CTAs of globaltimer at kernel entry, [1] max at exit (atomics; the caller
    // presets [0] = ~0, [1] = 0), [2..5] CTA 0's (clock64, globaltimer) at entry and exit; or null
    unsigned long long* stamps;
#ifdef XC_PROFILE
    int debug_skip;           // 1 = no TMA after the first ring fill, 2 = no MMA, 4 = no global stores, 8 = stores wrapped
    long long* trace;         // CTA 0 writes clock64() stamps here (see TC_TRACE_*), or null
#endif
    uint32_t tiles_inline[TC_INLINE_TILES];
};
constexpr int TC_TRACE_ITERS = 256;   // pipeline iterations traced; layout: [3 roles][TC_TRACE_ITERS][4] long long

#ifdef XC_PROFILE
#define XC_TRACE_STAMP(p, cond, role, it, slot) do { if ((p).trace && (cond) && (it) < TC_TRACE_ITERS) \
        (p).trace[((role) * TC_TRACE_ITERS + (it)) * 4 + (slot)] = clock64(); } while (0)
#define XC_SKIP(p, bit) (((p).debug_skip & (bit)) != 0)
#else
#define XC_TRACE_STAMP(p, cond, role, it, slot) do { } while (0)
#define XC_SKIP(p, bit) false
#endif

// The persistent walk (S1): work unit `unit` of `nunits` takes entries unit, unit + nunits, ... of the
// (channel-major) tile list.  Returns the global entry index, or -1 past the end.
__device__ __forceinline__ int walk(int n, int unit, int nunits, int total) {
    const long long w = static_cast<long long>(unit) + static_cast<long long>(n) * nunits;
    return w < total ? static_cast<int>(w) : -1;
}
// Entry w of the tile list -> channel, index into the tile table, origin shift of that channel (in bytes).
struct TcWork {
    int f, k, shift;
};
__device__ __forceinline__ TcWork tc_locate(const TcParams& p, int w) {
    TcWork r;
    const int per = w / p.per_total;
    const int rem = w - per * p.per_total;
    int c = 0;
    while (c + 1 < p.per_n && rem >= static_cast<int>(p.per_cum[c + 1])) ++c;
    r.f = per * p.per_n + c;
    r.k = rem - static_cast<int>(p.per_cum[c]);
    r.shift = static_cast<int>(p.per_shift[c]);
    return r;
}
// Tile table entry k of a channel: from the kernel parameters (constant bank: no global-memory latency in front of the
// first TMA load, which matters for microsecond-scale launches) or, for long tables, from global memory.
__device__ __forceinline__ uint32_t tile_at(const TcParams& p, int k) {
    return p.tiles_per_f <= TC_INLINE_TILES ? p.tiles_inline[k] : __ldg(p.tiles + k);
}

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
        if ((!MASKED || (i >= 0 && i <= j && j < N)) && !NOSTORE) {
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

// The whole life of one persistent CTA (CG = 1; TS = 2: of one CTA of a T-split cluster) or of one CTA of a pair
// (CG = 2): work unit `unit` of `nunits` walks the tile list of p.  `tmap` is the kernel's __grid_constant__ tensor map.
template <int UMMA_N, int CG, int BK_, int TS>
__device__ __forceinline__ void tc_body(const CUtensorMap& tmap, const TcParams& p, const int unit, const int nunits) {
    using Cfg = TcCfg<UMMA_N, CG, BK_, TS>;
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    // Barriers first, operand ring after, on a 1024-byte boundary (SWIZZLE_128B atoms).
    const uint32_t bar0 = smem_u32(smem_raw);
    auto full_bar = [&](uint32_t s) { return bar0 + 8u * s; };
    auto empty_bar = [&](uint32_t s) { return bar0 + 8u * (Cfg::STAGES + s); };
    auto tfull_bar = [&](uint32_t b) { return bar0 + 8u * (2 * Cfg::STAGES + b); };
    auto tempty_bar = [&](uint32_t b) { return bar0 + 8u * (2 * Cfg::STAGES + 2 + b); };
    const uint32_t pready_bar = bar0 + 8u * (2 * Cfg::STAGES + 4);   // T-split, in rank 0: rank 1's partial tile has landed
    const uint32_t pfree_bar = bar0 + 8u * (2 * Cfg::STAGES + 5);    // T-split, in rank 1: rank 0 has consumed it
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem_raw + 8 * (2 * Cfg::STAGES + 6));
    const uint32_t ring0 = (bar0 + Cfg::BAR_BYTES + 1023u) & ~1023u;
    const uint32_t red0 = ring0 + Cfg::STAGES * Cfg::STAGE_BYTES;    // T-split: reduction buffer (used in rank 0)

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;
    const uint32_t rank = (CG == 2 || TS == 2) ? cluster_ctarank() : 0u;   // CG = 2: 0 = leader of the pair; TS = 2: time half
    constexpr uint32_t TMEM_COLS = 2 * UMMA_N;                         // 512 or 256: a power of two >= 32
    constexpr bool CLUSTER = (CG == 2 || TS == 2);

    // timing stamps are taken by the last epilogue warp, which has nothing to do until the first accumulator is complete:
    // reading %globaltimer takes several hundred cycles and must not sit in the producer's or the issuer's path
    if (p.stamps && threadIdx.x == TC_THREADS - 32) {
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
        for (int s = 0; s < Cfg::STAGES; ++s) {
            mbar_init(full_bar(s), 1);     // producer's arrive.expect_tx (+ TMA bytes of the whole pair)
            mbar_init(empty_bar(s), 1);    // tcgen05.commit (multicast to both CTAs when CG = 2)
        }
        for (int b = 0; b < 2; ++b) {
            mbar_init(tfull_bar(b), 1);            // tcgen05.commit
            mbar_init(tempty_bar(b), TC_EPI_WARPS * CG);   // one arrival per epilogue warp of the pair (on the leader)
        }
        mbar_init(pready_bar, TC_EPI_WARPS);       // T-split: one arrival per epilogue warp of the other rank
        mbar_init(pfree_bar, TC_EPI_WARPS);
        fence_barrier_init();
    }
    // Rendezvous 1 (CTA or cluster): the barriers exist.  Threads only ARRIVE here; the TMEM allocation (several hundred
    // cycles) happens between arrive and wait, and the TMA producer, which needs no TMEM, leaves as soon as everybody has
    // arrived -- its first loads are in flight while warp 1 still allocates (-0.3 us on the microsecond-scale launches).
    if (CLUSTER) cluster_arrive_relaxed(); else __syncthreads();
    if (warp == 1) {
        tmem_alloc<CG>(smem_u32(tmem_slot), TMEM_COLS);
        tmem_relinquish<CG>();
        tc_fence_before();
    }
    if (CLUSTER) cluster_wait();
    uint32_t tmem_base = 0;
    if (warp != 0) {
        // Rendezvous 2 (MMA issuer + epilogue warps of this CTA): the TMEM base address is in shared memory
        named_bar_sync(1, TC_THREADS - 32);
        tc_fence_after();
        tmem_base = *tmem_slot;
    }
    // Programmatic dependent launch: everything above (barrier init, TMEM allocation, descriptor prefetch) touched no
    // global memory that a predecessor writes and may overlap the tail of the previous kernel in the stream; from here
    // on this kernel reads the input / tile table and writes vis, so it first waits for that kernel to complete.  The
    // next launch may in turn begin its own prologue while this grid drains.
    pdl_grid_dependency_wait();
    pdl_launch_dependents();

    // T-split: this CTA's share of the time axis (whole multiples of the MMA's K = 32, so a share ends on a K step)
    const int t_lo = (TS == 2) ? static_cast<int>(rank) * p.t_split : 0;
    const int t_hi = (TS == 2) ? min(p.T, t_lo + p.t_split) : p.T;
    const int Tr = t_hi - t_lo;                       // >= 1 (the host guarantees it)
    const int KB = (Tr + Cfg::BK - 1) / Cfg::BK;

    if (warp == 0) {
        // ===== TMA producer: the whole warp walks the loop, one elected lane issues =====
        const uint32_t elected = elect_one();
        uint32_t stage = 0, phase = 0;
        int it = 0;
        int w_next = walk(0, unit, nunits, p.total_tiles);
        TcWork wk_next = tc_locate(p, w_next >= 0 ? w_next : 0);
        uint32_t tb_next = (w_next >= 0) ? tile_at(p, wk_next.k) : 0u;
        for (int n = 0; w_next >= 0; ++n) {
            const int f = wk_next.f, shift = wk_next.shift;
            const uint32_t tb = __shfl_sync(0xffffffffu, tb_next, 0);
            // the next tile's table entry is fetched now so that its latency hides behind this tile's k loop
            w_next = walk(n + 1, unit, nunits, p.total_tiles);
            if (w_next >= 0) {
                wk_next = tc_locate(p, w_next);
                tb_next = tile_at(p, wk_next.k);
            }
            const int m_a = static_cast<int>(tb & 0xFFFFu) * Cfg::M + ((CG == 2) ? 128 * static_cast<int>(rank) : 0) - shift;
            const int m_b = static_cast<int>(tb >> 16) * UMMA_N + ((CG == 2) ? 128 * static_cast<int>(rank) : 0) - shift;
            const bool a_in_b = (m_a == m_b);     // diagonal tile: this CTA's A rows are its B rows -- one box serves both
            // A diagonal tile of the single-CTA kernel puts TWO consecutive time slices of its one box into the stage's two
            // slots (2 x BK samples per stage), so that a stage holds 512 tensor cycles like every other tile.
            const int h0 = (CG == 1 && a_in_b) ? 1 : 0;
            const uint32_t my_bytes = (a_in_b && !h0) ? static_cast<uint32_t>(Cfg::BOX_BYTES) : Cfg::STAGE_BYTES;
            const int KBt = h0 ? (Tr + 2 * Cfg::BK - 1) / (2 * Cfg::BK) : KB;
            for (int kb = 0; kb < KBt; ++kb) {
                XC_TRACE_STAMP(p, blockIdx.x == 0 && elected, 0, it, 0);
                mbar_wait(empty_bar(stage), phase ^ 1u);
                XC_TRACE_STAMP(p, blockIdx.x == 0 && elected, 0, it, 1);
                if (elected) {
                    const uint32_t sa = ring0 + stage * Cfg::STAGE_BYTES;
                    const uint32_t sb = sa + Cfg::BOX_BYTES;
                    const int t0 = t_lo + kb * Cfg::BK * (1 + h0);
                    if (XC_SKIP(p, 1) && (n != 0 || kb >= Cfg::STAGES)) {
                        if (rank == 0 || CG == 1) mbar_arrive(full_bar(stage));
                    } else if (h0) {
                        const bool two = t0 + Cfg::BK < t_hi;     // the second time slice exists
                        mbar_arrive_expect_tx(full_bar(stage), two ? 2 * Cfg::BOX_BYTES : Cfg::BOX_BYTES);
                        tma_load_3d(sa, &tmap, full_bar(stage), m_b, f, t0);
                        if (two) tma_load_3d(sb, &tmap, full_bar(stage), m_b, f, t0 + Cfg::BK);
                    } else if (CG == 1) {
                        mbar_arrive_expect_tx(full_bar(stage), my_bytes);
                        if (!a_in_b) tma_load_3d(sa, &tmap, full_bar(stage), m_a, f, t0);
                        tma_load_3d(sb, &tmap, full_bar(stage), m_b, f, t0);
                    } else {
                        // both CTAs' bytes are counted on the LEADER's barrier (a_in_b is the same in both)
                        const uint32_t lead_full = mapa_u32(full_bar(stage), 0);
                        if (rank == 0) mbar_arrive_expect_tx(full_bar(stage), 2 * my_bytes);
                        if (!a_in_b) tma_load_3d_2sm(sa, &tmap, lead_full, m_a, f, t0);
                        tma_load_3d_2sm(sb, &tmap, lead_full, m_b, f, t0);
                    }
                }
                __syncwarp();
                XC_TRACE_STAMP(p, blockIdx.x == 0 && elected, 0, it, 2);
                ++it;
                if (++stage == Cfg::STAGES) {
                    stage = 0;
                    phase ^= 1u;
                }
            }
        }
    } else if (warp == 1) {
        // ===== MMA issuer: leader CTA only (CG = 2); warp-uniform loop, one elected lane issues =====
        if (rank == 0 || CG == 1) {
            const uint32_t elected = elect_one();
            constexpr uint32_t idesc = make_idesc_i8_mn(Cfg::M, UMMA_N);
            uint32_t stage = 0, phase = 0, buf = 0, tphase = 0;   // tphase bit b = phase of accumulator b
            int it = 0;
            int w_next = walk(0, unit, nunits, p.total_tiles);
            uint32_t tb_next = (w_next >= 0) ? tile_at(p, tc_locate(p, w_next).k) : 0u;
            for (int n = 0; w_next >= 0; ++n) {
                const uint32_t tb = __shfl_sync(0xffffffffu, tb_next, 0);
                w_next = walk(n + 1, unit, nunits, p.total_tiles);
                if (w_next >= 0) tb_next = tile_at(p, tc_locate(p, w_next).k);
                const bool a_in_b = ((tb & 0xFFFFu) * Cfg::M == (tb >> 16) * UMMA_N);
                const uint32_t h0 = (CG == 1 && a_in_b) ? 1u : 0u;
                // byte offset of the A operand inside a stage: its own box (slot 0), or -- pair kernel on the diagonal -- the B box
                const uint32_t a_off = (a_in_b && !h0) ? static_cast<uint32_t>(Cfg::BOX_BYTES) : 0u;
                const uint32_t b_off = h0 ? 0u : static_cast<uint32_t>(Cfg::BOX_BYTES);
                const int BKt = Cfg::BK * (1 + static_cast<int>(h0));           // samples per stage of this tile
                const int KBt = (Tr + BKt - 1) / BKt;
                mbar_wait(tempty_bar(buf), ((tphase >> buf) & 1u) ^ 1u);  // epilogues have drained this accumulator
                tc_fence_after();
                const uint32_t d_tmem = tmem_base + buf * UMMA_N;
                for (int kb = 0; kb < KBt; ++kb) {
                    XC_TRACE_STAMP(p, blockIdx.x == 0 && elected, 1, it, 0);
                    mbar_wait(full_bar(stage), phase);
                    tc_fence_after();
                    XC_TRACE_STAMP(p, blockIdx.x == 0 && elected, 1, it, 1);
                    if (elected) {
                        const uint32_t sa = ring0 + stage * Cfg::STAGE_BYTES;
                        const uint64_t adesc = make_smem_desc_mn_sw128(sa + a_off, Cfg::BOX_BYTES, 1024);
                        const uint64_t bdesc = make_smem_desc_mn_sw128(sa + b_off, Cfg::BOX_BYTES, 1024);
                        const int rows = min(BKt, Tr - kb * BKt);                 // valid samples in this stage
                        const int nk = (rows + TC_UMMA_K - 1) / TC_UMMA_K;       // rows beyond T are TMA zero fill
#pragma unroll
                        for (int ks = 0; ks < ((CG == 1) ? 2 : 1) * Cfg::BK / TC_UMMA_K; ++ks) {
                            if (ks < nk && !XC_SKIP(p, 2)) {
                                // K advance: 32 samples = 4 swizzle atoms = 4096 B -> +256 in the address field (a two-slice
                                // stage simply runs on into its second box, which follows the first in shared memory)
                                umma_i8<CG>(d_tmem, adesc + static_cast<uint64_t>(ks * 256),
                                            bdesc + static_cast<uint64_t>(ks * 256), idesc, (kb | ks) ? 1u : 0u);
                            }
                        }
                        XC_TRACE_STAMP(p, blockIdx.x == 0, 1, it, 2);
                        umma_commit<CG>(empty_bar(stage));  // frees the ring slot (in both CTAs) when these MMAs retire
                        if (kb == KBt - 1) umma_commit<CG>(tfull_bar(buf));  // accumulator complete -> epilogues
                    }
                    __syncwarp();
                    XC_TRACE_STAMP(p, blockIdx.x == 0 && elected, 1, it, 3);
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
        uint32_t buf = 0, tphase = 0, pphase = 0;
        int it = 0;
        const uint32_t lead_tempty0 = (CG == 2) ? mapa_u32(tempty_bar(0), 0) : tempty_bar(0);
        // T-split: this warp's slice of the reduction buffer, [chunk][8 x int4][32 lanes]: a warp access is 512 contiguous bytes
        const uint32_t red_w = red0 + static_cast<uint32_t>(((warp - 2) * CHUNKS) * 4096 + lane * 16);
        int w_next = walk(0, unit, nunits, p.total_tiles);
        TcWork wk_next = tc_locate(p, w_next >= 0 ? w_next : 0);
        uint32_t tb_next = (w_next >= 0) ? tile_at(p, wk_next.k) : 0u;
        for (int n = 0; w_next >= 0; ++n) {
            XC_TRACE_STAMP(p, blockIdx.x == 0 && warp == 2 && lane == 0, 2, it, 0);
            const int f = wk_next.f;
            const int ds = wk_next.shift >> 2;                  // origin shift in stations: the tile grid starts at station -ds
            const uint32_t tb = tb_next;
            w_next = walk(n + 1, unit, nunits, p.total_tiles);
            if (w_next >= 0) {
                wk_next = tc_locate(p, w_next);
                tb_next = tile_at(p, wk_next.k);
            }
            const int i0 = static_cast<int>(tb & 0xFFFFu) * Cfg::SI + ((CG == 2) ? 32 * static_cast<int>(rank) : 0) + 8 * q - ds;
            const int col0 = 32 * CHUNKS * half;                                     // first accumulator column of this warp
            const int j0 = static_cast<int>(tb >> 16) * Cfg::SJ + col0 / 4 - ds;      // first station of this warp's columns
            const int i = i0 + (lane >> 2);                     // i0 = first station of this warp's rows
            int32_t* visf = p.vis + static_cast<long long>(f) * p.NB * 8;

            mbar_wait(tfull_bar(buf), (tphase >> buf) & 1u);
            tc_fence_after();
            XC_TRACE_STAMP(p, blockIdx.x == 0 && warp == 2 && lane == 0, 2, it, 1);
            const uint32_t taddr0 = tmem_base + (static_cast<uint32_t>(32 * q) << 16) + buf * UMMA_N + col0;
            if (TS == 2 && rank == 1) {
                // hand the partial accumulators to rank 0: wait until it has consumed the previous tile's, copy, signal
                mbar_wait(pfree_bar, pphase ^ 1u);
                const uint32_t dst = mapa_u32(red_w, 0);
#pragma unroll 1
                for (int cc = 0; cc < CHUNKS; ++cc) {
                    uint32_t v[32];
                    tmem_ld_32x32(taddr0 + static_cast<uint32_t>(32 * cc), v);
                    tmem_ld_wait();
#pragma unroll
                    for (int k = 0; k < 8; ++k)
                        st_shared_cluster_v4(dst + static_cast<uint32_t>(cc * 4096 + k * 512),
                                             make_int4(static_cast<int>(v[4 * k]), static_cast<int>(v[4 * k + 1]),
                                                       static_cast<int>(v[4 * k + 2]), static_cast<int>(v[4 * k + 3])));
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) {
                    mbar_arrive(tempty_bar(buf));
                    mbar_arrive_release_cluster(mapa_u32(pready_bar, 0));   // release: the stores above are visible to rank 0
                }
            } else {
                if (TS == 2) mbar_wait_acquire_cluster(pready_bar, pphase);   // rank 1's partial tile is in red0
#pragma unroll 1
                for (int cc = 0; cc < CHUNKS; ++cc) {
                    const int jbase = j0 + 8 * cc;
                    if (jbase >= p.N || jbase + 7 < i0 || jbase + 7 < 0) continue;  // warp-uniform: nothing of this chunk is stored
                    uint32_t v[32];
                    tmem_ld_32x32(taddr0 + static_cast<uint32_t>(32 * cc), v);
                    tmem_ld_wait();
                    if (TS == 2) {
#pragma unroll
                        for (int k = 0; k < 8; ++k) {
                            const int4 o = ld_shared_v4(red_w + static_cast<uint32_t>(cc * 4096 + k * 512));
                            v[4 * k] += static_cast<uint32_t>(o.x);
                            v[4 * k + 1] += static_cast<uint32_t>(o.y);
                            v[4 * k + 2] += static_cast<uint32_t>(o.z);
                            v[4 * k + 3] += static_cast<uint32_t>(o.w);
                        }
                    }
                    const bool full = (i0 >= 0) && (i0 + 7 <= jbase) && (jbase + 7 < p.N);  // warp-uniform: no masking needed
#ifdef XC_PROFILE
                    if (p.debug_skip & 4) { epi_chunk<true, false, true>(v, visf, i, jbase, p.N, lane); continue; }
                    if (p.debug_skip & 8) { epi_chunk<true, false, false, true>(v, p.vis, i, jbase, p.N, lane); continue; }
#endif
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
                if (lane == 0) {
                    if (CG == 2) mbar_arrive_cluster(lead_tempty0 + 8u * buf);
                    else mbar_arrive(tempty_bar(buf));
                    // the reduction buffer has been read (the loads above have returned their values): rank 1 may refill it
                    if (TS == 2) mbar_arrive_cluster(mapa_u32(pfree_bar, 1));
                }
            }
            XC_TRACE_STAMP(p, blockIdx.x == 0 && warp == 2 && lane == 0, 2, it, 2);
            ++it;
            tphase ^= 1u << buf;
            buf ^= 1u;
            pphase ^= 1u;
        }
    }

    // Teardown: nobody leaves (or frees TMEM) while a peer may still signal into this CTA (execution ordering only: the
    // kernel's end makes the global stores visible, a release here would only wait for them).
    tc_fence_before();
    if (CLUSTER) cluster_sync_relaxed(); else __syncthreads();
    if (warp == 1) {
        __syncwarp();
        tc_fence_after();
        tmem_dealloc<CG>(tmem_base, TMEM_COLS);
    }
    if (p.stamps && threadIdx.x == TC_THREADS - 32) {
        const unsigned long long c = static_cast<unsigned long long>(clock64());
        const unsigned long long gt = globaltimer_ns();
        atomicMax(p.stamps + 1, gt);
        if (blockIdx.x == 0) {
            p.stamps[4] = c;
            p.stamps[5] = gt;
        }
    }
}

// One tile shape per launch: every CTA (CG = 1), T-split cluster (TS = 2) or CTA pair (CG = 2) is one work unit.
template <int UMMA_N, int CG, int BK_, int TS>
__global__ void __launch_bounds__(TC_THREADS, 1)
xc_i8_tc_kernel(const __grid_constant__ CUtensorMap tmap, const __grid_constant__ TcParams p) {
    constexpr int CL = CG * TS;     // cluster size
    tc_body<UMMA_N, CG, BK_, TS>(tmap, p, static_cast<int>(blockIdx.x) / CL, static_cast<int>(gridDim.x) / CL);
}

}  // namespace xc
