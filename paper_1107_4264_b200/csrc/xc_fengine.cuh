// xc_fengine.cuh -- F-engine + corner turn in front of the X-engine.
//
// What it computes: for every station s, polarisation p and time block t the F-point Fourier transform
//      X[t][f][s][p] = sum_{k<F} volt[s][p][t*F + k] * exp(-2 pi i f k / F)
// of complex int8 voltages ("N (fast) Fourier transforms of length F ... once every F samples", PAPER.md:63 fn. 2),
// quantised to the X-engine's int8 (q = clip(rint(X * scale), -127, 127), "four to eight bits ... sufficient for both the
// Fourier transform and cross-multiplication") and written in the X-engine's input order
// [t][f][station][pol][re,im]: the corner turn ("a reordering of data necessitated by the
// station independence of the F-engine, and the frequency independence of the X-engine") is the store pattern of this kernel,
// not a pass of its own.  Rows are written `pitch` bytes apart, by default the 128-byte-multiple pitch the X-engine's TMA
// loads like best.
//
// How: the work is bandwidth- and ALU-shaped, not a dense contraction -- CUDA cores, fp32.  One CTA owns SB stations x 2
// polarisations x TT time blocks.  Its 256 threads transform G = 256 / (F / RMAX) signals at a time with a Stockham
// autosort FFT: ceil(log2 F / 4) passes of radix <= 16 (F = 512, 1024: two passes, the first of radix 32), every pass a
// register-resident butterfly per thread, passes
// exchanged through a shared-memory work buffer; the first pass reads the int8 samples straight from global memory, the
// last pass scales, rounds and drops its 2-byte results into a shared-memory tile [signal][tt * F + f] (column-major: a
// thread's outputs sit at compile-time offsets from one base; columns are padded by FE_COL_PAD bytes so that the last pass's stores
// and the row-wise read-out are conflict-free).  When all signals are done the tile is streamed out: every (t, f) row of the CTA is one contiguous run
// of SB x 4 bytes of the cube.
// Twiddles are computed in fp64 on the host (exact at eighth turns), stored per pass in the order the pass reads them
// ([k][r - 1] = exp(-2 pi i k r / (NS R))) and kept in shared memory.  Rounding = round-half-even in fp32, symmetric clip.
// What the ncu captures asked for, in order (profiles/r2_ncu_fengine.md): (1) the work buffer is padded by one complex slot
// per 16 (the Stockham scatter writes with a stride of R slots: 57 % of all shared-memory wavefronts were bank conflicts);
// (2) all complex arithmetic is packed fp32x2 (one instruction per complex add, two per complex multiply); (3) int8 <-> fp32
// conversions avoid the 16-lane conversion unit; (4) every shared-memory address of a pass is one per-thread base plus
// compile-time offsets (45 % of the instructions were integer address arithmetic).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace xc {

#ifndef XC_FE_RADIX32
#define XC_FE_RADIX32 1
#endif
constexpr int FE_THREADS = 256;
constexpr int FE_MAX_LOGF = 12;            // F <= 4096
constexpr int FE_COL_PAD = 36;             // bytes of padding per tile column: 9 words (odd: the row-wise read-out of 16 stations
                                           // hits 16 banks; >= 8: the two signals a warp writes in the last pass use disjoint banks)
constexpr int FE_TILE_BYTES = 32768;       // target size of the CTA's output tile (53 KB per CTA at F = 512: 4 CTAs per SM)

struct FeParams {
    int N, T;
    int SB, TT;               // stations / time blocks per CTA
    int nsb;                  // CTAs along the station axis
    long long pitch;          // bytes between (t, f) rows of the cube
    int f0, nf;               // channels [f0, f0 + nf) are stored, as rows (t * nf + f - f0) of the cube (whole spectrum: 0, F)
    const int8_t* volt;       // [N][2][T*F][2]
    int8_t* cube;             // quantised output (or null)
    float* spec;              // unquantised fp32 spectra [T][F][N][2][2] (or null); testing aid, strided stores
    const float2* tw;         // per-pass twiddle tables (fe_twiddle_layout), F - RMAX entries
    float scale;
};

// How log2 F bits are split over the passes (one table for the kernel templates and for the host's twiddle layout):
// at most 4 bits per pass (radix 16), balanced, the first passes one bit wider -- except that F = 512 and 1024 use a radix-32
// first pass so that they need two passes instead of three (the kernel is bound by the shared-memory traffic of the passes,
// profiles/r2_ncu_fengine.md): measured 0.624 against 0.648 ms (F = 512) and 0.623 against 0.645 ms (F = 1024); F = 32 in one
// radix-32 pass was slower (0.56 vs 0.32 ms), and F = 64 as 16 x 4 instead of 8 x 8 too (0.62 vs 0.59 ms at N = 1024, T = 2048).
__host__ __device__ constexpr int fe_num_passes(int logf) {
    return (logf + ((XC_FE_RADIX32 && (logf == 9 || logf == 10)) ? 5 : 4) - 1) / ((XC_FE_RADIX32 && (logf == 9 || logf == 10)) ? 5 : 4);
}
__host__ __device__ constexpr int fe_pass_bits(int logf, int i) {
    return fe_num_passes(logf) ? logf / fe_num_passes(logf) + (i < logf % fe_num_passes(logf) ? 1 : 0) : 0;
}

template <int LOGF>
struct FeCfg {
    static constexpr int F = 1 << LOGF;
    static constexpr int NP = fe_num_passes(LOGF);                           // passes (0 for F = 1)
    static constexpr int bits(int i) { return fe_pass_bits(LOGF, i); }
    static constexpr int RMAX = 1 << bits(0);                                // points per thread
    static constexpr int TPS = F / RMAX;                                     // threads per signal
    static constexpr int G = FE_THREADS / TPS;                               // signals per sub-batch
    static constexpr int FPAD = F + (F >> 4);                                // one padding slot per 16 complex slots
    static constexpr int WORK_BYTES = (NP > 1) ? G * FPAD * 8 : 0;           // [G][FPAD] float2
    static constexpr int TW_N = (NP > 1) ? F - RMAX : 0;                     // sum over passes i >= 1 of NS_i (R_i - 1)
    static constexpr int TW_BYTES = TW_N * 8;
    static constexpr int ns(int i) { return i == 0 ? 1 : ns(i - 1) << bits(i - 1); }   // product of the radices before pass i
    static constexpr int tw_off(int i) { return i <= 1 ? 0 : tw_off(i - 1) + ns(i - 1) * ((1 << bits(i - 1)) - 1); }
    // Two-pass transforms whose second pass needs at most 16 twiddles per thread keep them in registers for the CTA's whole
    // life (they depend on the thread only, not on the signal): a quarter of the kernel's shared-memory wavefronts were
    // twiddle loads (profiles/r2_ncu_fengine.md).  Measured: F = 64 0.595 -> 0.550 ms, F = 32 0.648 -> 0.605, F = 256
    // 0.533 -> 0.523; F = 128 (14 twiddles, 98 registers) got slower (0.558 -> 0.591) and F = 512 / 1024 would need 60.
    static constexpr int R1 = 1 << bits(1);
    static constexpr int NB1 = RMAX / R1;
    static constexpr bool TW_REGS = (NP == 2) && (NB1 * (R1 - 1) <= 8 || LOGF == 8);
    static constexpr int TWR_B = TW_REGS ? NB1 : 1, TWR_R = TW_REGS ? R1 - 1 : 1;
    static_assert(TPS <= FE_THREADS && TPS >= 1, "threads per signal");
};

// index -> padded index of the work buffer / twiddle table
__device__ __forceinline__ int fe_pad(int i) { return i + (i >> 4); }

// Packed fp32x2 arithmetic (sm_100): one instruction for both halves of a complex number.
__device__ __forceinline__ unsigned long long fe_pack(float2 a) {
    unsigned long long u;
    asm("mov.b64 %0, {%1, %2};" : "=l"(u) : "f"(a.x), "f"(a.y));
    return u;
}
__device__ __forceinline__ float2 fe_unpack(unsigned long long u) {
    float2 d;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(d.x), "=f"(d.y) : "l"(u));
    return d;
}
__device__ __forceinline__ float2 cadd(float2 a, float2 b) {
    unsigned long long d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(fe_pack(a)), "l"(fe_pack(b)));
    return fe_unpack(d);
}
__device__ __forceinline__ float2 csub(float2 a, float2 b) {
    unsigned long long d;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(fe_pack(a)), "l"(fe_pack(b)));
    return fe_unpack(d);
}
__device__ __forceinline__ float2 mul2(float2 a, float2 b) {
    unsigned long long d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(fe_pack(a)), "l"(fe_pack(b)));
    return fe_unpack(d);
}
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c) {
    unsigned long long d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(fe_pack(a)), "l"(fe_pack(b)), "l"(fe_pack(c)));
    return fe_unpack(d);
}
// a * w = (a.x w.x - a.y w.y, a.x w.y + a.y w.x): two packed instructions (the broadcasts and the rotated w are operand
// modifiers of the SASS instruction)
__device__ __forceinline__ float2 cmul(float2 a, float2 w) {
    return fma2(make_float2(a.y, a.y), make_float2(-w.y, w.x), mul2(make_float2(a.x, a.x), w));
}
__device__ __forceinline__ float2 mul_mi(float2 a) { return make_float2(a.y, -a.x); }   // a * (-i)
// a * (1 - i) / sqrt 2 and a * (-1 - i) / sqrt 2
__device__ __forceinline__ float2 mul_w8_1(float2 a) {
    constexpr float h = 0.70710678118654752440f;
    return mul2(cadd(a, mul_mi(a)), make_float2(h, h));            // ((x + y) h, (y - x) h)
}
__device__ __forceinline__ float2 mul_w8_3(float2 a) {
    constexpr float h = 0.70710678118654752440f;
    return mul2(csub(mul_mi(a), a), make_float2(h, h));            // ((y - x) h, -(x + y) h)
}

// R-point forward DFT in registers, natural order in and out: X[k] = sum_r v[r] exp(-2 pi i r k / R).
template <int R> struct Dft;
template <> struct Dft<1> { static __device__ __forceinline__ void run(float2 (&)[1]) {} };
template <> struct Dft<2> {
    static __device__ __forceinline__ void run(float2 (&v)[2]) {
        const float2 a = v[0], b = v[1];
        v[0] = cadd(a, b);
        v[1] = csub(a, b);
    }
};
template <> struct Dft<4> {
    static __device__ __forceinline__ void run(float2 (&v)[4]) {
        const float2 t0 = cadd(v[0], v[2]), t1 = csub(v[0], v[2]);
        const float2 t2 = cadd(v[1], v[3]), t3 = mul_mi(csub(v[1], v[3]));
        v[0] = cadd(t0, t2);
        v[1] = cadd(t1, t3);
        v[2] = csub(t0, t2);
        v[3] = csub(t1, t3);
    }
};
template <> struct Dft<8> {
    static __device__ __forceinline__ void run(float2 (&v)[8]) {
        float2 e[4] = {v[0], v[2], v[4], v[6]}, o[4] = {v[1], v[3], v[5], v[7]};
        Dft<4>::run(e);
        Dft<4>::run(o);
        o[1] = mul_w8_1(o[1]);                                                   // * (1 - i) / sqrt 2
        o[2] = mul_mi(o[2]);                                                     // * (-i)
        o[3] = mul_w8_3(o[3]);                                                   // * (-1 - i) / sqrt 2
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            v[k] = cadd(e[k], o[k]);
            v[k + 4] = csub(e[k], o[k]);
        }
    }
};
template <> struct Dft<16> {
    static __device__ __forceinline__ void run(float2 (&v)[16]) {
        float2 e[8], o[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            e[k] = v[2 * k];
            o[k] = v[2 * k + 1];
        }
        Dft<8>::run(e);
        Dft<8>::run(o);
        constexpr float c1 = 0.92387953251128675613f, s1 = 0.38268343236508977173f;
        // o[k] *= exp(-2 pi i k / 16) = cos(k pi / 8) - i sin(k pi / 8)
        o[1] = cmul(o[1], make_float2(c1, -s1));
        o[2] = mul_w8_1(o[2]);
        o[3] = cmul(o[3], make_float2(s1, -c1));
        o[4] = mul_mi(o[4]);
        o[5] = cmul(o[5], make_float2(-s1, -c1));
        o[6] = mul_w8_3(o[6]);
        o[7] = cmul(o[7], make_float2(-c1, -s1));
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            v[k] = cadd(e[k], o[k]);
            v[k + 8] = csub(e[k], o[k]);
        }
    }
};

template <> struct Dft<32> {
    static __device__ __forceinline__ void run(float2 (&v)[32]) {
        float2 e[16], o[16];
#pragma unroll
        for (int k = 0; k < 16; ++k) {
            e[k] = v[2 * k];
            o[k] = v[2 * k + 1];
        }
        Dft<16>::run(e);
        Dft<16>::run(o);
        // o[k] *= exp(-2 pi i k / 32)
        o[1] = cmul(o[1], make_float2(0.98078528040323043058f, -0.19509032201612824808f));
        o[2] = cmul(o[2], make_float2(0.92387953251128673848f, -0.38268343236508978178f));
        o[3] = cmul(o[3], make_float2(0.83146961230254523567f, -0.55557023301960217765f));
        o[4] = mul_w8_1(o[4]);
        o[5] = cmul(o[5], make_float2(0.55557023301960228867f, -0.83146961230254523567f));
        o[6] = cmul(o[6], make_float2(0.38268343236508983729f, -0.92387953251128673848f));
        o[7] = cmul(o[7], make_float2(0.19509032201612833135f, -0.98078528040323043058f));
        o[8] = mul_mi(o[8]);
        o[9] = cmul(o[9], make_float2(-0.19509032201612819257f, -0.98078528040323043058f));
        o[10] = cmul(o[10], make_float2(-0.38268343236508972627f, -0.92387953251128673848f));
        o[11] = cmul(o[11], make_float2(-0.55557023301960195560f, -0.83146961230254545772f));
        o[12] = mul_w8_3(o[12]);
        o[13] = cmul(o[13], make_float2(-0.83146961230254534669f, -0.55557023301960217765f));
        o[14] = cmul(o[14], make_float2(-0.92387953251128673848f, -0.38268343236508989280f));
        o[15] = cmul(o[15], make_float2(-0.98078528040323043058f, -0.19509032201612860891f));
#pragma unroll
        for (int k = 0; k < 16; ++k) {
            v[k] = cadd(e[k], o[k]);
            v[k + 16] = csub(e[k], o[k]);
        }
    }
};

// int8 -> fp32 without the conversion unit (I2F / F2I run on the 16-lane XU pipe: 4 conversions per sample were 21 % of the
// kernel's issue slots): the byte, biased by 128, becomes the low mantissa byte of 2^23, and 2^23 + 128 is subtracted.
__device__ __forceinline__ float2 fe_char2_to_float2(uint32_t raw16) {
    const uint32_t w = raw16 ^ 0x8080u;
    const float re = __uint_as_float(__byte_perm(w, 0x4B000000u, 0x7650));
    const float im = __uint_as_float(__byte_perm(w, 0x4B000000u, 0x7651));
    return csub(make_float2(re, im), make_float2(8388736.0f, 8388736.0f));
}
// q = clip(rint(y), -127, 127) for both components, round-half-even (reading 20): clamp (the bounds are integers,
// so clamping first changes nothing), add 1.5 * 2^23 -- the fp32 addition rounds to the nearest integer, ties to even --
// and take the low byte of each sum.  Returns re | im << 8.
__device__ __forceinline__ uint32_t fe_quant2(float2 y) {
    const float cx = fminf(fmaxf(y.x, -127.0f), 127.0f), cy = fminf(fmaxf(y.y, -127.0f), 127.0f);
    const float2 t = cadd(make_float2(cx, cy), make_float2(12582912.0f, 12582912.0f));
    return __byte_perm(__float_as_uint(t.x), __float_as_uint(t.y), 0x7740) & 0xFFFFu;
}

// One pass of the Stockham FFT for this thread's butterflies.  v[b][r]: butterfly b (j = tid_in_signal + b * TPS), leg r.
template <int LOGF, int PASS>
struct FePass {
    using C = FeCfg<LOGF>;
    static constexpr int R = 1 << C::bits(PASS);
    static constexpr int NB = C::RMAX / R;                // butterflies per thread
    static constexpr int NS = C::ns(PASS);                // length of the sub-transforms done so far
    static constexpr int STRIDE = C::F / R;               // distance of a butterfly's legs in the input of the pass
    static constexpr int TW_OFF = C::tw_off(PASS);        // where this pass's twiddle table starts

    static __host__ __device__ constexpr int padc(int c) { return c + (c >> 4); }     // fe_pad of a compile-time offset
    // fe_pad(x + c) = fe_pad(x) + padc(c) whenever x % 16 + c % 16 < 16, which holds for every (x, c) used below: c is a
    // multiple of 16, or x < the power-of-two stride that c is a multiple of (all sizes here are powers of two).
    static __device__ __forceinline__ void load_raw(uint32_t (&raw)[NB][R], const int8_t* __restrict__ x, int ts, bool ok) {
#pragma unroll
        for (int b = 0; b < NB; ++b)
#pragma unroll
            for (int r = 0; r < R; ++r)
                raw[b][r] = ok ? static_cast<uint32_t>(__ldg(reinterpret_cast<const uint16_t*>(x) + (ts + b * C::TPS + r * STRIDE))) : 0u;
    }
    static __device__ __forceinline__ void convert(float2 (&v)[NB][R], const uint32_t (&raw)[NB][R]) {
#pragma unroll
        for (int b = 0; b < NB; ++b)
#pragma unroll
            for (int r = 0; r < R; ++r) v[b][r] = fe_char2_to_float2(raw[b][r]);
    }
    static __device__ __forceinline__ void load_smem(float2 (&v)[NB][R], const float2* buf, int ts) {
#pragma unroll
        for (int b = 0; b < NB; ++b) {
            const float2* pb = buf + fe_pad(ts + b * C::TPS);
#pragma unroll
            for (int r = 0; r < R; ++r) v[b][r] = pb[padc(r * STRIDE)];
        }
    }
    // twr: this thread's twiddles of pass 1 in registers (FeCfg::TW_REGS), else unused
    static __device__ __forceinline__ void compute(float2 (&v)[NB][R], const float2* tw, int ts,
                                                   const float2 (&twr)[C::TWR_B][C::TWR_R]) {
#pragma unroll
        for (int b = 0; b < NB; ++b) {
            if constexpr (C::TW_REGS && PASS == 1) {
#pragma unroll
                for (int r = 1; r < R; ++r) v[b][r] = cmul(v[b][r], twr[b][r - 1]);
            } else if (NS > 1) {
                const float2* tk = tw + TW_OFF + ((ts + b * C::TPS) & (NS - 1)) * (R - 1);  // row k of this pass's table
#pragma unroll
                for (int r = 1; r < R; ++r) v[b][r] = cmul(v[b][r], tk[r - 1]);
            }
            Dft<R>::run(v[b]);
        }
    }
    // position of leg r of butterfly j in the output of the pass
    static __device__ __forceinline__ int out_index(int j, int r) { return (j / NS) * (NS * R) + (j & (NS - 1)) + r * NS; }
    static __device__ __forceinline__ void store_smem(const float2 (&v)[NB][R], float2* buf, int ts) {
#pragma unroll
        for (int b = 0; b < NB; ++b) {
            float2* pb = buf + fe_pad(out_index(ts + b * C::TPS, 0));
#pragma unroll
            for (int r = 0; r < R; ++r) pb[padc(r * NS)] = v[b][r];
        }
    }
};

template <int LOGF, int PASS>
struct FeRun {
    using C = FeCfg<LOGF>;
    using P = FePass<LOGF, PASS>;
    // Runs passes PASS .. NP-1 for this thread; `sink(f, value)` takes the final spectrum samples.
    // `raw`: pass 0's samples, fetched one sub-batch ahead by the caller (unused by the later passes)
    template <typename Raw, typename Sink>
    static __device__ __forceinline__ void run(const Raw& raw, float2* buf, const float2* tw, int ts,
                                               const float2 (&twr)[C::TWR_B][C::TWR_R], Sink&& sink) {
        float2 v[P::NB][P::R];
        if constexpr (PASS == 0) P::convert(v, raw);
        else P::load_smem(v, buf, ts);
        P::compute(v, tw, ts, twr);
        if constexpr (PASS >= C::NP - 1) {        // (>=: F = 1 has no pass at all and is its own spectrum)
#pragma unroll
            for (int b = 0; b < P::NB; ++b)
#pragma unroll
                for (int r = 0; r < P::R; ++r) sink(P::out_index(ts + b * C::TPS, r), v[b][r]);
            if (C::NP > 1) __syncthreads();        // the work buffer may be refilled by the next sub-batch
        } else {
            if (PASS > 0) __syncthreads();         // everybody has read the buffer
            P::store_smem(v, buf, ts);
            __syncthreads();
            FeRun<LOGF, PASS + 1>::run(raw, buf, tw, ts, twr, sink);
        }
    }
};

// SPEC = false: the product kernel (quantised cube).  SPEC = true: the fp32 spectra for the transform's own parity test.
template <int LOGF, bool SPEC>
__global__ void __launch_bounds__(FE_THREADS) xc_fengine_kernel(const FeParams p) {
    using C = FeCfg<LOGF>;
    constexpr int F = C::F;
    extern __shared__ __align__(16) uint8_t fe_smem[];
    // output tile, column-major: column sp (signal) holds the TT * F samples of the CTA's time blocks, 2 bytes each, columns
    // CS bytes apart (+4: the read-out below walks along sp)
    const int lsb = 32 - __clz(p.SB);                               // log2(2 SB): SB is 8, 16 or 32
    const uint32_t CS = static_cast<uint32_t>(p.TT) * F * 2u + FE_COL_PAD;
    const uint32_t tile_bytes = SPEC ? 0u : (2u * p.SB * CS + 15u) & ~15u;
    uint8_t* tile = fe_smem;
    float2* work = reinterpret_cast<float2*>(fe_smem + tile_bytes);                    // [G][FPAD]
    float2* tw = reinterpret_cast<float2*>(reinterpret_cast<uint8_t*>(work) + C::WORK_BYTES);

    const int tid = threadIdx.x;
    const int s0 = static_cast<int>(blockIdx.x % p.nsb) * p.SB;       // station groups fastest: neighbouring CTAs complete
    const int t0 = static_cast<int>(blockIdx.x / p.nsb) * p.TT;       // each other's 128-byte lines in L2
    if (C::NP > 1) {
        for (int m = tid; m < C::TW_N; m += FE_THREADS) tw[m] = __ldg(p.tw + m);
        __syncthreads();
    }
    const int g = tid / C::TPS;             // signal of the sub-batch this thread works on
    const int ts = tid % C::TPS;            // its index among the signal's threads
    float2* buf = work + g * C::FPAD;
    const int nq = 2 * p.SB * p.TT;         // (signal, time block) pairs of this CTA; sp fastest
    const long long TF = static_cast<long long>(p.T) * F;

    // (signal, time block) q of the CTA -> where its F samples start and whether it exists
    auto locate = [&](int q, int& sp, int& tt, int& s, int& pol, int& t) {
        sp = q & (2 * p.SB - 1);
        tt = q >> lsb;
        s = s0 + (sp >> 1);
        pol = sp & 1;
        t = t0 + tt;
        return (q < nq) && (s < p.N) && (t < p.T);
    };
    float2 twr[C::TWR_B][C::TWR_R];
    if constexpr (C::TW_REGS) {
        using P1 = FePass<LOGF, 1>;
#pragma unroll
        for (int b = 0; b < C::NB1; ++b)
#pragma unroll
            for (int r = 1; r < C::R1; ++r) twr[b][r - 1] = tw[P1::TW_OFF + ((ts + b * C::TPS) & (P1::NS - 1)) * (C::R1 - 1) + r - 1];
    } else {
        twr[0][0] = make_float2(0.f, 0.f);
    }
    using P0 = FePass<LOGF, 0>;
    uint32_t raw[P0::NB][P0::R];            // pass 0's samples of the NEXT sub-batch: their latency hides behind this one
    {
        int sp, tt, s, pol, t;
        const bool ok = locate(g, sp, tt, s, pol, t);
        P0::load_raw(raw, p.volt + ((static_cast<long long>(s) * 2 + pol) * TF + static_cast<long long>(t) * F) * 2, ts, ok);
    }
    for (int q0 = 0; q0 < nq; q0 += C::G) {
        int sp, tt, s, pol, t;
        const bool ok = locate(q0 + g, sp, tt, s, pol, t);
        uint32_t cur[P0::NB][P0::R];
#pragma unroll
        for (int b = 0; b < P0::NB; ++b)
#pragma unroll
            for (int r = 0; r < P0::R; ++r) cur[b][r] = raw[b][r];
        if (q0 + C::G < nq) {
            int sp2, tt2, s2, pol2, t2;
            const bool ok2 = locate(q0 + C::G + g, sp2, tt2, s2, pol2, t2);
            P0::load_raw(raw, p.volt + ((static_cast<long long>(s2) * 2 + pol2) * TF + static_cast<long long>(t2) * F) * 2, ts, ok2);
        }
        if constexpr (SPEC) {
            float2* dst = reinterpret_cast<float2*>(p.spec) + (static_cast<long long>(t) * F * p.N + s) * 2 + pol;
            const long long fstride = static_cast<long long>(p.N) * 2;
            auto sink = [&](int f, float2 X) {
                if (ok) dst[f * fstride] = X;
            };
            FeRun<LOGF, 0>::run(cur, buf, tw, ts, twr, sink);
        } else {
            // column sp, row tt * F: the thread's outputs f = j + r * NS land at compile-time offsets from here
            uint16_t* col = reinterpret_cast<uint16_t*>(tile + static_cast<uint32_t>(sp) * CS) + tt * F;
            const float2 sc2 = make_float2(p.scale, p.scale);
            const bool inq = (q0 + g) < nq;       // columns of stations >= N / blocks >= T exist in the tile and are masked at read-out
            auto sink = [&](int f, float2 X) {
                if (inq) col[f] = static_cast<uint16_t>(fe_quant2(mul2(X, sc2)));      // one rounding per component, like __fmul_rn
            };
            FeRun<LOGF, 0>::run(cur, buf, tw, ts, twr, sink);
        }
    }
    if constexpr (SPEC) return;
    __syncthreads();
    // Stream the tile out: one warp instruction writes 128 contiguous... bytes per cube row segment -- lane = (row, station)
    // with 128 / RB rows per instruction; a lane gathers its station's two polarisations (two 2-byte columns) into one word.
    const uint32_t lrb = static_cast<uint32_t>(lsb) + 1u;         // log2 of RB = 4 SB bytes per row segment
    const uint32_t lm = 7u - lrb, lw = lrb - 2u;                  // log2 of rows per instruction, of words (stations) per row
    const uint32_t nrows = static_cast<uint32_t>(p.TT) * F;
    const uint32_t lane = tid & 31, warp = tid >> 5;
    const uint32_t cw = lane & ((1u << lw) - 1u);                 // station s0 + cw
    const uint16_t* c0 = reinterpret_cast<const uint16_t*>(tile + (2u * cw) * CS);
    const uint16_t* c1 = reinterpret_cast<const uint16_t*>(tile + (2u * cw + 1u) * CS);
    const int s = s0 + static_cast<int>(cw);
    for (uint32_t rho = (warp << lm) + (lane >> lw); rho < nrows; rho += (FE_THREADS / 32) << lm) {
        const uint32_t tt = rho >> LOGF, f = rho & (F - 1);
        const int t = t0 + static_cast<int>(tt);
        const uint32_t fr = f - static_cast<uint32_t>(p.f0);      // row inside the stored channel range (unsigned: f < f0 wraps)
        if (t < p.T && s < p.N && fr < static_cast<uint32_t>(p.nf)) {
            const uint32_t w = static_cast<uint32_t>(c0[rho]) | (static_cast<uint32_t>(c1[rho]) << 16);
            int8_t* row = p.cube + (static_cast<long long>(t) * p.nf + fr) * p.pitch;
            __stcs(reinterpret_cast<uint32_t*>(row) + s, w);
        }
    }
}

}  // namespace xc
