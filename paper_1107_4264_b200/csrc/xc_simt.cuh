// xc_simt.cuh -- (a) a plain CUDA-core int8 X-engine, one thread per station pair, kept as a
// debugging aid for the tensor-core kernel (XC_I8_KERNEL_SIMT; never chosen by AUTO), and
// (b) the staging kernel of SURVEY 8(a) S0 that pads the station axis for TMA.
//
// (a) is the paper's simplest mapping, R = (1,1): each thread owns one
// station pair and its four polarisation products, reads both stations' samples straight from
// global memory (hardware-managed cache), and the thread-block grid covers the lower triangle
// through the closed-form map of PAPER.md:157-163.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace xc {

constexpr int SIMT_B = 16;  // stations per block edge

struct SimtParams {
    int N, F, T;
    long long NB;
    long long pitch;      // bytes between consecutive (t, f) rows of `in`
    const int8_t* in;
    int32_t* vis;
    int accumulate;
};

// by = floor(-1/2 + sqrt(1/4 + 2g)), bx = g - by(by+1)/2, with an integer
// fix-up because the floating square root is exact only for small g (SURVEY 8(c) reading 12).
__host__ __device__ inline void tri_inverse(long long g, long long* bx, long long* by) {
    long long y = static_cast<long long>(-0.5 + sqrt(0.25 + 2.0 * static_cast<double>(g)));
    if (y < 0) y = 0;
    while (y * (y + 1) / 2 > g) --y;
    while ((y + 1) * (y + 2) / 2 <= g) ++y;
    *by = y;
    *bx = g - y * (y + 1) / 2;
}

__global__ void __launch_bounds__(SIMT_B* SIMT_B) xc_i8_simt_kernel(const SimtParams p) {
    long long bx, by;
    tri_inverse(blockIdx.x, &bx, &by);  // bx <= by: block column (i side), block row (j side)
    const int f = blockIdx.y;
    const int i = static_cast<int>(bx) * SIMT_B + threadIdx.x;
    const int j = static_cast<int>(by) * SIMT_B + threadIdx.y;
    if (i > j || j >= p.N) return;  // super-diagonal threads exit
    int acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    for (int t = 0; t < p.T; ++t) {
        const int8_t* x = p.in + (static_cast<long long>(t) * p.F + f) * p.pitch;
        int a[4], b[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            a[k] = x[i * 4 + k];
            b[k] = x[j * 4 + k];
        }
#pragma unroll
        for (int pi = 0; pi < 2; ++pi)
#pragma unroll
            for (int pj = 0; pj < 2; ++pj) {
                acc[(pi * 2 + pj) * 2 + 0] += a[2 * pi] * b[2 * pj] + a[2 * pi + 1] * b[2 * pj + 1];
                acc[(pi * 2 + pj) * 2 + 1] += a[2 * pi + 1] * b[2 * pj] - a[2 * pi] * b[2 * pj + 1];
            }
    }
    int32_t* dst = p.vis + (static_cast<long long>(f) * p.NB + static_cast<long long>(j) * (j + 1) / 2 + i) * 8;
#pragma unroll
    for (int k = 0; k < 8; ++k) dst[k] = p.accumulate ? dst[k] + acc[k] : acc[k];
}

// (b) Staging: rows of 4N bytes, `pitch` bytes apart -> rows of 4*Npad bytes (the plan's 128-byte-multiple pitch), zero
// padded, written to a 128-byte-aligned workspace.  One thread per destination station (4 bytes).  Needed only when the
// input cannot be read by TMA in place: a base or row pitch that is not a multiple of 16 bytes (N % 4 != 0).
__global__ void xc_stage_pad_kernel(const int8_t* __restrict__ in, uint32_t* __restrict__ out, long long rows, int N,
                                    long long pitch, int Npad) {
    const long long total = rows * Npad;
    for (long long k = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x; k < total;
         k += static_cast<long long>(gridDim.x) * blockDim.x) {
        const long long r = k / Npad;
        const int s = static_cast<int>(k - r * Npad);
        uint32_t v = 0;
        if (s < N) {
            const uint8_t* src = reinterpret_cast<const uint8_t*>(in) + r * pitch + s * 4;
            v = static_cast<uint32_t>(src[0]) | (static_cast<uint32_t>(src[1]) << 8) |
                (static_cast<uint32_t>(src[2]) << 16) | (static_cast<uint32_t>(src[3]) << 24);
        }
        out[k] = v;
    }
}

// The same for channels [f0, f0 + nf) of every time sample only (rows r = t * F + f keep their place in the workspace), so
// that a block which needs staging can still be correlated range by range (xc_correlate_channels: one range per stream
// or per GPU); disjoint ranges write disjoint workspace rows.
__global__ void xc_stage_pad_range_kernel(const int8_t* __restrict__ in, uint32_t* __restrict__ out, int T, int F, int f0, int nf,
                                          int N, long long pitch, int Npad) {
    const long long per_t = static_cast<long long>(nf) * Npad;
    const long long total = per_t * T;
    for (long long k = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x; k < total;
         k += static_cast<long long>(gridDim.x) * blockDim.x) {
        const long long t = k / per_t;
        const long long rem = k - t * per_t;
        const long long r = t * F + f0 + rem / Npad;
        const int s = static_cast<int>(rem % Npad);
        uint32_t v = 0;
        if (s < N) {
            const uint8_t* src = reinterpret_cast<const uint8_t*>(in) + r * pitch + s * 4;
            v = static_cast<uint32_t>(src[0]) | (static_cast<uint32_t>(src[1]) << 8) |
                (static_cast<uint32_t>(src[2]) << 16) | (static_cast<uint32_t>(src[3]) << 24);
        }
        out[r * Npad + s] = v;
    }
}

// Same, 16 bytes (4 stations) per thread, for N % 4 == 0, a 16-byte aligned input and a 16-byte-multiple pitch: only
// reached with XC_OPT_FORCE_STAGE (a re-pitching copy into the workspace, for testing S0 on aligned shapes).
__global__ void xc_stage_pad16_kernel(const uint4* __restrict__ in, uint4* __restrict__ out, long long rows, int n4,
                                      int pitch16, int npad4) {
    const long long total = rows * npad4;
    for (long long k = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x; k < total;
         k += static_cast<long long>(gridDim.x) * blockDim.x) {
        const long long r = k / npad4;
        const int c = static_cast<int>(k - r * npad4);
        out[k] = (c < n4) ? __ldcs(in + r * pitch16 + c) : make_uint4(0u, 0u, 0u, 0u);
    }
}

// (b') Re-pitching for the host-buffer calls: the H2D copy lands dense rows (4N bytes: the copy engine moves dense blocks at
// full PCIe rate, a pitched 2-D copy of 2000-byte rows measured 4x slower), and this pass spreads channels [f0, f0 + nf) of
// every time sample to the plan's 128-byte-multiple pitch.  W bytes per thread: 16 when 4N is a multiple of 16, else 4.
template <typename W>
__global__ void xc_repitch_kernel(const W* __restrict__ in, W* __restrict__ out, int T, int F, int f0, int nf, int n_w,
                                  long long out_pitch_w) {
    const long long per_t = static_cast<long long>(nf) * n_w;
    const long long total = per_t * T;
    for (long long k = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x; k < total;
         k += static_cast<long long>(gridDim.x) * blockDim.x) {
        const long long t = k / per_t;
        const long long rem = k - t * per_t;
        const long long row = t * F + f0 + rem / n_w;
        const long long c = rem % n_w;
        out[row * out_pitch_w + c] = in[row * n_w + c];
    }
}

// (d) 4-bit complex samples (reading 17): one byte per (t, f, station, pol), low nibble = real,
// high nibble = imaginary, two's complement.  Unpacked into the int8 workspace the tensor-core kernel reads (station pitch
// Npad).  Four packed bytes (two stations) -> eight int8: per byte lane (n ^ 8) - 8 sign-extends the nibble.
__device__ __forceinline__ void unpack_i4_word(uint32_t w, uint32_t* o0, uint32_t* o1) {
    const uint32_t lo = __vsub4((w & 0x0F0F0F0Fu) ^ 0x08080808u, 0x08080808u);          // real parts, one per byte lane
    const uint32_t hi = __vsub4(((w >> 4) & 0x0F0F0F0Fu) ^ 0x08080808u, 0x08080808u);   // imaginary parts
    *o0 = __byte_perm(lo, hi, 0x5140);   // (re0, im0, re1, im1): station s,   pol 0 and 1
    *o1 = __byte_perm(lo, hi, 0x7362);   // (re2, im2, re3, im3): station s+1, pol 0 and 1
}
// Both kernels work on the channel range [f0, f0 + nf) of every time sample (row r = t * F + f), so that ranges of one
// block can be unpacked and correlated one after the other (xc_correlate_host_i4).
// general: one thread per destination station (2 packed bytes -> 4 int8), zero padding for s >= N
__global__ void xc_unpack_i4_kernel(const uint8_t* __restrict__ in4, uint32_t* __restrict__ out, int T, int F, int f0, int nf,
                                    int N, int Npad) {
    const long long per_t = static_cast<long long>(nf) * Npad;
    const long long total = per_t * T;
    for (long long k = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x; k < total;
         k += static_cast<long long>(gridDim.x) * blockDim.x) {
        const long long t = k / per_t;
        const long long rem = k - t * per_t;
        const long long r = t * F + f0 + rem / Npad;
        const int s = static_cast<int>(rem % Npad);
        uint32_t o0 = 0, o1 = 0;
        if (s < N) {
            const uint8_t* src = in4 + (r * N + s) * 2;
            unpack_i4_word(static_cast<uint32_t>(src[0]) | (static_cast<uint32_t>(src[1]) << 8), &o0, &o1);
        }
        out[r * Npad + s] = o0;
    }
}
// N % 8 == 0 and a 16-byte aligned input: 16 packed bytes (8 stations) -> 32 int8 per thread; n8 = N / 8, npad8 = Npad / 8
__global__ void xc_unpack_i4x8_kernel(const uint4* __restrict__ in4, uint4* __restrict__ out, int T, int F, int f0, int nf,
                                      int n8, int npad8) {
    const long long per_t = static_cast<long long>(nf) * n8;
    const long long total = per_t * T;
    for (long long k = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x; k < total;
         k += static_cast<long long>(gridDim.x) * blockDim.x) {
        const long long t = k / per_t;
        const long long rem = k - t * per_t;
        const long long row = t * F + f0 + rem / n8;
        const long long c = rem % n8;
        const uint4 w = __ldcs(in4 + row * n8 + c);
        uint4 a, b;
        unpack_i4_word(w.x, &a.x, &a.y);
        unpack_i4_word(w.y, &a.z, &a.w);
        unpack_i4_word(w.z, &b.x, &b.y);
        unpack_i4_word(w.w, &b.z, &b.w);
        out[2 * (row * npad8 + c)] = a;       // workspace rows are npad8 * 32 bytes apart (bytes beyond 4N are never read)
        out[2 * (row * npad8 + c) + 1] = b;
    }
}

// (c) Long integrations (I = N_p * I'): vis64 (+)= vis32, four values per thread.  int32 partial
// sums of at most XC_MAX_T samples are exact; this widening add makes any integration length exact in int64.
__global__ void xc_widen_kernel(const int4* __restrict__ v32, longlong2* __restrict__ v64, long long n4, int first) {
    for (long long k = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x; k < n4;
         k += static_cast<long long>(gridDim.x) * blockDim.x) {
        const int4 a = __ldcs(v32 + k);
        longlong2 lo = make_longlong2(a.x, a.y), hi = make_longlong2(a.z, a.w);
        if (!first) {
            const longlong2 o0 = v64[2 * k], o1 = v64[2 * k + 1];
            lo.x += o0.x; lo.y += o0.y; hi.x += o1.x; hi.y += o1.y;
        }
        v64[2 * k] = lo;
        v64[2 * k + 1] = hi;
    }
}

}  // namespace xc
