// xc_noalloc.cu -- xc_correlate_i4_noalloc (include/xc.h): the 4-bit X-engine call for callers that may not allocate
// device memory.
//
// Who that is.  A correlator back-end usually sits inside somebody else's process: a telescope's real-time capture loop
// that has to hand a block to the GPU every few milliseconds and cannot afford cudaMalloc (it serialises against all
// work in flight on the device and takes an unbounded time); a plug-in of a host application that owns all device
// memory itself and forbids its plug-ins to allocate; a process in which a framework's caching allocator or a memory
// pool has already claimed what HBM was left, so that a cudaMalloc issued by this library simply fails.  The ordinary
// 4-bit call, xc_correlate_i4, needs two things from the allocator: the int8 workspace its unpacking pass writes (the
// tensor-core kernel reads int8 through TMA) and the plan's small device tables.  This entry point needs neither: the
// workspace is the file-scope array below, part of the library's device image and therefore created by the driver when
// the image is loaded; the tile table travels in the kernel parameters; there is no plan.
//
// What it costs.  Every CUDA context that loads this translation unit's device image holds XC_NOALLOC_SCRATCH_BYTES
// (16 MiB) of device memory until the process exits, used or not.  One array per device serves every call on that device:
// see "sharing" in xc.h.
//
// The kernels are this file's own (an unpacking kernel, and thin __global__ wrappers around the tile body of
// xc_i8_tc.cuh), so nothing here touches a kernel, a table or a code path of xc_api.cu.
#include "../../include/xc.h"

#include <cuda.h>
#include <cuda_runtime.h>

#include <cstring>
#include <mutex>

#include "xc_i8_tc.cuh"

namespace {

// The scratch.  In HOST code this name is only a handle for the runtime's symbol calls -- it is not a device address, and
// a kernel handed `xc_noalloc_scratch` from the host side would fault (or, on a machine whose GPU can reach host memory,
// quietly use some host bytes).  Host code below therefore asks the runtime for the array's device address once per
// device (cudaGetSymbolAddress) and passes that pointer on.  256-byte alignment covers TMA's 16-byte rule and keeps the
// workspace rows (multiples of 128 bytes) on L2 line boundaries.
static __device__ __align__(256) unsigned char xc_noalloc_scratch[XC_NOALLOC_SCRATCH_BYTES];

// One packed 16-bit group (a station's two polarisations; per byte: low nibble = real, high nibble = imaginary, two's
// complement) -> four int8 (re0, im0, re1, im1).  (n ^ 8) - 8 sign-extends a nibble, per byte lane.
__device__ __forceinline__ uint32_t na_unpack_station(uint32_t w) {
    const uint32_t lo = __vsub4((w & 0x0F0F0F0Fu) ^ 0x08080808u, 0x08080808u);
    const uint32_t hi = __vsub4(((w >> 4) & 0x0F0F0F0Fu) ^ 0x08080808u, 0x08080808u);
    return __byte_perm(lo, hi, 0x5140);
}

// Unpacking pass: in4 [T*F rows][N][2 pol] packed bytes -> ws [T*F rows][Npad stations] of 4 int8, one thread per
// destination station.  Stations N..Npad of every row are written as zero (not that anybody reads them: the tensor map over
// the scratch ends at 4N bytes per row).  Every byte the X-engine reads was written by this call's own unpacking pass, so
// nothing of an earlier call (another N, another F) can show through; rows beyond T*F are not touched and not read.
__global__ void xc_noalloc_unpack_i4_kernel(const uint8_t* __restrict__ in4, uint32_t* __restrict__ ws, long long rows, int N,
                                            int Npad) {
    const long long total = rows * Npad;
    for (long long k = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x; k < total;
         k += static_cast<long long>(gridDim.x) * blockDim.x) {
        const long long r = k / Npad;
        const int s = static_cast<int>(k - r * Npad);
        uint32_t v = 0;
        if (s < N) {
            const uint8_t* src = in4 + (r * N + s) * 2;
            v = na_unpack_station(static_cast<uint32_t>(src[0]) | (static_cast<uint32_t>(src[1]) << 8));
        }
        ws[k] = v;
    }
}

// The same for N % 8 == 0 and a 16-byte aligned input: 16 packed bytes (8 stations) -> 32 int8 per thread (n8 = N / 8 groups
// per row, workspace rows npad8 * 32 bytes apart).  Bytes of a workspace row beyond 4N are not written here -- and never
// read: the tensor map over the scratch ends at 4N bytes per row, what lies beyond is hardware zero fill.
__global__ void xc_noalloc_unpack_i4x8_kernel(const uint4* __restrict__ in4, uint4* __restrict__ ws, long long rows, int n8,
                                              int npad8) {
    const long long total = rows * n8;
    for (long long k = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x; k < total;
         k += static_cast<long long>(gridDim.x) * blockDim.x) {
        const long long r = k / n8;
        const long long c = k - r * n8;
        const uint4 w = __ldcs(in4 + k);
        uint4 a, b;
        a.x = na_unpack_station(w.x & 0xFFFFu); a.y = na_unpack_station(w.x >> 16);
        a.z = na_unpack_station(w.y & 0xFFFFu); a.w = na_unpack_station(w.y >> 16);
        b.x = na_unpack_station(w.z & 0xFFFFu); b.y = na_unpack_station(w.z >> 16);
        b.z = na_unpack_station(w.w & 0xFFFFu); b.w = na_unpack_station(w.w >> 16);
        ws[2 * (r * npad8 + c)] = a;
        ws[2 * (r * npad8 + c) + 1] = b;
    }
}

// The X-engine proper: the persistent tcgen05 tile body of xc_i8_tc.cuh under kernel names of this file's own (CG = 2:
// CTA pairs on 256 x 256 tiles; CG = 1: single CTAs on 128 x 128 tiles; no T-split).
template <int UMMA_N, int CG, int BK>
__global__ void __launch_bounds__(xc::TC_THREADS, 1)
xc_noalloc_i8_tc_kernel(const __grid_constant__ CUtensorMap tmap, const __grid_constant__ xc::TcParams p) {
    xc::tc_body<UMMA_N, CG, BK, 1>(tmap, p, static_cast<int>(blockIdx.x) / CG, static_cast<int>(gridDim.x) / CG);
}

typedef CUresult (*PFN_encodeTiled)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                    const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                    CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// Per-device set-up, done by the first call on that device (with it current) and kept for the life of the process.
struct NaDevice {
    bool ready = false;
    void* scratch = nullptr;        // DEVICE address of xc_noalloc_scratch on this device
    int sm_count = 0;
    PFN_encodeTiled encode = nullptr;
};
constexpr int kMaxDevices = 64;
NaDevice g_dev[kMaxDevices];
std::mutex g_dev_mutex;

template <int UMMA_N, int CG, int BK>
cudaError_t na_opt_in() {
    return cudaFuncSetAttribute(xc_noalloc_i8_tc_kernel<UMMA_N, CG, BK>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                xc::TcCfg<UMMA_N, CG, BK, 1>::SMEM_BYTES);
}

int na_setup(int dev, NaDevice** out) {
    if (dev < 0 || dev >= kMaxDevices) return XC_ERR_UNSUPPORTED;
    std::lock_guard<std::mutex> lock(g_dev_mutex);
    NaDevice& d = g_dev[dev];
    *out = &d;
    if (d.ready) return XC_OK;
    int major = 0, sms = 0;
    if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        (void)cudaGetLastError();
        return XC_ERR_CUDA;
    }
    if (major != 10) return XC_ERR_UNSUPPORTED;      // tcgen05 / TMEM required; there is no other path
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn ||
        qres != cudaDriverEntryPointSuccess) {
        (void)cudaGetLastError();
        return XC_ERR_CUDA;
    }
    if (na_opt_in<256, 2, 128>() != cudaSuccess || na_opt_in<128, 1, 256>() != cudaSuccess) {
        (void)cudaGetLastError();
        return XC_ERR_CUDA;
    }
    // The one step that turns the host-side symbol into something a kernel (and a tensor map) can use: its address on
    // THIS device.  Asked with this device current; the answer differs from device to device.
    void* ptr = nullptr;
    if (cudaGetSymbolAddress(&ptr, xc_noalloc_scratch) != cudaSuccess || !ptr) {
        (void)cudaGetLastError();
        return XC_ERR_CUDA;
    }
    d.scratch = ptr;
    d.sm_count = sms;
    d.encode = reinterpret_cast<PFN_encodeTiled>(fn);
    d.ready = true;
    return XC_OK;
}

// Tiles of S x S stations that hold at least one pair i <= j < N, block row bj outermost, bi = 0 .. bj inside it (the
// paper's triangular order).  Returns the count; fills out[] (bi | bj << 16) when it fits.
int na_tiles(int N, int S, uint32_t* out, int cap) {
    const int nb = (N + S - 1) / S;
    int n = 0;
    for (int bj = 0; bj < nb; ++bj)
        for (int bi = 0; bi <= bj; ++bi, ++n)
            if (n < cap) out[n] = static_cast<uint32_t>(bi) | (static_cast<uint32_t>(bj) << 16);
    return n;
}

template <int UMMA_N, int CG, int BK>
cudaError_t na_launch(const CUtensorMap& tmap, const xc::TcParams& tp, int sm_count, cudaStream_t st) {
    long long units = sm_count / CG;
    if (units < 1) units = 1;
    if (units > tp.total_tiles) units = tp.total_tiles;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(static_cast<unsigned>(units * CG));
    cfg.blockDim = dim3(xc::TC_THREADS);
    cfg.dynamicSmemBytes = xc::TcCfg<UMMA_N, CG, BK, 1>::SMEM_BYTES;
    cfg.stream = st;
    cudaLaunchAttribute attr[2];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = CG;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    // as in the ordinary path: the tile kernel's prologue may overlap the unpacking pass; it executes griddepcontrol.wait
    // before its first global access, so it never reads the scratch before the unpacking pass has finished
    attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[1].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 2;
    return cudaLaunchKernelEx(&cfg, xc_noalloc_i8_tc_kernel<UMMA_N, CG, BK>, tmap, tp);
}

}  // namespace

extern "C" int xc_correlate_i4_noalloc(int N, int F, int T, const uint8_t* in4_dev, int32_t* vis_dev, int accumulate,
                                       void* cuda_stream) {
    if (N < 1 || F < 1 || T < 1 || !in4_dev || !vis_dev) return XC_ERR_INVALID_ARG;
    if (T > XC_MAX_T) return XC_ERR_OVERFLOW;
    if (N > XC_NOALLOC_MAX_N) return XC_ERR_UNSUPPORTED;
    if (reinterpret_cast<uintptr_t>(vis_dev) & 15u) return XC_ERR_ALIGNMENT;
    // the unpacked block: T*F rows of 4N int8, rows padded to a multiple of 128 bytes -- must fit the fixed scratch
    const unsigned long long pitch = (4ull * N + 127ull) & ~127ull;
    const unsigned long long rows = static_cast<unsigned long long>(T) * static_cast<unsigned long long>(F);
    if (rows > XC_NOALLOC_SCRATCH_BYTES / pitch) return XC_ERR_NO_WORKSPACE;

    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) {
        (void)cudaGetLastError();
        return XC_ERR_CUDA;
    }
    NaDevice* d = nullptr;
    int rc = na_setup(dev, &d);
    if (rc != XC_OK) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);

    // Tile shape by the library's usual model (units of one 128 x 128 Gram block over the integration on one SM: a pair
    // tile is 4 blocks on 2 SMs, a single-CTA tile is 1 block but ~1.25x slower per block); the table must fit the kernel
    // parameters, which XC_NOALLOC_MAX_N guarantees for the pair tile.
    xc::TcParams tp;
    memset(&tp, 0, sizeof tp);
    uint32_t t_pair[xc::TC_INLINE_TILES], t_solo[xc::TC_INLINE_TILES];
    const int n_pair = na_tiles(N, 64, t_pair, xc::TC_INLINE_TILES);
    const int n_solo = na_tiles(N, 32, t_solo, xc::TC_INLINE_TILES);
    if (n_pair > xc::TC_INLINE_TILES) return XC_ERR_UNSUPPORTED;
    const long long pairs = d->sm_count / 2 > 0 ? d->sm_count / 2 : 1;
    const double c_pair = 2.0 * static_cast<double>((static_cast<long long>(n_pair) * F + pairs - 1) / pairs);
    const double c_solo = 1.25 * static_cast<double>((static_cast<long long>(n_solo) * F + d->sm_count - 1) / d->sm_count);
    const bool solo = n_solo <= xc::TC_INLINE_TILES && c_solo < 0.8 * c_pair;
    const int n_tiles = solo ? n_solo : n_pair;
    const long long total = static_cast<long long>(n_tiles) * F;
    if (total > 0x7FFFFFFFLL) return XC_ERR_UNSUPPORTED;

    // 1. unpack the 4-bit block into the scratch (`d->scratch` is the array's device address, see na_setup)
    const int npad = static_cast<int>(pitch / 4);
    const bool wide = (N % 8 == 0) && !(reinterpret_cast<uintptr_t>(in4_dev) & 15u);
    const long long items = static_cast<long long>(rows) * (wide ? N / 8 : npad);
    long long blocks = (items + 255) / 256;
    const long long cap = static_cast<long long>(d->sm_count) * 32;
    if (blocks > cap) blocks = cap;
    if (wide)
        xc_noalloc_unpack_i4x8_kernel<<<static_cast<unsigned>(blocks), 256, 0, st>>>(
            reinterpret_cast<const uint4*>(in4_dev), static_cast<uint4*>(d->scratch), static_cast<long long>(rows), N / 8, npad / 8);
    else
        xc_noalloc_unpack_i4_kernel<<<static_cast<unsigned>(blocks), 256, 0, st>>>(in4_dev, static_cast<uint32_t*>(d->scratch),
                                                                                static_cast<long long>(rows), N, npad);
    if (cudaGetLastError() != cudaSuccess) return XC_ERR_CUDA;

    // 2. tensor map over the scratch (host-only encode; bytes beyond 4N of a row, samples beyond T read as zero)
    CUtensorMap tmap;
    const cuuint64_t gdim[3] = {static_cast<cuuint64_t>(4) * N, static_cast<cuuint64_t>(F), static_cast<cuuint64_t>(T)};
    const cuuint64_t gstride[2] = {static_cast<cuuint64_t>(pitch), static_cast<cuuint64_t>(pitch) * static_cast<cuuint64_t>(F)};
    const cuuint32_t box[3] = {128, 1, static_cast<cuuint32_t>(solo ? 256 : 128)};
    const cuuint32_t estr[3] = {1, 1, 1};
    if (d->encode(&tmap, CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, d->scratch, gdim, gstride, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                  CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return XC_ERR_CUDA;

    // 3. the X-engine on it, into the caller's cube
    tp.N = N;
    tp.F = F;
    tp.T = T;
    tp.NB = static_cast<long long>(N) * (N + 1) / 2;
    tp.tiles_per_f = n_tiles;
    tp.total_tiles = static_cast<int>(total);
    tp.per_n = 1;                      // rows are 128-byte multiples apart: no origin shift
    tp.per_total = n_tiles;
    tp.per_cum[0] = 0;
    tp.per_cum[1] = static_cast<uint32_t>(n_tiles);
    tp.t_split = T;
    tp.tiles = nullptr;                // the table is inline (n_tiles <= TC_INLINE_TILES)
    tp.vis = vis_dev;
    tp.accumulate = accumulate ? 1 : 0;
    tp.stamps = nullptr;
    for (int k = 0; k < n_tiles; ++k) tp.tiles_inline[k] = solo ? t_solo[k] : t_pair[k];
    const cudaError_t e = solo ? na_launch<128, 1, 256>(tmap, tp, d->sm_count, st) : na_launch<256, 2, 128>(tmap, tp, d->sm_count, st);
    if (e != cudaSuccess) {
        (void)cudaGetLastError();
        return XC_ERR_CUDA;
    }
    return XC_OK;
}
