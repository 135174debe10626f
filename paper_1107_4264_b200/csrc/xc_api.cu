// xc_api.cu -- the C ABI of include/xc.h: plan (tile schedule, S1), dispatch of the staging (S0),
// tensor-core (S2-S4), fp32 (S5) and two-stream (S6) paths.  Host code only launches this
// library's own kernels; there is no CPU compute path.
#include "../../include/xc.h"

#include <cuda.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "xc_f32.cuh"
#include "xc_f32_tc.cuh"
#include "xc_fengine.cuh"
#include "xc_i8_tc.cuh"
#include "xc_simt.cuh"

namespace {

typedef CUresult (*PFN_encodeTiled)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                    const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                    CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// Tiles (bi on the i side in blocks of si stations, bj on the j side in blocks of sj stations)
// that contain at least one stored pair i <= j < N, in the paper's triangular order
// (PAPER.md:157): block row bj outermost, bi ascending inside it.
std::vector<uint32_t> build_tiles(int N, int si, int sj) {
    std::vector<uint32_t> t;
    const int nbj = (N + sj - 1) / sj;
    const int nbi = (N + si - 1) / si;
    for (int bj = 0; bj < nbj; ++bj) {
        const int jmax = (bj + 1) * sj - 1 < N - 1 ? (bj + 1) * sj - 1 : N - 1;
        for (int bi = 0; bi < nbi; ++bi) {
            if (bi * si <= jmax) t.push_back(static_cast<uint32_t>(bi) | (static_cast<uint32_t>(bj) << 16));
        }
    }
    return t;
}

}  // namespace

struct xc_plan_s {
    int N = 0, P = 0, F = 0, T = 0;
    long long NB = 0;
    size_t in_pitch = 0;    // bytes between consecutive (t, f) rows of a device input block (default 4N; xc_set_in_pitch)
    size_t pad_pitch = 0;   // 4N rounded up to 128 bytes: row pitch of the staging workspace and of the host paths' device scratch
    int tile_mode = 0;      // XC_TILE_*: shape of the tensor-core tile actually in use
    int t_split = 1;        // CTAs sharing one tile's time axis (single-CTA tile only): 1 or 2
    std::vector<uint32_t> tiles_tc, tiles_f32;
    std::vector<uint32_t> tiles_f32tc;                   // fp32 tensor-core path: 64 x 64-station pair tiles
    uint32_t* d_tiles_f32tc = nullptr;
    CUtensorMap tmap_f32;
    const void* tmap_f32_src = nullptr;
    int tmap_f32_nf = 0;
    size_t in_pitch_f32 = 0, tmap_f32_pitch = 0;         // bytes between (t, f) rows of a float block (default 16N; xc_set_in_pitch_f32)
    int opt_f32_kernel = XC_F32_KERNEL_AUTO, f32_kernel_used = 0;
    std::vector<uint32_t> tiles_tc_ext;                  // the same schedule with one more block row (origin shift): tiles_tc is its prefix
    int shift_period = 1, shift_bytes[8] = {0, 0, 0, 0, 0, 0, 0, 0}, shift_tiles[8] = {0, 0, 0, 0, 0, 0, 0, 0};   // what the last call used
    // device state (created lazily on the device current at first compute call)
    bool dev_ready = false, tiles_uploaded = false;
    int device = -1, sm_count = 0;
    uint32_t* d_tiles_tc = nullptr;
    uint32_t* d_tiles_f32 = nullptr;
    float2* d_twiddle = nullptr;                         // F-engine: exp(-2 pi i m / F), m < F (F a power of two <= 4096)
    int logf = -1;                                       // log2 F, or -1 when the F-engine cannot serve this F
    PFN_encodeTiled encode = nullptr;
    void* ws = nullptr;
    size_t ws_bytes = 0;
    bool ws_owned = false;
    cudaEvent_t ev_ws = nullptr;                         // recorded after the last consumer of the staging workspace
    int opt_kernel = XC_I8_KERNEL_AUTO, opt_max_ctas = 0, opt_force_stage = 0, opt_pdl = 1, opt_tsplit = 0;
    int opt_tile = XC_TILE_AUTO, opt_origin_shift = 1;
    unsigned long long* stamps = nullptr;                // xc_set_timing_buffer
#ifdef XC_PROFILE
    int opt_debug_skip = 0;
    long long* trace = nullptr;
#endif
    CUtensorMap tmap;
    const void* tmap_src = nullptr;
    size_t tmap_pitch = 0;
    int tmap_bk = 0, tmap_nf = 0, tmap_fchan = 0;
    cudaStream_t s_h2d = nullptr, s_d2h = nullptr;       // xc_correlate_host: plan-owned copy streams
    std::vector<cudaEvent_t> ev_chunk;                   // xc_correlate_host: per-chunk events
    cudaEvent_t ev_copied[2] = {nullptr, nullptr}, ev_free[2] = {nullptr, nullptr}, ev_entry = nullptr;
    int last_launches = 0;
    int copy_launches = 0;      // re-pitch kernels enqueued by copy_in_rows since the caller last reset it
    std::string last_err;
};

namespace {

int cuda_fail(xc_plan_t* p, cudaError_t e, const char* where) {
    if (p) p->last_err = std::string(where) + ": " + cudaGetErrorString(e);
    (void)cudaGetLastError();
    return XC_ERR_CUDA;
}
#define XC_CUDA(p, call)                                              \
    do {                                                              \
        cudaError_t e__ = (call);                                     \
        if (e__ != cudaSuccess) return cuda_fail((p), e__, #call);    \
    } while (0)

void tile_shape(int mode, int* si, int* sj) {
    *si = *sj = (mode == XC_TILE_2CTA_256x256) ? 64 : 32;
}

// T-split (single-CTA tile only): two CTAs of a cluster share one tile's time axis.  Worth it when (a) it leaves no SM
// without work it could have had, i.e. even the doubled unit count fits the machine in one wave, and (b) the tensor work
// it takes off the critical path -- T tensor-core cycles, half of a 128 x 128 tile's 2T -- exceeds what the cluster launch,
// the DSMEM hand-over of 64 KB of partial sums and its release/acquire pair cost: measured ~3.3 us ~ 6000 cycles
// (N = 32, F = 64: 7.0 us with the split against 5.0 us without at T = 2048), hence T >= 8192.
// Each rank needs at least one sample; a share is a whole multiple of the MMA's K = 32.
constexpr int kTSplitMinT = 8192;
int pick_t_split(const xc_plan_t* p, int nf, int sms) {
    if (p->tile_mode != XC_TILE_1CTA_128x128 || p->opt_tsplit == 1) return 1;
    const int share = ((p->T + 1) / 2 + 31) & ~31;
    if (share >= p->T) return 1;
    if (p->opt_tsplit == 2) return 2;
    return (p->T >= kTSplitMinT && static_cast<long long>(p->tiles_tc.size()) * nf * 2 <= sms) ? 2 : 1;
}

// S1: pick the tensor-core tile and build its per-channel schedule.
void set_tile_mode(xc_plan_t* p, int mode) {
    p->opt_tile = mode;
    if (mode == XC_TILE_AUTO) {
        // Modelled in units of "one 128 x 128 Gram block over the whole integration on one SM" (the paper's wasted-work
        // model, per SM): a CTA-pair 256x256 tile is 4 blocks on 2 SMs = 2 time units; single-CTA
        // 128x128 tiles are 1 unit each but bound by shared-memory bandwidth (measured ~1.25x slower per block), so they
        // only serve tiny problems.
        const double sms = p->sm_count > 0 ? p->sm_count : 148.0;
        const double n2 = static_cast<double>(build_tiles(p->N, 64, 64).size()) * p->F;
        const double n1 = static_cast<double>(build_tiles(p->N, 32, 32).size()) * p->F;
        const double t_pair = std::ceil(n2 / std::floor(sms / 2)) * 2.0;
        const double t_solo = std::ceil(n1 / sms) * 1.25;
        mode = (t_solo < 0.8 * t_pair) ? XC_TILE_1CTA_128x128 : XC_TILE_2CTA_256x256;
    }
    int si, sj;
    tile_shape(mode, &si, &sj);
    p->tile_mode = mode;
    p->tiles_tc = build_tiles(p->N, si, sj);
    p->tiles_tc_ext = build_tiles(p->N + si, si, sj);    // square tiles: block row bj holds bi = 0 .. bj, so tiles_tc is a prefix
    p->tiles_uploaded = false;
}

int upload_table(xc_plan_t* p, uint32_t** dst, const std::vector<uint32_t>& src) {
    if (*dst) XC_CUDA(p, cudaFree(*dst));   // synchronising; only after xc_set_option(XC_OPT_TILE)
    *dst = nullptr;
    if (src.empty()) return XC_OK;
    XC_CUDA(p, cudaMalloc(dst, src.size() * sizeof(uint32_t)));
    XC_CUDA(p, cudaMemcpy(*dst, src.data(), src.size() * sizeof(uint32_t), cudaMemcpyHostToDevice));
    return XC_OK;
}

int upload_tiles(xc_plan_t* p) {
    if (p->tiles_uploaded) return XC_OK;
    int rc = upload_table(p, &p->d_tiles_tc, p->tiles_tc_ext);
    if (rc != XC_OK) return rc;
    p->tiles_uploaded = true;
    return XC_OK;
}

template <int UMMA_N, int CG, int BK, int TS>
int launch_tc(xc_plan_t* p, const xc::TcParams& tp, cudaStream_t st) {
    using Cfg = xc::TcCfg<UMMA_N, CG, BK, TS>;
    constexpr int CL = CG * TS;                          // CTAs per work unit = cluster size
    long long units = (p->opt_max_ctas > 0 ? p->opt_max_ctas : p->sm_count) / CL;
    if (units < 1) units = 1;
    if (units > tp.total_tiles) units = tp.total_tiles;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(static_cast<unsigned>(units * CL));
    cfg.blockDim = dim3(xc::TC_THREADS);
    cfg.dynamicSmemBytes = Cfg::SMEM_BYTES;
    cfg.stream = st;
    cudaLaunchAttribute attr[2];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = CL;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    // programmatic dependent launch: this kernel's prologue may overlap the previous kernel's tail (it executes
    // griddepcontrol.wait before its first global access)
    attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[1].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    // With the timing buffer on, the kernel stamps it in its prologue, i.e. before griddepcontrol.wait: under programmatic
    // serialization that could run ahead of a preceding kernel that presets the buffer.  Timed launches are plain launches.
    cfg.numAttrs = (p->opt_pdl && !p->stamps) ? 2 : 1;
    XC_CUDA(p, cudaLaunchKernelEx(&cfg, xc::xc_i8_tc_kernel<UMMA_N, CG, BK, TS>, p->tmap, tp));
    p->last_launches += 1;
    return XC_OK;
}

// The dynamic shared-memory opt-in is per function and per device: done once per plan, for the device the plan binds to.
template <int UMMA_N, int CG, int BK, int TS>
cudaError_t opt_in_smem() {
    return cudaFuncSetAttribute(xc::xc_i8_tc_kernel<UMMA_N, CG, BK, TS>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                xc::TcCfg<UMMA_N, CG, BK, TS>::SMEM_BYTES);
}

// ---- F-engine host side --------------------------------------------------------------------------------
// exp(-2 pi i m / F) in fp64, then rounded to fp32.  The angle is folded into the first eighth of a turn so that the table
// is exact at quarter turns (0, +-1) and symmetric at odd eighth turns: integer-valued voltages then give exactly integer
// spectra in the bins 0, F/4, F/2, 3F/4, whatever the ties of the quantiser are.
void fe_twiddle(int F, int m, float* re, float* im) {
    const double kTwoPi = 6.283185307179586476925286766559;
    int e = static_cast<int>((8LL * m) / F);                     // eighth of the turn, 0..7
    long long rem = 8LL * m - static_cast<long long>(e) * F;     // in units of 1/(8F) turn, 0 <= rem < F
    bool mirror = (e & 1) != 0;                                  // odd eighths are reflected: angle = (e + 1) / 8 turn - theta
    if (mirror) rem = F - rem;
    const double theta = kTwoPi * static_cast<double>(rem) / (8.0 * static_cast<double>(F));
    double c = std::cos(theta), s = std::sin(theta);
    if (rem == 0) { c = 1.0; s = 0.0; }
    if (rem == F) { c = s = std::sqrt(0.5); }
    if (mirror) s = -s;
    const int quarter = ((e + (mirror ? 1 : 0)) / 2) & 3;        // quarter turns to add, exactly
    double cc = c, ss = s;
    if (quarter == 1) { cc = -s; ss = c; }
    else if (quarter == 2) { cc = -c; ss = -s; }
    else if (quarter == 3) { cc = s; ss = -c; }
    *re = static_cast<float>(cc);
    *im = static_cast<float>(-ss);
}

template <int LOGF>
cudaError_t fe_opt_in() {
    cudaError_t e = cudaFuncSetAttribute(xc::xc_fengine_kernel<LOGF, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(xc::xc_fengine_kernel<LOGF, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
}
template <int LOGF>
void fe_launch_one(const xc::FeParams& fp, unsigned grid, size_t tile, cudaStream_t st) {
    const size_t extra = xc::FeCfg<LOGF>::WORK_BYTES + xc::FeCfg<LOGF>::TW_BYTES;
    if (fp.spec) xc::xc_fengine_kernel<LOGF, true><<<grid, xc::FE_THREADS, extra, st>>>(fp);
    else xc::xc_fengine_kernel<LOGF, false><<<grid, xc::FE_THREADS, tile + extra, st>>>(fp);
}

#define XC_FE_FOR_ALL(X) X(0) X(1) X(2) X(3) X(4) X(5) X(6) X(7) X(8) X(9) X(10) X(11) X(12)

int fe_prepare(xc_plan_t* p) {
    p->logf = -1;
    for (int l = 0; l <= xc::FE_MAX_LOGF; ++l)
        if ((1 << l) == p->F) p->logf = l;
    if (p->logf < 0) return XC_OK;            // the F-engine calls will answer XC_ERR_UNSUPPORTED
    // Per-pass tables in the order the kernel reads them (xc_fengine.cuh, FeCfg): the log2 F bits are split over
    // NP passes (radix <= 16, or <= 32 for F = 512, 1024), the first (log2 F mod NP) passes one bit wider; pass i >= 1 with radix R_i on
    // sub-transforms of length NS_i multiplies leg r of butterfly k by exp(-2 pi i k r / (NS_i R_i)): entry [k][r - 1].
    std::vector<float2> tw;
    const int L = p->logf, NP = xc::fe_num_passes(L);
    int ns = 1;
    for (int i = 0; i < NP; ++i) {
        const int R = 1 << xc::fe_pass_bits(L, i);
        if (i >= 1)
            for (int k = 0; k < ns; ++k)
                for (int r = 1; r < R; ++r) {
                    float2 w;
                    fe_twiddle(p->F, k * r * (p->F / (ns * R)), &w.x, &w.y);
                    tw.push_back(w);
                }
        ns *= R;
    }
    if (tw.empty()) tw.push_back(make_float2(1.f, 0.f));
    if (!p->d_twiddle) XC_CUDA(p, cudaMalloc(&p->d_twiddle, sizeof(float2) * tw.size()));
    XC_CUDA(p, cudaMemcpy(p->d_twiddle, tw.data(), sizeof(float2) * tw.size(), cudaMemcpyHostToDevice));
    switch (p->logf) {
#define X(L) case L: XC_CUDA(p, fe_opt_in<L>()); break;
        XC_FE_FOR_ALL(X)
#undef X
        default: break;
    }
    return XC_OK;
}

int ensure_device(xc_plan_t* p);

// volt -> cube (quantised, rows `pitch` bytes apart) and / or spec (fp32, dense cube order)
int fengine_launch(xc_plan_t* p, const int8_t* volt, float scale, int8_t* cube, size_t pitch, float* spec, cudaStream_t st,
                   int f0 = 0, int nf = -1) {
    if (!p || !volt || (!cube && !spec)) return XC_ERR_INVALID_ARG;
    if (nf < 0) nf = p->F;
    if (f0 < 0 || nf < 1 || f0 + nf > p->F) return XC_ERR_INVALID_ARG;
    int rc = ensure_device(p);
    if (rc != XC_OK) return rc;
    if (p->logf < 0) {
        p->last_err = "the F-engine needs F to be a power of two <= 4096";
        return XC_ERR_UNSUPPORTED;
    }
    if ((reinterpret_cast<uintptr_t>(volt) & 1u) || (reinterpret_cast<uintptr_t>(cube) & 3u) || (reinterpret_cast<uintptr_t>(spec) & 7u))
        return XC_ERR_ALIGNMENT;
    if (cube && (pitch < static_cast<size_t>(4) * p->N || (pitch & 3u))) return XC_ERR_INVALID_ARG;
    // stations per CTA: 32 (128-byte rows) while the tile of one time block fits, else 16 or 8; never more than N needs
    int SB = 32;
    while (SB > 8 && (static_cast<long long>(SB) * 4 * p->F > xc::FE_TILE_BYTES || SB / 2 >= p->N)) SB /= 2;
    long long TT = xc::FE_TILE_BYTES / (static_cast<long long>(SB) * 4 * p->F);
    if (TT < 1) TT = 1;
    if (TT > p->T) TT = p->T;
    xc::FeParams fp;
    fp.N = p->N;
    fp.T = p->T;
    fp.SB = SB;
    fp.TT = static_cast<int>(TT);
    fp.nsb = (p->N + SB - 1) / SB;
    fp.pitch = static_cast<long long>(pitch);
    fp.f0 = f0;
    fp.nf = nf;
    fp.volt = volt;
    fp.cube = cube;
    fp.spec = spec;
    fp.tw = p->d_twiddle;
    fp.scale = scale;
    const long long grid = static_cast<long long>(fp.nsb) * ((p->T + TT - 1) / TT);
    if (grid > 0x7FFFFFFFLL) return XC_ERR_UNSUPPORTED;
    // output tile: 2 SB columns (signals) of TT * F two-byte samples, FE_COL_PAD bytes of padding per column
    const size_t tile = (static_cast<size_t>(2) * SB * (static_cast<size_t>(TT) * p->F * 2 + xc::FE_COL_PAD) + 15) & ~static_cast<size_t>(15);
    switch (p->logf) {
#define X(L) case L: fe_launch_one<L>(fp, static_cast<unsigned>(grid), tile, st); break;
        XC_FE_FOR_ALL(X)
#undef X
        default: return XC_ERR_UNSUPPORTED;
    }
    XC_CUDA(p, cudaGetLastError());
    p->last_launches = 1;
    return XC_OK;
}

int ensure_device(xc_plan_t* p) {
    int dev = 0;
    XC_CUDA(p, cudaGetDevice(&dev));
    if (p->dev_ready) {
        if (dev != p->device) {   // the plan's tables, workspace and streams live on the device of its first compute call
            p->last_err = "plan is bound to another CUDA device than the current one";
            return XC_ERR_INVALID_ARG;
        }
        return XC_OK;
    }
    int major = 0, sms = 0;
    XC_CUDA(p, cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
    XC_CUDA(p, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    if (major != 10) {
        p->last_err = "device is not sm_100 (tcgen05/TMEM required); there is no fallback path";
        return XC_ERR_UNSUPPORTED;
    }
    p->device = dev;
    if (sms != p->sm_count) {
        p->sm_count = sms;
        if (p->opt_tile == XC_TILE_AUTO) set_tile_mode(p, XC_TILE_AUTO);   // the model uses the real SM count
    }
    p->tiles_uploaded = false;
    int rc_up = upload_tiles(p);
    if (rc_up != XC_OK) return rc_up;
    if (!p->d_tiles_f32) {   // (a retry after a later failure re-uses what already exists)
        XC_CUDA(p, cudaMalloc(&p->d_tiles_f32, p->tiles_f32.size() * sizeof(uint32_t)));
        XC_CUDA(p, cudaMemcpy(p->d_tiles_f32, p->tiles_f32.data(), p->tiles_f32.size() * sizeof(uint32_t),
                              cudaMemcpyHostToDevice));
    }
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    XC_CUDA(p, cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres));
    if (!fn || qres != cudaDriverEntryPointSuccess) {
        p->last_err = "cuTensorMapEncodeTiled not available from the driver";
        return XC_ERR_CUDA;
    }
    p->encode = reinterpret_cast<PFN_encodeTiled>(fn);
    XC_CUDA(p, cudaFuncSetAttribute(xc::xc_f32_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                    xc::F32_SMEM_BYTES));
    if (!p->d_tiles_f32tc) {
        XC_CUDA(p, cudaMalloc(&p->d_tiles_f32tc, p->tiles_f32tc.size() * sizeof(uint32_t)));
        XC_CUDA(p, cudaMemcpy(p->d_tiles_f32tc, p->tiles_f32tc.data(), p->tiles_f32tc.size() * sizeof(uint32_t),
                              cudaMemcpyHostToDevice));
    }
    XC_CUDA(p, cudaFuncSetAttribute(xc::xc_f32_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, xc::FT_SMEM_BYTES));
    XC_CUDA(p, (opt_in_smem<256, 2, 128, 1>()));
    XC_CUDA(p, (opt_in_smem<128, 1, 256, 1>()));
    XC_CUDA(p, (opt_in_smem<128, 1, 256, 2>()));
    int rc_fe = fe_prepare(p);
    if (rc_fe != XC_OK) return rc_fe;
    p->dev_ready = true;
    return XC_OK;
}

bool needs_staging(const xc_plan_t* p, const void* in_dev, int fmt_i4) {
    if (fmt_i4 || p->opt_force_stage) return true;
    return (p->in_pitch & 15u) || (reinterpret_cast<uintptr_t>(in_dev) & 15u);
}

// S0: decide whether the staging kernel is needed and run it; *src / *pitch describe what TMA reads.
int stage_if_needed(xc_plan_t* p, const int8_t* in_dev, cudaStream_t st, const void** src, size_t* pitch, int fmt_i4 = 0,
                    int f0 = 0, int nf = -1) {
    if (nf < 0) nf = p->F;
    if (!needs_staging(p, in_dev, fmt_i4)) {
        *src = in_dev;
        *pitch = p->in_pitch;
        return XC_OK;
    }
    const size_t want = xc_workspace_bytes(p);
    if (!p->ws) {
        XC_CUDA(p, cudaMalloc(&p->ws, want));  // synchronising; documented in xc.h
        p->ws_bytes = want;
        p->ws_owned = true;
    }
    if (p->ws_bytes < want) return XC_ERR_NO_WORKSPACE;
    // the workspace is plan-wide: a call on another stream must not overwrite it while the previous call's X-engine reads it
    if (!p->ev_ws) XC_CUDA(p, cudaEventCreateWithFlags(&p->ev_ws, cudaEventDisableTiming));
    else XC_CUDA(p, cudaStreamWaitEvent(st, p->ev_ws, 0));
    const int npad = static_cast<int>(p->pad_pitch / 4);          // stations per workspace row (zero padded)
    const long long rows = static_cast<long long>(p->T) * p->F;
    const long long cap = static_cast<long long>(p->sm_count) * 32;
    auto grid = [&](long long items) {
        long long b = (items + 255) / 256;
        return static_cast<unsigned>(b < 1 ? 1 : (b > cap ? cap : b));
    };
    if (fmt_i4) {
        // 4-bit samples: the staging pass is the unpacking pass (in_dev then points at 2*N*F*T packed bytes)
        const long long units = static_cast<long long>(p->T) * nf * npad;
        if (p->N % 8 == 0 && !(reinterpret_cast<uintptr_t>(in_dev) & 15u)) {
            xc::xc_unpack_i4x8_kernel<<<grid(static_cast<long long>(p->T) * nf * (p->N / 8)), 256, 0, st>>>(
                reinterpret_cast<const uint4*>(in_dev), static_cast<uint4*>(p->ws), p->T, p->F, f0, nf, p->N / 8, npad / 8);
        } else {
            xc::xc_unpack_i4_kernel<<<grid(units), 256, 0, st>>>(
                reinterpret_cast<const uint8_t*>(in_dev), static_cast<uint32_t*>(p->ws), p->T, p->F, f0, nf, p->N, npad);
        }
    } else if (f0 != 0 || nf != p->F) {
        // a channel range of a block that needs staging: only the range's rows are copied (they keep their workspace rows)
        xc::xc_stage_pad_range_kernel<<<grid(static_cast<long long>(p->T) * nf * npad), 256, 0, st>>>(
            in_dev, static_cast<uint32_t*>(p->ws), p->T, p->F, f0, nf, p->N, static_cast<long long>(p->in_pitch), npad);
    } else if (p->N % 4 == 0 && p->in_pitch % 16 == 0 && !(reinterpret_cast<uintptr_t>(in_dev) & 15u)) {
        xc::xc_stage_pad16_kernel<<<grid(rows * (npad / 4)), 256, 0, st>>>(
            reinterpret_cast<const uint4*>(in_dev), static_cast<uint4*>(p->ws), rows, p->N / 4,
            static_cast<int>(p->in_pitch / 16), npad / 4);
    } else {
        xc::xc_stage_pad_kernel<<<grid(rows * npad), 256, 0, st>>>(in_dev, static_cast<uint32_t*>(p->ws), rows, p->N,
                                                                   static_cast<long long>(p->in_pitch), npad);
    }
    XC_CUDA(p, cudaGetLastError());
    p->last_launches += 1;
    *src = p->ws;
    *pitch = p->pad_pitch;
    return XC_OK;
}

// Tensor map over channels [.., nf) of the block that starts at src: rows of 4N valid bytes, `pitch` bytes apart (the
// channel pitch stays the plan's F).  Bytes beyond 4N of a row, stations beyond N and samples beyond T read as zero.
int encode_tmap(xc_plan_t* p, const void* src, size_t pitch, int bk, int nf, int fchan) {
    if (p->tmap_src == src && p->tmap_pitch == pitch && p->tmap_bk == bk && p->tmap_nf == nf && p->tmap_fchan == fchan) return XC_OK;
    const cuuint64_t gdim[3] = {static_cast<cuuint64_t>(4) * p->N, static_cast<cuuint64_t>(nf),
                                static_cast<cuuint64_t>(p->T)};
    const cuuint64_t gstride[2] = {static_cast<cuuint64_t>(pitch), static_cast<cuuint64_t>(pitch) * static_cast<cuuint64_t>(fchan)};
    const cuuint32_t box[3] = {128, 1, static_cast<cuuint32_t>(bk)};
    const cuuint32_t estr[3] = {1, 1, 1};
    CUresult r = p->encode(&p->tmap, CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, const_cast<void*>(src), gdim, gstride, box, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        char buf[96];
        snprintf(buf, sizeof buf, "cuTensorMapEncodeTiled failed with CUresult %d", static_cast<int>(r));
        p->last_err = buf;
        p->tmap_src = nullptr;
        return XC_ERR_CUDA;
    }
    p->tmap_src = src;
    p->tmap_pitch = pitch;
    p->tmap_bk = bk;
    p->tmap_nf = nf;
    p->tmap_fchan = fchan;
    return XC_OK;
}

// Origin shift ("rows aligned to the memory line").  Rows of the block TMA reads start at
// base + f pitch + t pitch F.  When pitch F is a multiple of 128 bytes the offset of a row inside its 128-byte line depends
// on f only, with a period of at most 8 channels (base and pitch are multiples of 16).  A box row that starts `shift` bytes
// into a line straddles two lines (two L2 requests, 5 sectors instead of 4: N = 500 ran 31 % slower than with padded
// rows); moving channel f's whole tile grid `shift` bytes to the left makes every box row exactly one line.  The price is
// that a class whose 4N + shift bytes need one more block row has more tiles; such a class keeps the unshifted grid when
// the extra tiles would cost more than the misaligned loads do (x 1.25, measured at N = 500).
// Fills the per-class fields of tp and the plan's record of them; returns the number of tiles of the nf channels.
long long plan_origin_shift(xc_plan_t* p, xc::TcParams* tp, const void* base, size_t pitch, int nf) {
    int si, sj;
    tile_shape(p->tile_mode, &si, &sj);
    const int mbytes = 4 * si;                                    // Gram rows (= bytes of a row) per tile
    const int n0 = (4 * p->N + mbytes - 1) / mbytes;
    const uintptr_t b = reinterpret_cast<uintptr_t>(base);
    int per = 1;
    const bool can = p->opt_origin_shift && ((pitch * static_cast<size_t>(p->F)) % 128u == 0);
    if (can && (pitch % 128u)) {
        per = 8;
        while (per > 1 && ((pitch * static_cast<size_t>(per / 2)) % 128u == 0)) per /= 2;
    }
    long long cum = 0;
    tp->per_n = per;
    tp->tiles_per_f = 0;
    tp->per_cum[0] = 0;
    for (int c = 0; c < 8; ++c) p->shift_bytes[c] = p->shift_tiles[c] = 0;
    for (int c = 0; c < per; ++c) {
        int shift = can ? static_cast<int>((b + static_cast<uintptr_t>(c) * pitch) & 127u) : 0;
        int n = (4 * p->N + shift + mbytes - 1) / mbytes;
        if (n > n0 && 4LL * n * (n + 1) > 5LL * n0 * (n0 + 1)) {   // more than 1.25 x the tiles: keep the unshifted grid
            shift = 0;
            n = n0;
        }
        const int tiles = n * (n + 1) / 2;
        tp->per_shift[c] = static_cast<uint8_t>(shift);
        cum += tiles;
        tp->per_cum[c + 1] = static_cast<uint32_t>(cum);
        if (tiles > tp->tiles_per_f) tp->tiles_per_f = tiles;
        p->shift_bytes[c] = shift;
        p->shift_tiles[c] = tiles;
    }
    tp->per_total = static_cast<int>(cum);
    p->shift_period = per;
    return static_cast<long long>(nf / per) * cum + tp->per_cum[nf % per];
}

// X-engine on channels [f0, f0 + nf) of the block at in_dev / the cube at vis_dev (both addressed with the plan's F).
// pitch_override != 0: in_dev is a device block with that row pitch (the host paths' re-pitched scratch, the F-engine's cube).
// range_only: in_dev holds ONLY the range's channels, nf rows per time sample (the F-engine's pruned cube, xc_fx_channels).
int correlate_i8(xc_plan_t* p, const int8_t* in_dev, int32_t* vis_dev, void* stream, int accumulate, int f0 = 0,
                 int nf = -1, int fmt_i4 = 0, size_t pitch_override = 0, bool range_only = false) {
    if (!p || !in_dev || !vis_dev) return XC_ERR_INVALID_ARG;
    if (nf < 0) nf = p->F;
    if (f0 < 0 || nf < 1 || f0 + nf > p->F) return XC_ERR_INVALID_ARG;
    const bool sub = (f0 != 0 || nf != p->F);
    if (reinterpret_cast<uintptr_t>(vis_dev) & 15u) return XC_ERR_ALIGNMENT;
    int rc = ensure_device(p);
    if (rc != XC_OK) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    p->last_launches = 0;

    const size_t pitch_saved = p->in_pitch;
    struct Restore { xc_plan_t* p; size_t v; ~Restore() { p->in_pitch = v; } } restore{p, pitch_saved};
    if (pitch_override) p->in_pitch = pitch_override;

    // a channel sub-range is read through its own tensor map (in place, or from its rows of the staging workspace): not
    // with the SIMT kernel
    if (sub && p->opt_kernel == XC_I8_KERNEL_SIMT) return XC_ERR_UNSUPPORTED;
    if (fmt_i4 && p->opt_kernel == XC_I8_KERNEL_SIMT) return XC_ERR_UNSUPPORTED;
    if (p->opt_kernel == XC_I8_KERNEL_SIMT) {
        if (p->F > 65535) return XC_ERR_UNSUPPORTED;
        xc::SimtParams sp{p->N, p->F, p->T, p->NB, static_cast<long long>(p->in_pitch), in_dev, vis_dev, accumulate};
        const long long nb = (p->N + xc::SIMT_B - 1) / xc::SIMT_B;
        dim3 grid(static_cast<unsigned>(nb * (nb + 1) / 2), static_cast<unsigned>(p->F));
        xc::xc_i8_simt_kernel<<<grid, dim3(xc::SIMT_B, xc::SIMT_B), 0, st>>>(sp);
        XC_CUDA(p, cudaGetLastError());
        p->last_launches += 1;
        return XC_OK;
    }

    const void* src = nullptr;
    size_t pitch = 0;
    rc = stage_if_needed(p, in_dev, st, &src, &pitch, fmt_i4, f0, nf);
    if (rc != XC_OK) return rc;
    const bool staged_in = (src != in_dev);
    const bool pair = (p->tile_mode == XC_TILE_2CTA_256x256);
    if (range_only && staged_in) return XC_ERR_UNSUPPORTED;       // a pruned cube is read in place (the library laid it out itself)
    const int8_t* base = static_cast<const int8_t*>(src) + (range_only ? 0 : pitch * static_cast<size_t>(f0));
    rc = encode_tmap(p, base, pitch, pair ? 128 : 256, nf, range_only ? nf : p->F);
    if (rc != XC_OK) return rc;

    rc = upload_tiles(p);
    if (rc != XC_OK) return rc;
    xc::TcParams tp;
    memset(&tp, 0, sizeof tp);
    tp.N = p->N;
    tp.F = nf;
    tp.T = p->T;
    tp.NB = p->NB;
    tp.vis = vis_dev + static_cast<size_t>(f0) * p->NB * 8;
    tp.accumulate = accumulate;
    tp.stamps = p->stamps;
#ifdef XC_PROFILE
    tp.debug_skip = p->opt_debug_skip;
    tp.trace = p->trace;
#endif
    const long long total = plan_origin_shift(p, &tp, base, pitch, nf);
    tp.tiles = p->d_tiles_tc;
    if (tp.tiles_per_f <= xc::TC_INLINE_TILES)
        for (int k = 0; k < tp.tiles_per_f; ++k) tp.tiles_inline[k] = p->tiles_tc_ext[k];
    if (total > 0x7FFFFFFFLL) return XC_ERR_UNSUPPORTED;
    tp.total_tiles = static_cast<int>(total);
    p->t_split = pick_t_split(p, nf, p->opt_max_ctas > 0 ? p->opt_max_ctas : p->sm_count);
    tp.t_split = p->t_split == 2 ? (((p->T + 1) / 2 + 31) & ~31) : p->T;
    if (pair) rc = launch_tc<256, 2, 128, 1>(p, tp, st);
    else if (p->t_split == 2) rc = launch_tc<128, 1, 256, 2>(p, tp, st);
    else rc = launch_tc<128, 1, 256, 1>(p, tp, st);
    if (rc == XC_OK && staged_in) XC_CUDA(p, cudaEventRecord(p->ev_ws, st));
    return rc;
}


// fp32 samples on the tensor cores (xc_f32_tc.cuh): tensor map over the dense float block, persistent CTA pairs.
int correlate_f32_tc(xc_plan_t* p, const float* in_dev, float* vis_dev, int accumulate, cudaStream_t st, int f0 = 0, int nf = -1) {
    if (nf < 0) nf = p->F;
    const size_t pitch = p->in_pitch_f32;                  // bytes between rows (16N unless xc_set_in_pitch_f32 was called)
    in_dev = reinterpret_cast<const float*>(reinterpret_cast<const char*>(in_dev) + pitch * static_cast<size_t>(f0));   // channels [f0, f0 + nf): the map starts at row f0, channel pitch stays F
    vis_dev += static_cast<size_t>(f0) * p->NB * 8;
    if (p->tmap_f32_src != in_dev || p->tmap_f32_nf != nf || p->tmap_f32_pitch != pitch) {
        const cuuint64_t gdim[3] = {static_cast<cuuint64_t>(4) * p->N, static_cast<cuuint64_t>(nf), static_cast<cuuint64_t>(p->T)};
        const cuuint64_t gstride[2] = {static_cast<cuuint64_t>(pitch), static_cast<cuuint64_t>(pitch) * static_cast<cuuint64_t>(p->F)};
        const cuuint32_t box[3] = {32, 1, static_cast<cuuint32_t>(xc::FT_BK)};
        const cuuint32_t estr[3] = {1, 1, 1};
        CUresult r = p->encode(&p->tmap_f32, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<float*>(in_dev), gdim, gstride, box, estr,
                               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) {
            char buf[96];
            snprintf(buf, sizeof buf, "cuTensorMapEncodeTiled (fp32) failed with CUresult %d", static_cast<int>(r));
            p->last_err = buf;
            p->tmap_f32_src = nullptr;
            return XC_ERR_CUDA;
        }
        p->tmap_f32_src = in_dev;
        p->tmap_f32_nf = nf;
        p->tmap_f32_pitch = pitch;
    }
    xc::F32TcParams tp;
    memset(&tp, 0, sizeof tp);
    tp.N = p->N;
    tp.F = nf;
    tp.T = p->T;
    tp.NB = p->NB;
    tp.vis = vis_dev;
    tp.accumulate = accumulate ? 1 : 0;
    tp.stamps = p->stamps;
    tp.tiles_per_f = static_cast<int>(p->tiles_f32tc.size());
    tp.tiles = p->d_tiles_f32tc;
    if (tp.tiles_per_f <= xc::FT_INLINE_TILES)
        for (int k = 0; k < tp.tiles_per_f; ++k) tp.tiles_inline[k] = p->tiles_f32tc[k];
    const long long total = static_cast<long long>(nf) * tp.tiles_per_f;
    if (total > 0x7FFFFFFFLL) return XC_ERR_UNSUPPORTED;
    tp.total_tiles = static_cast<int>(total);
    long long units = (p->opt_max_ctas > 0 ? p->opt_max_ctas : p->sm_count) / 2;
    if (units < 1) units = 1;
    if (units > total) units = total;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(static_cast<unsigned>(units * 2));
    cfg.blockDim = dim3(xc::FT_THREADS);
    cfg.dynamicSmemBytes = xc::FT_SMEM_BYTES;
    cfg.stream = st;
    cudaLaunchAttribute attr[2];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = 2;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[1].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = (p->opt_pdl && !p->stamps) ? 2 : 1;     // timed launches are plain launches (see launch_tc)
    XC_CUDA(p, cudaLaunchKernelEx(&cfg, xc::xc_f32_tc_kernel, p->tmap_f32, tp));
    p->last_launches = 1;
    return XC_OK;
}

}  // namespace

extern "C" {

int xc_plan(xc_plan_t** out, int N, int P, int F, int T, int layout) {
    if (!out) return XC_ERR_INVALID_ARG;
    *out = nullptr;
    if (N < 1 || F < 1 || T < 1) return XC_ERR_INVALID_ARG;
    if (P != 2 || layout != XC_LAYOUT_TFSPC) return XC_ERR_UNSUPPORTED;
    if (T > XC_MAX_T) return XC_ERR_OVERFLOW;
    if (N > 32768) return XC_ERR_UNSUPPORTED;  // tile indices are 16-bit; 4N*F*T must also fit the address space
    xc_plan_t* p = new (std::nothrow) xc_plan_s();
    if (!p) return XC_ERR_NO_MEMORY;
    p->N = N;
    p->P = P;
    p->F = F;
    p->T = T;
    p->NB = static_cast<long long>(N) * (N + 1) / 2;
    // Row pitch seen by TMA: a multiple of 16 bytes is mandatory.  A pitch that is not a multiple of 128 bytes makes
    // every 128-byte box row straddle two L2 lines (N = 500: 5 sectors per row instead of 4, ~25 % slower than N = 512,
    // PAPER.md:112, 149 "line-aligned rows").  Dense device input is read in place whenever the 16-byte rule holds (a
    // separate re-pitching pass costs more than it saves); everything the library lays out itself -- the
    // staging workspace, the device scratch of the host-buffer calls, the F-engine's cube -- uses the 128-byte pitch.
    p->in_pitch = static_cast<size_t>(4) * N;
    p->pad_pitch = (static_cast<size_t>(4) * N + 127) & ~static_cast<size_t>(127);
    p->in_pitch_f32 = static_cast<size_t>(16) * N;
    set_tile_mode(p, XC_TILE_AUTO);
    p->tiles_f32 = build_tiles(N, xc::F32_SI, xc::F32_SJ);
    p->tiles_f32tc = build_tiles(N, 64, 64);
    memset(&p->tmap_f32, 0, sizeof p->tmap_f32);
    memset(&p->tmap, 0, sizeof p->tmap);
    *out = p;
    return XC_OK;
}

void xc_destroy(xc_plan_t* p) {
    if (!p) return;
    if (p->d_tiles_tc) cudaFree(p->d_tiles_tc);
    if (p->d_tiles_f32) cudaFree(p->d_tiles_f32);
    if (p->d_tiles_f32tc) cudaFree(p->d_tiles_f32tc);
    if (p->d_twiddle) cudaFree(p->d_twiddle);
    if (p->ws && p->ws_owned) cudaFree(p->ws);
    for (int k = 0; k < 2; ++k) {
        if (p->ev_copied[k]) cudaEventDestroy(p->ev_copied[k]);
        if (p->ev_free[k]) cudaEventDestroy(p->ev_free[k]);
    }
    if (p->ev_entry) cudaEventDestroy(p->ev_entry);
    if (p->ev_ws) cudaEventDestroy(p->ev_ws);
    for (cudaEvent_t e : p->ev_chunk) cudaEventDestroy(e);
    if (p->s_h2d) cudaStreamDestroy(p->s_h2d);
    if (p->s_d2h) cudaStreamDestroy(p->s_d2h);
    delete p;
}

size_t xc_in_bytes(const xc_plan_t* p) { return p ? p->in_pitch * p->F * p->T : 0; }
size_t xc_in_pitch(const xc_plan_t* p) { return p ? p->in_pitch : 0; }
size_t xc_in_bytes_i4(const xc_plan_t* p) { return p ? static_cast<size_t>(2) * p->N * p->F * p->T : 0; }
size_t xc_in_bytes_f32(const xc_plan_t* p) { return p ? p->in_pitch_f32 * p->F * p->T : 0; }
size_t xc_in_pitch_f32(const xc_plan_t* p) { return p ? p->in_pitch_f32 : 0; }
int xc_set_in_pitch_f32(xc_plan_t* p, size_t row_pitch_bytes) {
    if (!p) return XC_ERR_INVALID_ARG;
    const size_t dense = static_cast<size_t>(16) * p->N;
    if (row_pitch_bytes == 0) row_pitch_bytes = dense;
    if (row_pitch_bytes < dense || (row_pitch_bytes & 15u)) return XC_ERR_INVALID_ARG;
    p->in_pitch_f32 = row_pitch_bytes;
    p->tmap_f32_src = nullptr;
    return XC_OK;
}
size_t xc_vis_bytes(const xc_plan_t* p) { return p ? static_cast<size_t>(32) * p->NB * p->F : 0; }
size_t xc_n_baselines(const xc_plan_t* p) { return p ? static_cast<size_t>(p->NB) : 0; }
size_t xc_scratch_pitch(const xc_plan_t* p) { return p ? p->pad_pitch : 0; }
size_t xc_scratch_in_bytes(const xc_plan_t* p) {
    if (!p) return 0;
    const size_t dense = (static_cast<size_t>(4) * p->N * p->F * p->T + 127) & ~static_cast<size_t>(127);   // halves of dev_buf2 stay aligned
    return p->pad_pitch * p->F * p->T + (p->pad_pitch == static_cast<size_t>(4) * p->N ? 0 : dense);
}
size_t xc_workspace_bytes(const xc_plan_t* p) { return p ? p->pad_pitch * p->F * p->T : 0; }

int xc_set_in_pitch(xc_plan_t* p, size_t row_pitch_bytes) {
    if (!p) return XC_ERR_INVALID_ARG;
    const size_t dense = static_cast<size_t>(4) * p->N;
    if (row_pitch_bytes == 0) row_pitch_bytes = dense;
    if (row_pitch_bytes < dense) return XC_ERR_INVALID_ARG;
    p->in_pitch = row_pitch_bytes;
    p->tmap_src = nullptr;
    return XC_OK;
}

int xc_set_workspace(xc_plan_t* p, void* ws_dev, size_t bytes) {
    if (!p) return XC_ERR_INVALID_ARG;
    if (ws_dev && (reinterpret_cast<uintptr_t>(ws_dev) & 127u)) return XC_ERR_ALIGNMENT;
    if (ws_dev && bytes < xc_workspace_bytes(p)) return XC_ERR_NO_WORKSPACE;
    if (p->ws && p->ws_owned) cudaFree(p->ws);
    p->ws = ws_dev;
    p->ws_bytes = ws_dev ? bytes : 0;
    p->ws_owned = false;
    p->tmap_src = nullptr;
    return XC_OK;
}

int xc_set_timing_buffer(xc_plan_t* p, uint64_t* stamps_dev) {
    if (!p) return XC_ERR_INVALID_ARG;
    if (reinterpret_cast<uintptr_t>(stamps_dev) & 7u) return XC_ERR_ALIGNMENT;
    p->stamps = reinterpret_cast<unsigned long long*>(stamps_dev);
    return XC_OK;
}

int xc_set_option(xc_plan_t* p, int option, int value) {
    if (!p) return XC_ERR_INVALID_ARG;
    switch (option) {
        case XC_OPT_I8_KERNEL:
            if (value < XC_I8_KERNEL_AUTO || value > XC_I8_KERNEL_SIMT) return XC_ERR_INVALID_ARG;
            p->opt_kernel = value;
            return XC_OK;
        case XC_OPT_MAX_CTAS:
            if (value < 0) return XC_ERR_INVALID_ARG;
            p->opt_max_ctas = value;
            return XC_OK;
        case XC_OPT_FORCE_STAGE:
            p->opt_force_stage = value ? 1 : 0;
            return XC_OK;
        case XC_OPT_TILE:
            if (value != XC_TILE_AUTO && value != XC_TILE_1CTA_128x128 && value != XC_TILE_2CTA_256x256) return XC_ERR_INVALID_ARG;
            set_tile_mode(p, value);
            return XC_OK;
        case XC_OPT_TSPLIT:
            if (value < 0 || value > 2) return XC_ERR_INVALID_ARG;
            p->opt_tsplit = value;
            return XC_OK;
        case XC_OPT_PDL:
            p->opt_pdl = value ? 1 : 0;
            return XC_OK;
        case XC_OPT_ORIGIN_SHIFT:
            p->opt_origin_shift = value ? 1 : 0;
            return XC_OK;
        case XC_OPT_F32_KERNEL:
            if (value < XC_F32_KERNEL_AUTO || value > XC_F32_KERNEL_TC) return XC_ERR_INVALID_ARG;
            p->opt_f32_kernel = value;
            return XC_OK;
#ifdef XC_PROFILE
        case XC_OPT_DEBUG_SKIP:
            p->opt_debug_skip = value & 15;
            return XC_OK;
#endif
        default:
            return XC_ERR_INVALID_ARG;
    }
}

int xc_correlate(xc_plan_t* p, const int8_t* in_dev, int32_t* vis_dev, void* stream) {
    return correlate_i8(p, in_dev, vis_dev, stream, 0);
}
int xc_correlate_acc(xc_plan_t* p, const int8_t* in_dev, int32_t* vis_dev, void* stream) {
    return correlate_i8(p, in_dev, vis_dev, stream, 1);
}

int xc_correlate_i4(xc_plan_t* p, const uint8_t* in4_dev, int32_t* vis_dev, int accumulate, void* stream) {
    return correlate_i8(p, reinterpret_cast<const int8_t*>(in4_dev), vis_dev, stream, accumulate ? 1 : 0, 0, -1, 1);
}

int xc_correlate_f32(xc_plan_t* p, const float* in_dev, float* vis_dev, int accumulate, void* stream) {
    if (!p || !in_dev || !vis_dev) return XC_ERR_INVALID_ARG;
    if ((reinterpret_cast<uintptr_t>(in_dev) & 15u) || (reinterpret_cast<uintptr_t>(vis_dev) & 15u))
        return XC_ERR_ALIGNMENT;
    int rc = ensure_device(p);
    if (rc != XC_OK) return rc;
    p->last_launches = 0;
    // Tensor cores (three TF32 MMAs per product, xc_f32_tc.cuh) by default: measured faster at every N (N = 8 .. 256, F T =
    // 131072: 3.3x .. 4.8x); the CUDA-core kernel (xc_f32.cuh, the paper's own register tiling) on request.
    const bool tc = p->opt_f32_kernel != XC_F32_KERNEL_CUDA_CORES;
    if (!tc && p->in_pitch_f32 != static_cast<size_t>(16) * p->N) return XC_ERR_UNSUPPORTED;   // the CUDA-core kernel reads dense rows
    p->f32_kernel_used = tc ? XC_F32_KERNEL_TC : XC_F32_KERNEL_CUDA_CORES;
    if (tc) return correlate_f32_tc(p, in_dev, vis_dev, accumulate, static_cast<cudaStream_t>(stream));
    xc::F32Params fp;
    fp.N = p->N;
    fp.F = p->F;
    fp.T = p->T;
    fp.tiles_per_f = static_cast<int>(p->tiles_f32.size());
    fp.NB = p->NB;
    fp.tiles = p->d_tiles_f32;
    fp.in = reinterpret_cast<const float4*>(in_dev);
    fp.vis = vis_dev;
    fp.accumulate = accumulate ? 1 : 0;
    const long long total = static_cast<long long>(p->F) * fp.tiles_per_f;
    if (total > 0x7FFFFFFFLL) return XC_ERR_UNSUPPORTED;
    xc::xc_f32_kernel<<<static_cast<unsigned>(total), xc::F32_THREADS, xc::F32_SMEM_BYTES,
                        static_cast<cudaStream_t>(stream)>>>(fp);
    XC_CUDA(p, cudaGetLastError());
    p->last_launches = 1;
    return XC_OK;
}

int xc_correlate_f32_channels(xc_plan_t* p, const float* in_dev, float* vis_dev, int f0, int nf, int accumulate, void* stream) {
    if (!p || !in_dev || !vis_dev) return XC_ERR_INVALID_ARG;
    if (f0 < 0 || nf < 1 || f0 + nf > p->F) return XC_ERR_INVALID_ARG;
    if ((reinterpret_cast<uintptr_t>(in_dev) & 15u) || (reinterpret_cast<uintptr_t>(vis_dev) & 15u)) return XC_ERR_ALIGNMENT;
    if (p->opt_f32_kernel == XC_F32_KERNEL_CUDA_CORES && (f0 != 0 || nf != p->F)) return XC_ERR_UNSUPPORTED;
    if (f0 == 0 && nf == p->F) return xc_correlate_f32(p, in_dev, vis_dev, accumulate, stream);
    int rc = ensure_device(p);
    if (rc != XC_OK) return rc;
    p->last_launches = 0;
    p->f32_kernel_used = XC_F32_KERNEL_TC;
    return correlate_f32_tc(p, in_dev, vis_dev, accumulate, static_cast<cudaStream_t>(stream), f0, nf);
}

int xc_f32_kernel_used(const xc_plan_t* p) { return p ? p->f32_kernel_used : 0; }

}  // extern "C"

namespace {

// Host -> device copy of channels [f0, f0 + nf) of one dense host block ([T][F] rows of 4N bytes) into the device
// scratch.  When 4N is a multiple of 128 the scratch is the dense block itself.  Otherwise the scratch holds two areas:
// [0, pad_pitch*F*T) the block with rows pad_pitch bytes apart (what the X-engine reads: line-aligned rows, PAPER.md:112,
// 149, and no 16-byte rule to break whatever N is), then the dense landing area of the copy; a small kernel spreads the
// rows (a pitched 2-D copy would do it in one step but runs at a quarter of the PCIe rate for 2000-byte rows: measured).
int copy_in_rows(xc_plan_t* p, int8_t* scratch, const int8_t* host, int f0, int nf, cudaStream_t st) {
    const size_t row = static_cast<size_t>(4) * p->N, dp = p->pad_pitch;
    int8_t* dense = (dp == row) ? scratch : scratch + dp * p->F * p->T;
    if (nf == p->F) {
        XC_CUDA(p, cudaMemcpyAsync(dense, host, row * p->F * p->T, cudaMemcpyHostToDevice, st));
    } else {
        XC_CUDA(p, cudaMemcpy2DAsync(dense + row * f0, row * p->F, host + row * f0, row * p->F, row * nf,
                                     static_cast<size_t>(p->T), cudaMemcpyHostToDevice, st));
    }
    if (dp == row) return XC_OK;
    const long long cap = static_cast<long long>(p->sm_count) * 16;
    auto grid = [&](long long items) {
        long long b = (items + 255) / 256;
        return static_cast<unsigned>(b < 1 ? 1 : (b > cap ? cap : b));
    };
    if (row % 16 == 0)
        xc::xc_repitch_kernel<uint4><<<grid(static_cast<long long>(p->T) * nf * (row / 16)), 256, 0, st>>>(
            reinterpret_cast<const uint4*>(dense), reinterpret_cast<uint4*>(scratch), p->T, p->F, f0, nf,
            static_cast<int>(row / 16), static_cast<long long>(dp / 16));
    else
        xc::xc_repitch_kernel<uint32_t><<<grid(static_cast<long long>(p->T) * nf * p->N), 256, 0, st>>>(
            reinterpret_cast<const uint32_t*>(dense), reinterpret_cast<uint32_t*>(scratch), p->T, p->F, f0, nf, p->N,
            static_cast<long long>(dp / 4));
    XC_CUDA(p, cudaGetLastError());
    p->copy_launches += 1;
    return XC_OK;
}

int make_pipeline_events(xc_plan_t* p) {
    for (int k = 0; k < 2; ++k) {
        if (!p->ev_copied[k]) XC_CUDA(p, cudaEventCreateWithFlags(&p->ev_copied[k], cudaEventDisableTiming));
        if (!p->ev_free[k]) XC_CUDA(p, cudaEventCreateWithFlags(&p->ev_free[k], cudaEventDisableTiming));
    }
    if (!p->ev_entry) XC_CUDA(p, cudaEventCreateWithFlags(&p->ev_entry, cudaEventDisableTiming));
    return XC_OK;
}

// Algorithm 1 read as textbook double buffering; vis64_dev != null adds the int64 widening of xc_integrate.
int pipeline_blocks(xc_plan_t* p, const int8_t* in_host, int n_blocks, int8_t* dev_buf2, int32_t* vis32_dev,
                    int64_t* vis64_dev, int64_t* vis64_host, void* compute_stream, void* copy_stream) {
    if (reinterpret_cast<uintptr_t>(dev_buf2) & 127u) return XC_ERR_ALIGNMENT;
    int rc = ensure_device(p);
    if (rc != XC_OK) return rc;
    rc = make_pipeline_events(p);
    if (rc != XC_OK) return rc;
    cudaStream_t cs = static_cast<cudaStream_t>(compute_stream), xs = static_cast<cudaStream_t>(copy_stream);
    const size_t blk_host = static_cast<size_t>(4) * p->N * p->F * p->T;
    const size_t blk_dev = xc_scratch_in_bytes(p);
    const int group = XC_MAX_T / p->T;              // blocks whose int32 partial sum cannot overflow (>= 1)
    const long long n4 = static_cast<long long>(p->F) * p->NB * 2;   // int4 quadruples in the cube
    long long wblocks = (n4 + 255) / 256;
    if (wblocks > static_cast<long long>(p->sm_count) * 16) wblocks = static_cast<long long>(p->sm_count) * 16;
    int launches = 0;
    p->copy_launches = 0;
    // Earlier work on the compute stream may still read dev_buf2: copies start after it.
    XC_CUDA(p, cudaEventRecord(p->ev_entry, cs));
    XC_CUDA(p, cudaStreamWaitEvent(xs, p->ev_entry, 0));
    rc = copy_in_rows(p, dev_buf2, in_host, 0, p->F, xs);
    if (rc != XC_OK) return rc;
    XC_CUDA(p, cudaEventRecord(p->ev_copied[0], xs));
    for (int b = 0; b < n_blocks; ++b) {
        if (b + 1 < n_blocks) {
            const int nb = (b + 1) & 1;
            if (b >= 1) XC_CUDA(p, cudaStreamWaitEvent(xs, p->ev_free[nb], 0));  // X-engine on block b-1 is done with it
            rc = copy_in_rows(p, dev_buf2 + nb * blk_dev, in_host + static_cast<size_t>(b + 1) * blk_host, 0, p->F, xs);
            if (rc != XC_OK) return rc;
            XC_CUDA(p, cudaEventRecord(p->ev_copied[nb], xs));
        }
        XC_CUDA(p, cudaStreamWaitEvent(cs, p->ev_copied[b & 1], 0));
        const int acc = vis64_dev ? ((b % group) ? 1 : 0) : (b > 0 ? 1 : 0);
        rc = correlate_i8(p, dev_buf2 + (b & 1) * blk_dev, vis32_dev, compute_stream, acc, 0, -1, 0, p->pad_pitch);
        if (rc != XC_OK) return rc;
        launches += p->last_launches;
        XC_CUDA(p, cudaEventRecord(p->ev_free[b & 1], cs));
        if (vis64_dev && ((b + 1) % group == 0 || b + 1 == n_blocks)) {
            xc::xc_widen_kernel<<<static_cast<unsigned>(wblocks), 256, 0, cs>>>(
                reinterpret_cast<const int4*>(vis32_dev), reinterpret_cast<longlong2*>(vis64_dev), n4, b < group ? 1 : 0);
            XC_CUDA(p, cudaGetLastError());
            launches += 1;
        }
    }
    if (vis64_dev && vis64_host)
        XC_CUDA(p, cudaMemcpyAsync(vis64_host, vis64_dev, 2 * xc_vis_bytes(p), cudaMemcpyDeviceToHost, cs));
    p->last_launches = launches + p->copy_launches;
    return XC_OK;
}

int correlate_host_impl(xc_plan_t* p, const int8_t* in_host, int32_t* vis_host, int8_t* in_dev_scratch,
                        int32_t* vis_dev_scratch, void* stream, int fmt_i4) {
    if (!p || !in_host || !vis_host || !in_dev_scratch || !vis_dev_scratch) return XC_ERR_INVALID_ARG;
    if (reinterpret_cast<uintptr_t>(in_dev_scratch) & 15u) return XC_ERR_ALIGNMENT;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    int rc = ensure_device(p);
    if (rc != XC_OK) return rc;
    const size_t in_bytes = fmt_i4 ? xc_in_bytes_i4(p) : static_cast<size_t>(4) * p->N * p->F * p->T;
    const size_t pitch = fmt_i4 ? 0 : p->pad_pitch;     // int8: the device scratch is re-pitched by the copy itself
    int chunks = p->F < 16 ? p->F : 16;
    if ((!fmt_i4 && p->opt_force_stage) || p->opt_kernel == XC_I8_KERNEL_SIMT || in_bytes < (static_cast<size_t>(8) << 20)) chunks = 1;
    p->copy_launches = 0;
    if (chunks == 1) {
        if (fmt_i4) XC_CUDA(p, cudaMemcpyAsync(in_dev_scratch, in_host, in_bytes, cudaMemcpyHostToDevice, st));
        else if ((rc = copy_in_rows(p, in_dev_scratch, in_host, 0, p->F, st)) != XC_OK) return rc;
        rc = correlate_i8(p, in_dev_scratch, vis_dev_scratch, stream, 0, 0, -1, fmt_i4, pitch);
        if (rc != XC_OK) return rc;
        p->last_launches += p->copy_launches;
        XC_CUDA(p, cudaMemcpyAsync(vis_host, vis_dev_scratch, xc_vis_bytes(p), cudaMemcpyDeviceToHost, st));
        XC_CUDA(p, cudaStreamSynchronize(st));
        return XC_OK;
    }
    // Channels are independent, so the block is cut into channel ranges and the three legs of the
    // paper's integrated run (host->device, X-engine, device->host: Fig. 7) overlap: range c+1 is
    // copied in (a strided copy: T slices of the range's rows) while range c is correlated and range c-1 is
    // copied out, on two plan-owned copy streams ordered against the caller's stream by events.
    if (!p->s_h2d) XC_CUDA(p, cudaStreamCreateWithFlags(&p->s_h2d, cudaStreamNonBlocking));
    if (!p->s_d2h) XC_CUDA(p, cudaStreamCreateWithFlags(&p->s_d2h, cudaStreamNonBlocking));
    while (p->ev_chunk.size() < static_cast<size_t>(2 * chunks + 2)) {
        cudaEvent_t e = nullptr;
        XC_CUDA(p, cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        p->ev_chunk.push_back(e);
    }
    cudaEvent_t ev_entry = p->ev_chunk[2 * chunks], ev_done = p->ev_chunk[2 * chunks + 1];
    XC_CUDA(p, cudaEventRecord(ev_entry, st));           // earlier work on the caller's stream may still use the scratch
    XC_CUDA(p, cudaStreamWaitEvent(p->s_h2d, ev_entry, 0));
    XC_CUDA(p, cudaStreamWaitEvent(p->s_d2h, ev_entry, 0));
    const size_t row4 = static_cast<size_t>(2) * p->N;    // 4-bit: bytes of one (t, f) row
    int launches = 0;
    for (int c = 0; c < chunks; ++c) {
        const int f0 = static_cast<int>(static_cast<long long>(p->F) * c / chunks);
        const int f1 = static_cast<int>(static_cast<long long>(p->F) * (c + 1) / chunks);
        if (fmt_i4) {
            XC_CUDA(p, cudaMemcpy2DAsync(in_dev_scratch + row4 * f0, row4 * p->F, in_host + row4 * f0, row4 * p->F,
                                         row4 * (f1 - f0), static_cast<size_t>(p->T), cudaMemcpyHostToDevice, p->s_h2d));
        } else if ((rc = copy_in_rows(p, in_dev_scratch, in_host, f0, f1 - f0, p->s_h2d)) != XC_OK) {
            return rc;
        }
        XC_CUDA(p, cudaEventRecord(p->ev_chunk[2 * c], p->s_h2d));
        XC_CUDA(p, cudaStreamWaitEvent(st, p->ev_chunk[2 * c], 0));
        rc = correlate_i8(p, in_dev_scratch, vis_dev_scratch, stream, 0, f0, f1 - f0, fmt_i4, pitch);
        if (rc != XC_OK) return rc;
        launches += p->last_launches;
        XC_CUDA(p, cudaEventRecord(p->ev_chunk[2 * c + 1], st));
        XC_CUDA(p, cudaStreamWaitEvent(p->s_d2h, p->ev_chunk[2 * c + 1], 0));
        const size_t voff = static_cast<size_t>(f0) * p->NB * 8;
        XC_CUDA(p, cudaMemcpyAsync(vis_host + voff, vis_dev_scratch + voff, static_cast<size_t>(f1 - f0) * p->NB * 32,
                                   cudaMemcpyDeviceToHost, p->s_d2h));
    }
    XC_CUDA(p, cudaEventRecord(ev_done, p->s_d2h));
    XC_CUDA(p, cudaStreamWaitEvent(st, ev_done, 0));
    XC_CUDA(p, cudaStreamSynchronize(st));
    p->last_launches = launches + p->copy_launches;
    return XC_OK;
}

}  // namespace

extern "C" {

int xc_correlate_pipelined(xc_plan_t* p, const int8_t* in_host, int n_blocks, int8_t* dev_buf2, int32_t* vis_dev,
                           void* compute_stream, void* copy_stream) {
    if (!p || !in_host || !dev_buf2 || !vis_dev || n_blocks < 1) return XC_ERR_INVALID_ARG;
    return pipeline_blocks(p, in_host, n_blocks, dev_buf2, vis_dev, nullptr, nullptr, compute_stream, copy_stream);
}

int xc_integrate(xc_plan_t* p, const int8_t* in_host, int n_blocks, int8_t* dev_buf2, int32_t* vis32_dev,
                 int64_t* vis64_dev, int64_t* vis64_host, void* compute_stream, void* copy_stream) {
    if (!p || !in_host || !dev_buf2 || !vis32_dev || !vis64_dev || n_blocks < 1) return XC_ERR_INVALID_ARG;
    if (reinterpret_cast<uintptr_t>(vis64_dev) & 15u) return XC_ERR_ALIGNMENT;
    return pipeline_blocks(p, in_host, n_blocks, dev_buf2, vis32_dev, vis64_dev, vis64_host, compute_stream, copy_stream);
}

int xc_correlate_channels(xc_plan_t* p, const int8_t* in_dev, int32_t* vis_dev, int f0, int nf, int accumulate,
                          void* stream) {
    return correlate_i8(p, in_dev, vis_dev, stream, accumulate ? 1 : 0, f0, nf);
}

int xc_correlate_host(xc_plan_t* p, const int8_t* in_host, int32_t* vis_host, int8_t* in_dev_scratch,
                      int32_t* vis_dev_scratch, void* stream) {
    return correlate_host_impl(p, in_host, vis_host, in_dev_scratch, vis_dev_scratch, stream, 0);
}

int xc_correlate_host_i4(xc_plan_t* p, const uint8_t* in4_host, int32_t* vis_host, uint8_t* in4_dev_scratch,
                         int32_t* vis_dev_scratch, void* stream) {
    return correlate_host_impl(p, reinterpret_cast<const int8_t*>(in4_host), vis_host, reinterpret_cast<int8_t*>(in4_dev_scratch),
                               vis_dev_scratch, stream, 1);
}

#ifdef XC_PROFILE
int xc_debug_set_trace(xc_plan_t* p, void* trace_dev) {
    if (!p) return XC_ERR_INVALID_ARG;
    p->trace = static_cast<long long*>(trace_dev);
    return XC_OK;
}
#endif

size_t xc_volt_bytes(const xc_plan_t* p) { return p ? static_cast<size_t>(4) * p->N * p->F * p->T : 0; }
size_t xc_cube_bytes(const xc_plan_t* p) { return p ? p->pad_pitch * p->F * p->T : 0; }

int xc_fengine(xc_plan_t* p, const int8_t* volt_dev, float scale, int8_t* cube_dev, size_t cube_pitch, void* stream) {
    if (!p || !cube_dev) return XC_ERR_INVALID_ARG;
    return fengine_launch(p, volt_dev, scale, cube_dev, cube_pitch ? cube_pitch : p->pad_pitch, nullptr,
                          static_cast<cudaStream_t>(stream));
}

int xc_fengine_f32(xc_plan_t* p, const int8_t* volt_dev, float* spec_dev, void* stream) {
    if (!p || !spec_dev) return XC_ERR_INVALID_ARG;
    return fengine_launch(p, volt_dev, 1.0f, nullptr, 0, spec_dev, static_cast<cudaStream_t>(stream));
}

int xc_fx(xc_plan_t* p, const int8_t* volt_dev, float scale, int8_t* cube_scratch_dev, int32_t* vis_dev, int accumulate,
          void* stream) {
    if (!p || !cube_scratch_dev || !vis_dev) return XC_ERR_INVALID_ARG;
    if (reinterpret_cast<uintptr_t>(cube_scratch_dev) & 15u) return XC_ERR_ALIGNMENT;
    int rc = fengine_launch(p, volt_dev, scale, cube_scratch_dev, p->pad_pitch, nullptr, static_cast<cudaStream_t>(stream));
    if (rc != XC_OK) return rc;
    rc = correlate_i8(p, cube_scratch_dev, vis_dev, stream, accumulate ? 1 : 0, 0, -1, 0, p->pad_pitch);
    if (rc == XC_OK) p->last_launches += 1;
    return rc;
}

int xc_fengine_channels(xc_plan_t* p, const int8_t* volt_dev, float scale, int8_t* cube_dev, size_t cube_pitch, int f0, int nf,
                        void* stream) {
    if (!p || !cube_dev) return XC_ERR_INVALID_ARG;
    return fengine_launch(p, volt_dev, scale, cube_dev, cube_pitch ? cube_pitch : p->pad_pitch, nullptr,
                          static_cast<cudaStream_t>(stream), f0, nf);
}

int xc_fx_channels(xc_plan_t* p, const int8_t* volt_dev, float scale, int8_t* cube_scratch_dev, int32_t* vis_dev, int f0, int nf,
                   int accumulate, void* stream) {
    if (!p || !cube_scratch_dev || !vis_dev) return XC_ERR_INVALID_ARG;
    if (reinterpret_cast<uintptr_t>(cube_scratch_dev) & 15u) return XC_ERR_ALIGNMENT;
    if (p->opt_kernel == XC_I8_KERNEL_SIMT || p->opt_force_stage) return XC_ERR_UNSUPPORTED;
    int rc = fengine_launch(p, volt_dev, scale, cube_scratch_dev, p->pad_pitch, nullptr, static_cast<cudaStream_t>(stream), f0, nf);
    if (rc != XC_OK) return rc;
    rc = correlate_i8(p, cube_scratch_dev, vis_dev, stream, accumulate ? 1 : 0, f0, nf, 0, p->pad_pitch, true);
    if (rc == XC_OK) p->last_launches += 1;
    return rc;
}

int xc_tile_count(const xc_plan_t* p) { return p ? static_cast<int>(p->tiles_tc.size()) : 0; }

int xc_tile_get(const xc_plan_t* p, int k, int* bi, int* bj, int* si, int* sj) {
    if (!p || k < 0 || k >= static_cast<int>(p->tiles_tc.size())) return XC_ERR_INVALID_ARG;
    const uint32_t e = p->tiles_tc[k];
    int a = 0, b = 0;
    tile_shape(p->tile_mode, &a, &b);
    if (bi) *bi = static_cast<int>(e & 0xFFFFu);
    if (bj) *bj = static_cast<int>(e >> 16);
    if (si) *si = a;
    if (sj) *sj = b;
    return XC_OK;
}

int xc_t_split(const xc_plan_t* p) { return p ? p->t_split : 0; }

int xc_origin_shift_plan(xc_plan_t* p, uint64_t base_addr, size_t row_pitch_bytes, int* shift_bytes, int* tiles) {
    if (!p || (base_addr & 15u) || (row_pitch_bytes & 15u) || row_pitch_bytes < static_cast<size_t>(4) * p->N) return 0;
    xc::TcParams tp;
    memset(&tp, 0, sizeof tp);
    plan_origin_shift(p, &tp, reinterpret_cast<const void*>(static_cast<uintptr_t>(base_addr)), row_pitch_bytes, p->F);
    return xc_origin_shift(p, shift_bytes, tiles);
}

int xc_origin_shift(const xc_plan_t* p, int* shift_bytes, int* tiles) {
    if (!p) return 0;
    for (int c = 0; c < p->shift_period; ++c) {
        if (shift_bytes) shift_bytes[c] = p->shift_bytes[c];
        if (tiles) tiles[c] = p->shift_tiles[c];
    }
    return p->shift_period;
}

int64_t xc_tri_index(int64_t bx, int64_t by) { return by * (by + 1) / 2 + bx; }

void xc_tri_inverse(int64_t g, int64_t* bx, int64_t* by) {
    long long x = 0, y = 0;
    xc::tri_inverse(g, &x, &y);
    if (bx) *bx = x;
    if (by) *by = y;
}

int xc_last_launches(const xc_plan_t* p) { return p ? p->last_launches : 0; }

const char* xc_status_string(int s) {
    switch (s) {
        case XC_OK: return "XC_OK";
        case XC_ERR_INVALID_ARG: return "XC_ERR_INVALID_ARG";
        case XC_ERR_UNSUPPORTED: return "XC_ERR_UNSUPPORTED";
        case XC_ERR_OVERFLOW: return "XC_ERR_OVERFLOW";
        case XC_ERR_ALIGNMENT: return "XC_ERR_ALIGNMENT";
        case XC_ERR_CUDA: return "XC_ERR_CUDA";
        case XC_ERR_NO_WORKSPACE: return "XC_ERR_NO_WORKSPACE";
        case XC_ERR_NO_MEMORY: return "XC_ERR_NO_MEMORY";
        default: return "XC_ERR_UNKNOWN";
    }
}

const char* xc_last_cuda_error(const xc_plan_t* p) { return p ? p->last_err.c_str() : ""; }

const char* xc_version(void) {
#ifdef XC_PROFILE
    return "xcorr-b200 0.2 (sm_100a, tcgen05 kind::i8) [XC_PROFILE build]";
#else
    return "xcorr-b200 0.2 (sm_100a, tcgen05 kind::i8)";
#endif
}

}  // extern "C"
