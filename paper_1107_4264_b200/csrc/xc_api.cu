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

// XC_TILE_SPLIT, diagonal part: per 64-station diagonal block k two single-CTA sub-tiles, rows 2k (32 stations)
// against both 32-station column boxes of block k, and rows 2k+1 against the second box only (padding entry
// 0xFFFFFFFF where that row block starts beyond N).  Always two entries per k: the kernel walks them as a group.
std::vector<uint32_t> build_tiles_diag(int N) {
    std::vector<uint32_t> t;
    const int nb = (N + 63) / 64;
    for (int k = 0; k < nb; ++k) {
        t.push_back(static_cast<uint32_t>(2 * k) | (static_cast<uint32_t>(k) << 16));
        t.push_back((2 * k + 1) * 32 < N ? (static_cast<uint32_t>(2 * k + 1) | (static_cast<uint32_t>(k) << 16)) : 0xFFFFFFFFu);
    }
    return t;
}
// XC_TILE_SPLIT, off-diagonal part: the 64 x 64-station blocks strictly below the diagonal (bi < bj), CTA pairs.
std::vector<uint32_t> build_tiles_off(int N) {
    std::vector<uint32_t> t;
    const int nb = (N + 63) / 64;
    for (int bj = 0; bj < nb; ++bj)
        for (int bi = 0; bi < bj; ++bi) t.push_back(static_cast<uint32_t>(bi) | (static_cast<uint32_t>(bj) << 16));
    return t;
}

// XC_TILE_MIXED: how many of the `clusters` 2-CTA clusters work as two single CTAs on diagonal blocks (3 time units
// per block per CTA); the others work as pairs on off-diagonal tiles (2 units per tile).  Minimises the modelled
// makespan; *t_out receives it.
int mixed_split(int N, int F, int clusters, double* t_out) {
    const double gd = static_cast<double>((N + 63) / 64) * F;
    const double go = static_cast<double>(build_tiles_off(N).size()) * F;
    int best_n = clusters;
    double best_t = std::ceil(gd / (2.0 * clusters)) * 3.0;
    if (go > 0) {
        best_t = 1e300;
        for (int n = 1; n < clusters; ++n) {
            const double t = std::max(std::ceil(gd / (2.0 * n)) * 3.0, std::ceil(go / (clusters - n)) * 2.0);
            if (t < best_t) { best_t = t; best_n = n; }
        }
    }
    if (t_out) *t_out = best_t;
    return best_n;
}

}  // namespace

struct xc_plan_s {
    int N = 0, P = 0, F = 0, T = 0;
    long long NB = 0;
    int Npad = 0;
    int tile_mode = 0;  // XC_TILE_*: shape of the tensor-core tile actually in use
    std::vector<uint32_t> tiles_tc, tiles_f32;
    std::vector<uint32_t> tiles_diag;   // XC_TILE_SPLIT: diagonal sub-tiles (tiles_tc then holds the off-diagonal pair tiles)
    // device state (created lazily on the device current at first compute call)
    bool dev_ready = false, tiles_uploaded = false;
    int device = -1, sm_count = 0;
    uint32_t* d_tiles_tc = nullptr;
    uint32_t* d_tiles_diag = nullptr;
    uint32_t* d_tiles_f32 = nullptr;
    PFN_encodeTiled encode = nullptr;
    void* ws = nullptr;
    size_t ws_bytes = 0;
    bool ws_owned = false;
    int opt_kernel = XC_I8_KERNEL_AUTO, opt_max_ctas = 0, opt_force_stage = 0, opt_debug_skip = 0, opt_epilogue = 0, opt_bk = 0, opt_pdl = 1;
    long long* trace = nullptr;
    CUtensorMap tmap;
    const void* tmap_src = nullptr;
    int tmap_nrow = 0, tmap_bk = 0, tmap_nf = 0;
    cudaStream_t s_h2d = nullptr, s_d2h = nullptr;       // xc_correlate_host: plan-owned copy streams
    std::vector<cudaEvent_t> ev_chunk;                   // xc_correlate_host: per-chunk events
    cudaEvent_t ev_copied[2] = {nullptr, nullptr}, ev_free[2] = {nullptr, nullptr}, ev_entry = nullptr;
    int last_launches = 0;
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
    *si = (mode == XC_TILE_2CTA_256x256 || mode == XC_TILE_SPLIT || mode == XC_TILE_MIXED) ? 64 : 32;
    *sj = (mode == XC_TILE_1CTA_128x128) ? 32 : 64;
}

// S1: pick the tensor-core tile and build its per-channel schedule.
void set_tile_mode(xc_plan_t* p, int mode) {
    if (mode == XC_TILE_AUTO) {
        // Modelled in units of "one 128 x 128 Gram block over the whole integration on one SM" (the paper's wasted-work
        // model, per SM): a CTA-pair 256x256 tile is 4 blocks on 2 SMs = 2 time units; single-CTA
        // 128x128 tiles are 1 unit each but fill-bound (measured ~1.25x slower per block), so they only serve tiny
        // problems.  XC_TILE_MIXED / XC_TILE_SPLIT compute 5-17 % fewer blocks but measured 15-25 % SLOWER (their
        // single-CTA workers are bound by the per-stage barrier round trip and the epilogue): never AUTO.
        const double sms = 148.0;
        const double n2 = static_cast<double>(build_tiles(p->N, 64, 64).size()) * p->F;
        const double n1 = static_cast<double>(build_tiles(p->N, 32, 32).size()) * p->F;
        const double t_pair = std::ceil(n2 / (sms / 2)) * 2.0;
        const double t_solo = std::ceil(n1 / sms) * 1.25;
        mode = (t_solo < 0.8 * t_pair) ? XC_TILE_1CTA_128x128 : XC_TILE_2CTA_256x256;
    }
    int si, sj;
    tile_shape(mode, &si, &sj);
    p->tile_mode = mode;
    if (mode == XC_TILE_SPLIT || mode == XC_TILE_MIXED) {
        p->tiles_tc = build_tiles_off(p->N);
        p->tiles_diag = build_tiles_diag(p->N);
    } else {
        p->tiles_tc = build_tiles(p->N, si, sj);
        p->tiles_diag.clear();
    }
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
    int rc = upload_table(p, &p->d_tiles_tc, p->tiles_tc);
    if (rc != XC_OK) return rc;
    rc = upload_table(p, &p->d_tiles_diag, p->tiles_diag);
    if (rc != XC_OK) return rc;
    p->tiles_uploaded = true;
    return XC_OK;
}

template <int UMMA_N, int CG, bool STAGED, int BK = 128, bool DIAG = false>
int launch_tc(xc_plan_t* p, const xc::TcParams& tp, cudaStream_t st) {
    using Cfg = xc::TcCfg<UMMA_N, CG, STAGED, BK, DIAG>;
    long long units = (p->opt_max_ctas > 0 ? p->opt_max_ctas : p->sm_count) / CG;
    if (units < 1) units = 1;
    const long long groups = tp.total_tiles >> tp.group_shift;
    if (units > groups) units = groups;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(static_cast<unsigned>(units * CG));
    cfg.blockDim = dim3(xc::TC_THREADS);
    cfg.dynamicSmemBytes = Cfg::SMEM_BYTES;
    cfg.stream = st;
    cudaLaunchAttribute attr[2];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = CG;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    // programmatic dependent launch: this kernel's prologue may overlap the previous kernel's tail (it executes
    // griddepcontrol.wait before its first global access)
    attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[1].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = p->opt_pdl ? 2 : 1;
    auto kern = xc::xc_i8_tc_kernel<UMMA_N, CG, STAGED, false, BK, DIAG>;
    if (CG == 2 && UMMA_N == 256 && BK == 128 && tp.trace)
        kern = xc::xc_i8_tc_kernel<UMMA_N, CG, STAGED, (CG == 2 && UMMA_N == 256 && BK == 128), BK, DIAG>;
    // the shared-memory opt-in is per function and per device: set once per (kernel variant, device), not per call
    static int attr_done_dev[2] = {-1, -1};
    int& done = attr_done_dev[tp.trace ? 1 : 0];
    if (done != p->device) {
        XC_CUDA(p, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg::SMEM_BYTES));
        done = p->device;
    }
    XC_CUDA(p, cudaLaunchKernelEx(&cfg, kern, p->tmap, tp));
    p->last_launches += 1;
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
    p->sm_count = sms;
    p->tiles_uploaded = false;
    int rc_up = upload_tiles(p);
    if (rc_up != XC_OK) return rc_up;
    XC_CUDA(p, cudaMalloc(&p->d_tiles_f32, p->tiles_f32.size() * sizeof(uint32_t)));
    XC_CUDA(p, cudaMemcpy(p->d_tiles_f32, p->tiles_f32.data(), p->tiles_f32.size() * sizeof(uint32_t),
                          cudaMemcpyHostToDevice));
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
    p->dev_ready = true;
    return XC_OK;
}

// S0: decide whether the padding kernel is needed and run it; *src / *nrow describe what TMA reads.
int stage_if_needed(xc_plan_t* p, const int8_t* in_dev, cudaStream_t st, const void** src, int* nrow, int fmt_i4 = 0,
                    int f0 = 0, int nf = -1) {
    if (nf < 0) nf = p->F;
    const bool need = fmt_i4 || p->opt_force_stage || (p->Npad != p->N) || (reinterpret_cast<uintptr_t>(in_dev) & 15u);
    if (!need) {
        *src = in_dev;
        *nrow = p->N;
        return XC_OK;
    }
    const size_t want = xc_workspace_bytes(p);
    if (!p->ws) {
        XC_CUDA(p, cudaMalloc(&p->ws, want));  // synchronising; documented in xc.h
        p->ws_bytes = want;
        p->ws_owned = true;
    }
    if (p->ws_bytes < want) return XC_ERR_NO_WORKSPACE;
    const long long rows = static_cast<long long>(p->T) * p->F;
    const long long total = rows * p->Npad;
    long long blocks = (total + 255) / 256;
    if (blocks > 148LL * 32) blocks = 148LL * 32;
    if (fmt_i4) {
        // 4-bit samples: the staging pass is the unpacking pass (in_dev then points at 2*N*F*T packed bytes)
        const long long units = static_cast<long long>(p->T) * nf * p->Npad;
        if (p->N % 8 == 0 && !(reinterpret_cast<uintptr_t>(in_dev) & 15u)) {
            long long b16 = (units / 8 + 255) / 256;
            if (b16 > 148LL * 32) b16 = 148LL * 32;
            xc::xc_unpack_i4x8_kernel<<<static_cast<unsigned>(b16 < 1 ? 1 : b16), 256, 0, st>>>(
                reinterpret_cast<const uint4*>(in_dev), static_cast<uint4*>(p->ws), p->T, p->F, f0, nf, p->N / 8);
        } else {
            long long b1 = (units + 255) / 256;
            if (b1 > 148LL * 32) b1 = 148LL * 32;
            xc::xc_unpack_i4_kernel<<<static_cast<unsigned>(b1), 256, 0, st>>>(
                reinterpret_cast<const uint8_t*>(in_dev), static_cast<uint32_t*>(p->ws), p->T, p->F, f0, nf, p->N, p->Npad);
        }
    } else if (p->N % 4 == 0 && !(reinterpret_cast<uintptr_t>(in_dev) & 15u)) {
        xc::xc_stage_pad16_kernel<<<static_cast<unsigned>(blocks), 256, 0, st>>>(
            reinterpret_cast<const uint4*>(in_dev), static_cast<uint4*>(p->ws), rows, p->N / 4, p->Npad / 4);
    } else {
        xc::xc_stage_pad_kernel<<<static_cast<unsigned>(blocks), 256, 0, st>>>(in_dev, static_cast<uint32_t*>(p->ws), rows,
                                                                                 p->N, p->Npad);
    }
    XC_CUDA(p, cudaGetLastError());
    p->last_launches += 1;
    *src = p->ws;
    *nrow = p->Npad;
    return XC_OK;
}

// Tensor map over channels [.., nf) of the block that starts at src (the channel pitch stays the plan's F).
int encode_tmap(xc_plan_t* p, const void* src, int nrow, int bk, int nf) {
    if (p->tmap_src == src && p->tmap_nrow == nrow && p->tmap_bk == bk && p->tmap_nf == nf) return XC_OK;
    const cuuint64_t gdim[3] = {static_cast<cuuint64_t>(4) * nrow, static_cast<cuuint64_t>(nf),
                                static_cast<cuuint64_t>(p->T)};
    const cuuint64_t gstride[2] = {static_cast<cuuint64_t>(4) * nrow,
                                   static_cast<cuuint64_t>(4) * nrow * static_cast<cuuint64_t>(p->F)};
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
    p->tmap_nrow = nrow;
    p->tmap_bk = bk;
    p->tmap_nf = nf;
    return XC_OK;
}

// X-engine on channels [f0, f0 + nf) of the block at in_dev / the cube at vis_dev (both addressed with the plan's F).
int correlate_i8(xc_plan_t* p, const int8_t* in_dev, int32_t* vis_dev, void* stream, int accumulate, int f0 = 0,
                 int nf = -1, int fmt_i4 = 0) {
    if (!p || !in_dev || !vis_dev) return XC_ERR_INVALID_ARG;
    if (nf < 0) nf = p->F;
    if (f0 < 0 || nf < 1 || f0 + nf > p->F) return XC_ERR_INVALID_ARG;
    const bool sub = (f0 != 0 || nf != p->F);
    if (reinterpret_cast<uintptr_t>(vis_dev) & 15u) return XC_ERR_ALIGNMENT;
    int rc = ensure_device(p);
    if (rc != XC_OK) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    p->last_launches = 0;

    // a channel sub-range is read in place through its own tensor map: not with the SIMT kernel, not through staging
    const bool need_stage = fmt_i4 || p->opt_force_stage || (p->Npad != p->N) || (reinterpret_cast<uintptr_t>(in_dev) & 15u);
    if (sub && (p->opt_kernel == XC_I8_KERNEL_SIMT || (need_stage && !fmt_i4))) return XC_ERR_UNSUPPORTED;
    if (fmt_i4 && p->opt_kernel == XC_I8_KERNEL_SIMT) return XC_ERR_UNSUPPORTED;
    if (p->opt_kernel == XC_I8_KERNEL_SIMT) {
        if (p->F > 65535) return XC_ERR_UNSUPPORTED;
        xc::SimtParams sp{p->N, p->F, p->T, p->NB, in_dev, vis_dev, accumulate};
        const long long nb = (p->N + xc::SIMT_B - 1) / xc::SIMT_B;
        dim3 grid(static_cast<unsigned>(nb * (nb + 1) / 2), static_cast<unsigned>(p->F));
        xc::xc_i8_simt_kernel<<<grid, dim3(xc::SIMT_B, xc::SIMT_B), 0, st>>>(sp);
        XC_CUDA(p, cudaGetLastError());
        p->last_launches += 1;
        return XC_OK;
    }

    const void* src = nullptr;
    int nrow = 0;
    rc = stage_if_needed(p, in_dev, st, &src, &nrow, fmt_i4, f0, nf);
    if (rc != XC_OK) return rc;
    const bool bkopt = p->tile_mode == XC_TILE_2CTA_256x256 && p->opt_epilogue != XC_EPI_STAGED;
    const bool bk256 = bkopt && p->opt_bk == 256, bk64 = bkopt && p->opt_bk == 64;
    const bool solo128_bk256 = p->tile_mode == XC_TILE_1CTA_128x128 && p->opt_epilogue != XC_EPI_STAGED && p->opt_bk != 128;
    const int bk = (bk256 || solo128_bk256) ? 256 : (bk64 ? 64 : 128);
    rc = encode_tmap(p, static_cast<const int8_t*>(src) + static_cast<size_t>(4) * nrow * f0, nrow, bk, nf);
    if (rc != XC_OK) return rc;

    rc = upload_tiles(p);
    if (rc != XC_OK) return rc;
    xc::TcParams tp;
    tp.N = p->N;
    tp.F = nf;
    tp.T = p->T;
    tp.NB = p->NB;
    tp.vis = vis_dev + static_cast<size_t>(f0) * p->NB * 8;
    tp.accumulate = accumulate;
    tp.debug_skip = p->opt_debug_skip;
    tp.trace = p->trace;
    auto set_table = [&](const std::vector<uint32_t>& host, const uint32_t* dev, int group_shift) {
        tp.tiles_per_f = static_cast<int>(host.size());
        tp.tiles = dev;
        tp.group_shift = group_shift;
        if (static_cast<long long>(nf) * tp.tiles_per_f > 0x7FFFFFFFLL) return false;
        tp.total_tiles = nf * tp.tiles_per_f;
        return true;
    };
    const bool staged = p->opt_epilogue == XC_EPI_STAGED;   // AUTO = direct stores (measured faster)
    if (p->tile_mode == XC_TILE_MIXED) {
        // one launch, clusters of 2: some clusters are two single-CTA diagonal workers, the others are CTA pairs
        xc::TcParams td = tp;
        if (!set_table(p->tiles_diag, p->d_tiles_diag, 1)) return XC_ERR_UNSUPPORTED;
        td = tp;
        xc::TcParams to = tp;
        to.total_tiles = 0;
        if (!p->tiles_tc.empty()) {
            if (!set_table(p->tiles_tc, p->d_tiles_tc, 0)) return XC_ERR_UNSUPPORTED;
            to = tp;
        }
        int clusters = (p->opt_max_ctas > 0 ? p->opt_max_ctas : p->sm_count) / 2;
        if (clusters < 2) clusters = 2;
        const int n_solo = p->tiles_tc.empty() ? clusters : mixed_split(p->N, nf, clusters, nullptr);
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(static_cast<unsigned>(2 * clusters));
        cfg.blockDim = dim3(xc::TC_THREADS);
        cfg.dynamicSmemBytes = xc::TcCfg<256, 2, false, 128, false>::SMEM_BYTES;
        static_assert(xc::TcCfg<256, 2, false, 128, false>::SMEM_BYTES == xc::TcCfg<256, 1, false, 128, true>::SMEM_BYTES,
                      "both worker kinds of the mixed kernel use the same ring");
        cfg.stream = st;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = 2;
        attr[0].val.clusterDim.y = 1;
        attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        XC_CUDA(p, cudaFuncSetAttribute(xc::xc_i8_tc_mixed_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                        static_cast<int>(cfg.dynamicSmemBytes)));
        XC_CUDA(p, cudaLaunchKernelEx(&cfg, xc::xc_i8_tc_mixed_kernel, p->tmap, td, to, n_solo));
        p->last_launches += 1;
        return XC_OK;
    }
    if (p->tile_mode == XC_TILE_SPLIT) {
        // two launches with disjoint outputs: diagonal 64-station blocks on single CTAs, the rest on CTA pairs
        if (!set_table(p->tiles_diag, p->d_tiles_diag, 1)) return XC_ERR_UNSUPPORTED;
        rc = launch_tc<256, 1, false, 128, true>(p, tp, st);
        if (rc != XC_OK) return rc;
        if (!p->tiles_tc.empty()) {
            if (!set_table(p->tiles_tc, p->d_tiles_tc, 0)) return XC_ERR_UNSUPPORTED;
            rc = staged ? launch_tc<256, 2, true>(p, tp, st) : launch_tc<256, 2, false>(p, tp, st);
        }
        return rc;
    }
    if (!set_table(p->tiles_tc, p->d_tiles_tc, 0)) return XC_ERR_UNSUPPORTED;
    if (p->tile_mode == XC_TILE_2CTA_256x256)
        rc = staged ? launch_tc<256, 2, true>(p, tp, st)
                    : (bk256 ? launch_tc<256, 2, false, 256>(p, tp, st)
                             : (bk64 ? launch_tc<256, 2, false, 64>(p, tp, st) : launch_tc<256, 2, false>(p, tp, st)));
    else if (p->tile_mode == XC_TILE_1CTA_128x256)
        rc = staged ? launch_tc<256, 1, true>(p, tp, st) : launch_tc<256, 1, false>(p, tp, st);
    else
        rc = staged ? launch_tc<128, 1, true>(p, tp, st)
                    : (solo128_bk256 ? launch_tc<128, 1, false, 256>(p, tp, st) : launch_tc<128, 1, false>(p, tp, st));
    return rc;
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
    if (!p) return XC_ERR_INVALID_ARG;
    p->N = N;
    p->P = P;
    p->F = F;
    p->T = T;
    p->NB = static_cast<long long>(N) * (N + 1) / 2;
    // Row pitch seen by TMA: a multiple of 16 bytes is mandatory (N % 4 == 0).  A pitch that is not a multiple of 128
    // bytes makes every box row straddle two 128-byte lines; re-pitching such inputs with the staging kernel was worth
    // 5 % in an early version of the kernel and costs 6 % today (N = 500: 276 us staged, 259 us direct), so rows are
    // only ever padded to the mandatory 16 bytes.
    p->Npad = (N + 3) & ~3;
    set_tile_mode(p, XC_TILE_AUTO);
    p->tiles_f32 = build_tiles(N, xc::F32_SI, xc::F32_SJ);
    memset(&p->tmap, 0, sizeof p->tmap);
    *out = p;
    return XC_OK;
}

void xc_destroy(xc_plan_t* p) {
    if (!p) return;
    if (p->d_tiles_tc) cudaFree(p->d_tiles_tc);
    if (p->d_tiles_diag) cudaFree(p->d_tiles_diag);
    if (p->d_tiles_f32) cudaFree(p->d_tiles_f32);
    if (p->ws && p->ws_owned) cudaFree(p->ws);
    for (int k = 0; k < 2; ++k) {
        if (p->ev_copied[k]) cudaEventDestroy(p->ev_copied[k]);
        if (p->ev_free[k]) cudaEventDestroy(p->ev_free[k]);
    }
    if (p->ev_entry) cudaEventDestroy(p->ev_entry);
    for (cudaEvent_t e : p->ev_chunk) cudaEventDestroy(e);
    if (p->s_h2d) cudaStreamDestroy(p->s_h2d);
    if (p->s_d2h) cudaStreamDestroy(p->s_d2h);
    delete p;
}

size_t xc_in_bytes(const xc_plan_t* p) { return p ? static_cast<size_t>(4) * p->N * p->F * p->T : 0; }
size_t xc_in_bytes_i4(const xc_plan_t* p) { return p ? static_cast<size_t>(2) * p->N * p->F * p->T : 0; }
size_t xc_in_bytes_f32(const xc_plan_t* p) { return p ? static_cast<size_t>(16) * p->N * p->F * p->T : 0; }
size_t xc_vis_bytes(const xc_plan_t* p) { return p ? static_cast<size_t>(32) * p->NB * p->F : 0; }
size_t xc_n_baselines(const xc_plan_t* p) { return p ? static_cast<size_t>(p->NB) : 0; }
size_t xc_workspace_bytes(const xc_plan_t* p) { return p ? static_cast<size_t>(4) * p->Npad * p->F * p->T : 0; }

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
            if (value < XC_TILE_AUTO || value > XC_TILE_MIXED) return XC_ERR_INVALID_ARG;
            set_tile_mode(p, value);
            return XC_OK;
        case XC_OPT_BK:
            if (value != 0 && value != 64 && value != 128 && value != 256) return XC_ERR_INVALID_ARG;
            p->opt_bk = value;
            return XC_OK;
        case XC_OPT_EPILOGUE:
            if (value < XC_EPI_AUTO || value > XC_EPI_STAGED) return XC_ERR_INVALID_ARG;
            p->opt_epilogue = value;
            return XC_OK;
        case XC_OPT_PDL:
            p->opt_pdl = value ? 1 : 0;
            return XC_OK;
        case XC_OPT_DEBUG_SKIP:
            p->opt_debug_skip = value & 15;
            return XC_OK;
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

int xc_correlate_pipelined(xc_plan_t* p, const int8_t* in_host, int n_blocks, int8_t* dev_buf2, int32_t* vis_dev,
                           void* compute_stream, void* copy_stream) {
    if (!p || !in_host || !dev_buf2 || !vis_dev || n_blocks < 1) return XC_ERR_INVALID_ARG;
    if (reinterpret_cast<uintptr_t>(dev_buf2) & 127u) return XC_ERR_ALIGNMENT;
    int rc = ensure_device(p);
    if (rc != XC_OK) return rc;
    cudaStream_t cs = static_cast<cudaStream_t>(compute_stream), xs = static_cast<cudaStream_t>(copy_stream);
    for (int k = 0; k < 2; ++k) {
        if (!p->ev_copied[k]) XC_CUDA(p, cudaEventCreateWithFlags(&p->ev_copied[k], cudaEventDisableTiming));
        if (!p->ev_free[k]) XC_CUDA(p, cudaEventCreateWithFlags(&p->ev_free[k], cudaEventDisableTiming));
    }
    if (!p->ev_entry) XC_CUDA(p, cudaEventCreateWithFlags(&p->ev_entry, cudaEventDisableTiming));
    const size_t blk = xc_in_bytes(p);
    const size_t half = blk;  // a half that ends up not 16-byte aligned simply goes through staging (S0)
    int launches = 0;
    // Earlier work on the compute stream may still read dev_buf2: copies start after it.
    XC_CUDA(p, cudaEventRecord(p->ev_entry, cs));
    XC_CUDA(p, cudaStreamWaitEvent(xs, p->ev_entry, 0));
    XC_CUDA(p, cudaMemcpyAsync(dev_buf2, in_host, blk, cudaMemcpyHostToDevice, xs));
    XC_CUDA(p, cudaEventRecord(p->ev_copied[0], xs));
    for (int b = 0; b < n_blocks; ++b) {
        if (b + 1 < n_blocks) {
            const int nb = (b + 1) & 1;
            if (b >= 1) XC_CUDA(p, cudaStreamWaitEvent(xs, p->ev_free[nb], 0));  // X-engine on block b-1 is done with it
            XC_CUDA(p, cudaMemcpyAsync(dev_buf2 + nb * half, in_host + static_cast<size_t>(b + 1) * blk, blk,
                                       cudaMemcpyHostToDevice, xs));
            XC_CUDA(p, cudaEventRecord(p->ev_copied[nb], xs));
        }
        XC_CUDA(p, cudaStreamWaitEvent(cs, p->ev_copied[b & 1], 0));
        rc = correlate_i8(p, dev_buf2 + (b & 1) * half, vis_dev, compute_stream, b > 0 ? 1 : 0);
        if (rc != XC_OK) return rc;
        launches += p->last_launches;
        XC_CUDA(p, cudaEventRecord(p->ev_free[b & 1], cs));
    }
    p->last_launches = launches;
    return XC_OK;
}

int xc_integrate(xc_plan_t* p, const int8_t* in_host, int n_blocks, int8_t* dev_buf2, int32_t* vis32_dev,
                 int64_t* vis64_dev, int64_t* vis64_host, void* compute_stream, void* copy_stream) {
    if (!p || !in_host || !dev_buf2 || !vis32_dev || !vis64_dev || n_blocks < 1) return XC_ERR_INVALID_ARG;
    if ((reinterpret_cast<uintptr_t>(dev_buf2) & 127u) || (reinterpret_cast<uintptr_t>(vis64_dev) & 15u)) return XC_ERR_ALIGNMENT;
    int rc = ensure_device(p);
    if (rc != XC_OK) return rc;
    cudaStream_t cs = static_cast<cudaStream_t>(compute_stream), xs = static_cast<cudaStream_t>(copy_stream);
    for (int k = 0; k < 2; ++k) {
        if (!p->ev_copied[k]) XC_CUDA(p, cudaEventCreateWithFlags(&p->ev_copied[k], cudaEventDisableTiming));
        if (!p->ev_free[k]) XC_CUDA(p, cudaEventCreateWithFlags(&p->ev_free[k], cudaEventDisableTiming));
    }
    if (!p->ev_entry) XC_CUDA(p, cudaEventCreateWithFlags(&p->ev_entry, cudaEventDisableTiming));
    const size_t blk = xc_in_bytes(p);
    const int group = XC_MAX_T / p->T;              // blocks whose int32 partial sum cannot overflow (>= 1)
    const long long n4 = static_cast<long long>(p->F) * p->NB * 2;   // int4 quadruples in the cube
    long long wblocks = (n4 + 255) / 256;
    if (wblocks > 148LL * 16) wblocks = 148LL * 16;
    int launches = 0;
    XC_CUDA(p, cudaEventRecord(p->ev_entry, cs));
    XC_CUDA(p, cudaStreamWaitEvent(xs, p->ev_entry, 0));
    XC_CUDA(p, cudaMemcpyAsync(dev_buf2, in_host, blk, cudaMemcpyHostToDevice, xs));
    XC_CUDA(p, cudaEventRecord(p->ev_copied[0], xs));
    for (int b = 0; b < n_blocks; ++b) {
        if (b + 1 < n_blocks) {
            const int nb = (b + 1) & 1;
            if (b >= 1) XC_CUDA(p, cudaStreamWaitEvent(xs, p->ev_free[nb], 0));
            XC_CUDA(p, cudaMemcpyAsync(dev_buf2 + nb * blk, in_host + static_cast<size_t>(b + 1) * blk, blk,
                                       cudaMemcpyHostToDevice, xs));
            XC_CUDA(p, cudaEventRecord(p->ev_copied[nb], xs));
        }
        XC_CUDA(p, cudaStreamWaitEvent(cs, p->ev_copied[b & 1], 0));
        rc = correlate_i8(p, dev_buf2 + (b & 1) * blk, vis32_dev, compute_stream, (b % group) ? 1 : 0);
        if (rc != XC_OK) return rc;
        launches += p->last_launches;
        XC_CUDA(p, cudaEventRecord(p->ev_free[b & 1], cs));
        if ((b + 1) % group == 0 || b + 1 == n_blocks) {
            xc::xc_widen_kernel<<<static_cast<unsigned>(wblocks), 256, 0, cs>>>(
                reinterpret_cast<const int4*>(vis32_dev), reinterpret_cast<longlong2*>(vis64_dev), n4, b < group ? 1 : 0);
            XC_CUDA(p, cudaGetLastError());
            launches += 1;
        }
    }
    if (vis64_host)
        XC_CUDA(p, cudaMemcpyAsync(vis64_host, vis64_dev, 2 * xc_vis_bytes(p), cudaMemcpyDeviceToHost, cs));
    p->last_launches = launches;
    return XC_OK;
}

int xc_correlate_channels(xc_plan_t* p, const int8_t* in_dev, int32_t* vis_dev, int f0, int nf, int accumulate,
                          void* stream) {
    return correlate_i8(p, in_dev, vis_dev, stream, accumulate ? 1 : 0, f0, nf);
}

static int correlate_host_impl(xc_plan_t* p, const int8_t* in_host, int32_t* vis_host, int8_t* in_dev_scratch,
                               int32_t* vis_dev_scratch, void* stream, int fmt_i4) {
    if (!p || !in_host || !vis_host || !in_dev_scratch || !vis_dev_scratch) return XC_ERR_INVALID_ARG;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    int rc = ensure_device(p);
    if (rc != XC_OK) return rc;
    // int8 blocks that need the staging pass work on whole blocks only; 4-bit blocks are unpacked range by range
    const bool need_stage = !fmt_i4 && (p->opt_force_stage || (p->Npad != p->N) || (reinterpret_cast<uintptr_t>(in_dev_scratch) & 15u));
    const size_t in_bytes = fmt_i4 ? xc_in_bytes_i4(p) : xc_in_bytes(p);
    int chunks = p->F < 16 ? p->F : 16;
    if (need_stage || p->opt_kernel == XC_I8_KERNEL_SIMT || in_bytes < (static_cast<size_t>(8) << 20)) chunks = 1;
    if (chunks == 1) {
        XC_CUDA(p, cudaMemcpyAsync(in_dev_scratch, in_host, in_bytes, cudaMemcpyHostToDevice, st));
        rc = correlate_i8(p, in_dev_scratch, vis_dev_scratch, stream, 0, 0, -1, fmt_i4);
        if (rc != XC_OK) return rc;
        XC_CUDA(p, cudaMemcpyAsync(vis_host, vis_dev_scratch, xc_vis_bytes(p), cudaMemcpyDeviceToHost, st));
        XC_CUDA(p, cudaStreamSynchronize(st));
        return XC_OK;
    }
    // Channels are independent, so the block is cut into channel ranges and the three legs of the
    // paper's integrated run (host->device, X-engine, device->host: Fig. 7) overlap: range c+1 is
    // copied in (a strided 2-D copy: T rows of the range's bytes) while range c is correlated and range c-1 is
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
    const size_t row = static_cast<size_t>(fmt_i4 ? 2 : 4) * p->N;    // bytes of one (t, f) row
    const size_t pitch = row * p->F;
    int launches = 0;
    for (int c = 0; c < chunks; ++c) {
        const int f0 = static_cast<int>(static_cast<long long>(p->F) * c / chunks);
        const int f1 = static_cast<int>(static_cast<long long>(p->F) * (c + 1) / chunks);
        XC_CUDA(p, cudaMemcpy2DAsync(in_dev_scratch + row * f0, pitch, in_host + row * f0, pitch, row * (f1 - f0),
                                     static_cast<size_t>(p->T), cudaMemcpyHostToDevice, p->s_h2d));
        XC_CUDA(p, cudaEventRecord(p->ev_chunk[2 * c], p->s_h2d));
        XC_CUDA(p, cudaStreamWaitEvent(st, p->ev_chunk[2 * c], 0));
        rc = correlate_i8(p, in_dev_scratch, vis_dev_scratch, stream, 0, f0, f1 - f0, fmt_i4);
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
    p->last_launches = launches;
    return XC_OK;
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

int xc_debug_set_trace(xc_plan_t* p, void* trace_dev) {
    if (!p) return XC_ERR_INVALID_ARG;
    p->trace = static_cast<long long*>(trace_dev);
    return XC_OK;
}

int xc_tile_count(const xc_plan_t* p) {
    if (!p) return 0;
    int n = static_cast<int>(p->tiles_tc.size());
    for (uint32_t e : p->tiles_diag) n += (e != 0xFFFFFFFFu);
    return n;
}

int xc_tile_get(const xc_plan_t* p, int k, int* bi, int* bj, int* si, int* sj) {
    if (!p || k < 0) return XC_ERR_INVALID_ARG;
    uint32_t e = 0;
    int a = 0, b = 0;
    bool found = false;
    for (uint32_t d : p->tiles_diag) {          // XC_TILE_SPLIT: diagonal sub-tiles first (32 x 64 stations each)
        if (d == 0xFFFFFFFFu) continue;
        if (k-- == 0) { e = d; a = 32; b = 64; found = true; break; }
    }
    if (!found) {
        if (k >= static_cast<int>(p->tiles_tc.size())) return XC_ERR_INVALID_ARG;
        e = p->tiles_tc[k];
        tile_shape(p->tile_mode, &a, &b);
    }
    if (bi) *bi = static_cast<int>(e & 0xFFFFu);
    if (bj) *bj = static_cast<int>(e >> 16);
    if (si) *si = a;
    if (sj) *sj = b;
    return XC_OK;
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
        default: return "XC_ERR_UNKNOWN";
    }
}

const char* xc_last_cuda_error(const xc_plan_t* p) { return p ? p->last_err.c_str() : ""; }

const char* xc_version(void) { return "xcorr-b200 0.1 (sm_100a, tcgen05 kind::i8)"; }

}  // extern "C"
