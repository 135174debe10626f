/*
 * xc.h -- C ABI of the B200-native X-engine (radio-astronomy cross-correlator).
 *
 * Operation (Sec. 2.1, Eq. 4): for every frequency channel f, the
 * time-integrated self outer product of the complex sample vector of N stations x 2
 * polarisations,
 *
 *      V_f[(i,pi),(j,pj)] = sum_{t<T}  x_{t,f,i,pi} * conj(x_{t,f,j,pj})
 *
 * kept for the lower-triangle station pairs 0 <= i <= j < N ("1/2 N(N+1) correlation
 * pairs including the auto-correlation of self pairs"), all four
 * polarisation products per pair.
 *
 * Layouts (BASELINE.json north_star; input order = PAPER.md:149 "station fastest, then
 * frequency, then time", i.e. the corner turn is already applied):
 *
 *   in  : [t][f][station][pol][re,im]      flat ((((t*F + f)*N + s)*2 + p)*2 + c)
 *         int8 for the integer path, float for the fp32 path
 *   vis : [f][b][pol_i][pol_j][re,im]      flat ((((f*NB + b)*2 + pi)*2 + pj)*2 + c)
 *         b = j(j+1)/2 + i  (the paper's triangular block order, applied at
 *         station level),  NB = N(N+1)/2;  int32 for the integer path, float for fp32
 *
 * Every *_dev pointer is DEVICE memory owned by the caller (allocate it with PyTorch);
 * every *_host pointer is HOST memory owned by the caller.  The library never frees or
 * retains caller memory beyond the call (except the workspace handed to
 * xc_set_workspace, which it uses until the plan is destroyed or the workspace replaced).
 * Streams are cudaStream_t passed as void*; all device work is enqueued on the stream
 * given, asynchronously, with no hidden device synchronisation unless stated (the one
 * exception that uses streams of its own, xc_correlate_host, says so).  The tensor-core
 * kernels are launched with programmatic stream serialization (XC_OPT_PDL): they wait for
 * the preceding kernel of the stream before their first global access, so stream order is
 * kept; calls can be captured into CUDA graphs once the plan has made one compute call.
 *
 * A plan binds to the CUDA device that is current at its first compute call (its tile table, workspace and helper
 * streams live there; later calls with another device current return XC_ERR_INVALID_ARG).  A plan is not thread-safe:
 * calls on one plan must not overlap in time on the host; different plans are independent.
 *
 * Every function returns an xc_status (0 = OK, negative = error); nothing is thrown
 * across this boundary; on error no output is promised.  There is no CPU fallback: on a
 * machine without an sm_100 GPU every compute entry point returns XC_ERR_CUDA /
 * XC_ERR_UNSUPPORTED.
 */
#ifndef XC_H_
#define XC_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct xc_plan_s xc_plan_t; /* opaque; created by xc_plan, freed by xc_destroy */

typedef enum {
    XC_OK = 0,
    XC_ERR_INVALID_ARG = -1,  /* null pointer, N/F/T < 1, bad option ...                      */
    XC_ERR_UNSUPPORTED = -2,  /* P != 2, unknown layout, device is not sm_100                  */
    XC_ERR_OVERFLOW = -3,     /* T > XC_MAX_T: one call could leave int32 (2*128^2*T >= 2^31)  */
    XC_ERR_ALIGNMENT = -4,    /* pointer alignment not met and no staging workspace available  */
    XC_ERR_CUDA = -5,         /* a CUDA call failed; see xc_last_cuda_error                    */
    XC_ERR_NO_WORKSPACE = -6, /* staging needed but workspace too small                        */
    XC_ERR_NO_MEMORY = -7     /* host memory for the plan could not be allocated               */
} xc_status;

typedef enum {
    XC_LAYOUT_TFSPC = 0 /* [t][f][station][pol][re,im] -- PAPER.md:149; the only layout */
} xc_layout;

/* Largest T of one integer call: |V| <= 2 * 128^2 * T must stay < 2^31 ("a larger number of
 * bits used for the accumulator to prevent overflow"). Across xc_correlate_acc
 * calls the caller owns the bound. */
#define XC_MAX_T 65535

/* Kernel choice for the integer path (xc_set_option(XC_OPT_I8_KERNEL, ...)). */
enum {
    XC_I8_KERNEL_AUTO = 0, /* tcgen05 tensor-core kernel (the product path)                   */
    XC_I8_KERNEL_TC = 1,   /* same, forced                                                    */
    XC_I8_KERNEL_SIMT = 2  /* plain CUDA-core kernel, one thread per baseline: a debugging    */
                           /* aid that shares no device code with the tensor-core kernel     */
};
/* Kernels of the fp32 path, xc_set_option(XC_OPT_F32_KERNEL, ...). */
enum {
    XC_F32_KERNEL_AUTO = 0,       /* = XC_F32_KERNEL_TC (measured faster at every N)                                 */
    XC_F32_KERNEL_CUDA_CORES = 1, /* the paper's own scheme: register tile of station pairs per thread, packed FMAs  */
    XC_F32_KERNEL_TC = 2          /* tcgen05 kind::tf32, every product from three TF32 MMAs (hi/lo split), fp32 sums */
};
/* Tensor-core tile shapes (Gram rows x Gram columns; 4 Gram rows = 1 station), xc_set_option(XC_OPT_TILE, ...).
 * Round 1 also built 128x256 single-CTA tiles, a staged (bulk-store) epilogue, 64/256-sample stages and two
 * diagonal-specialised schedules (SPLIT, MIXED); all measured slower than these two and were removed. */
enum {
    XC_TILE_AUTO = 0,         /* chosen from N, F and the SM count                                 */
    XC_TILE_1CTA_128x128 = 1, /* 32 x 32 stations on one CTA (small N)                             */
    XC_TILE_2CTA_256x256 = 3  /* 64 x 64 stations on a CTA pair (tcgen05 cta_group::2)             */
};
typedef enum {
    XC_OPT_I8_KERNEL = 0,     /* one of XC_I8_KERNEL_*                                                                       */
    XC_OPT_MAX_CTAS = 1,      /* cap on persistent CTAs of the tensor-core kernel (0 = SM count)                             */
    XC_OPT_FORCE_STAGE = 2,   /* 1 = always run the staging (re-pitch/copy) kernel, for testing S0                           */
    /* 3 = XC_OPT_DEBUG_SKIP (profiling build only, below); 5 and 6 were round 1's epilogue and schedule choices (staged     */
    /* bulk-store epilogue, SPLIT/MIXED diagonal schedules): measured slower, removed, ids retired -> XC_ERR_INVALID_ARG     */
    XC_OPT_TILE = 4,          /* one of XC_TILE_*; rebuilds the tile schedule (synchronising on next call)                   */
    XC_OPT_PDL = 7,           /* 1 (default) = launch the tensor-core kernels with programmatic stream serialization: the    */
                              /* prologue overlaps the previous kernel's tail; 0 = plain launch                              */
    XC_OPT_TSPLIT = 8,        /* T-split of the single-CTA tile over a cluster of 2 (the paper's small-N future work,        */
                              /* PAPER.md:311-313): 0 = auto (on when 2 * tiles * F <= SM count and T >= 8192: the hand-over */
                              /* costs ~3 us), 1 = off, 2 = on whenever T allows it.  Same bits either way.                  */
    XC_OPT_ORIGIN_SHIFT = 9,  /* 1 (default) = when the rows of the block are not 128 bytes apart (dense N % 32 != 0) but    */
                              /* row pitch x F is, move every channel's tile grid left by the offset of its rows inside      */
                              /* their 128-byte line, so that TMA fetches whole lines ("rows aligned to    */
                              /* the memory line"); 0 = off (for comparison).  Same bits either way.                         */
    XC_OPT_F32_KERNEL = 10    /* one of XC_F32_KERNEL_* (xc_correlate_f32)                                                   */
#ifdef XC_PROFILE
    , XC_OPT_DEBUG_SKIP = 3   /* PROFILING BUILD ONLY (-DXC_PROFILE), results become meaningless: bit 0 = no TMA loads after */
                              /* the first ring fill, bit 1 = no MMAs, bit 2 = no stores, bit 3 = all stores wrapped into    */
                              /* an 8 MB window                                                                              */
#endif
} xc_option;

/* xc_plan -- north_star's xc_plan(N, P=2, F, T, layout).
 *   N stations (>=1), P polarisations (must be 2), F channels (>=1), T samples per call
 *   (1..XC_MAX_T), layout = XC_LAYOUT_TFSPC.  Builds the triangular tile schedule
 *   (only tiles that intersect i <= j are scheduled) and uploads it to the
 *   current CUDA device (plan-owned, a few KB).  *out receives the plan.
 *   Errors: INVALID_ARG, UNSUPPORTED, OVERFLOW, NO_MEMORY, CUDA. */
int xc_plan(xc_plan_t** out, int N, int P, int F, int T, int layout);

/* Frees the plan and the device memory it owns (tile table, and a staging workspace only if
 * the library allocated it itself).  NULL is allowed. */
void xc_destroy(xc_plan_t* plan);

/* Sizes in bytes of one input block / one output cube for this plan. */
size_t xc_in_bytes(const xc_plan_t* plan);      /* int8 path, one DEVICE block: xc_in_pitch()*F*T = 4*N*F*T unless xc_set_in_pitch was called; host blocks are always 4*N*F*T */
size_t xc_in_bytes_f32(const xc_plan_t* plan);  /* fp32 path, one device block: xc_in_pitch_f32()*F*T = 16*N*F*T unless xc_set_in_pitch_f32 was called */
size_t xc_in_bytes_i4(const xc_plan_t* plan);   /* 4-bit path: 2*N*F*T            */
size_t xc_vis_bytes(const xc_plan_t* plan);     /* 32*NB*F (int32 and float alike) */
/* N(N+1)/2. */
size_t xc_n_baselines(const xc_plan_t* plan);

/* Row pitch of device input blocks (the paper's coalescing rule -- rows aligned to the memory
 * line -- is, for TMA, a row pitch that is a multiple of 128 bytes).  By default an input block is dense: the rows
 * (t, f) of 4N bytes follow each other (pitch 4N).  xc_set_in_pitch declares that the in_dev blocks handed to
 * xc_correlate / _acc / _channels have their rows row_pitch_bytes apart (>= 4N; bytes beyond 4N of a row are ignored;
 * 0 restores the dense default).  A producer that is free to choose (the F-engine below, a capture card) should use
 * xc_scratch_pitch(): with N = 500 the X-engine then runs at the speed of N = 512 instead of ~25 % slower.
 * xc_in_pitch returns the current value. */
int xc_set_in_pitch(xc_plan_t* plan, size_t row_pitch_bytes);
size_t xc_in_pitch(const xc_plan_t* plan);
/* The same for float blocks (xc_correlate_f32 / _f32_channels): rows of 16N bytes, row_pitch_bytes apart (a multiple of 16,
 * >= 16N; 0 restores the dense default).  With N % 8 != 0 dense float rows straddle 128-byte lines exactly as dense int8
 * rows with N % 32 != 0 do; a producer that can choose should pad the rows to a multiple of 128 bytes.  Tensor-core kernel
 * only: with XC_F32_KERNEL_CUDA_CORES selected a pitched plan answers XC_ERR_UNSUPPORTED. */
int xc_set_in_pitch_f32(xc_plan_t* plan, size_t row_pitch_bytes);
size_t xc_in_pitch_f32(const xc_plan_t* plan);
/* The library's own pitch, 4N rounded up to 128 bytes (the row pitch of the staging workspace, of the host-buffer
 * calls' device blocks and of the F-engine's cube), and the size of in_dev_scratch of xc_correlate_host / of each half
 * of dev_buf2 of xc_correlate_pipelined / xc_integrate: one block with that pitch, plus -- when 4N is not already a
 * multiple of 128 -- a dense landing area for the host->device copy (a small kernel spreads the rows: the copy engine
 * moves dense blocks at the full PCIe rate, pitched 2000-byte rows at a quarter of it). */
size_t xc_scratch_pitch(const xc_plan_t* plan);
size_t xc_scratch_in_bytes(const xc_plan_t* plan);

/* Staging.  The tensor-core kernel reads the input through TMA, which
 * needs a 16-byte-aligned base and a 16-byte-multiple row pitch (dense rows: N % 4 == 0).
 * Otherwise the input is first copied by a staging kernel into a workspace of
 * xc_workspace_bytes() = xc_scratch_pitch() * F * T bytes (the 4-bit path always unpacks into it; NOT xc_scratch_in_bytes(),
 * which adds the dense landing area of the host-buffer calls).  The caller may hand one
 * in (device memory, 128-byte aligned, kept until xc_destroy or replaced); if none was set the
 * library cudaMallocs one on first need (a synchronising call) and frees it in xc_destroy.  The workspace is
 * plan-wide: staged calls issued on different streams are ordered against each other by an event. */
size_t xc_workspace_bytes(const xc_plan_t* plan);
int xc_set_workspace(xc_plan_t* plan, void* ws_dev, size_t bytes);

/* Kernel timing without a profiler: stamps_dev = device buffer of 6 uint64 (or NULL to switch off).  Every CTA of the
 * tensor-core kernel then atomically folds the global nanosecond timer into [0] (min, at kernel entry) and [1] (max, at
 * exit) -- the caller presets [0] = UINT64_MAX and [1] = 0 before the launch (in stream order: while a timing buffer is set
 * the kernels are launched without programmatic serialization, so a preset enqueued before the call is complete when the
 * kernel's first stamp is taken), and [1] - [0] is the kernel's duration --
 * and CTA 0 writes (clock64, globaltimer) at its entry into [2], [3] and at its exit into [4], [5], from which the SM
 * clock the kernel really ran at follows.  Costs two atomics per CTA; nothing when off. */
int xc_set_timing_buffer(xc_plan_t* plan, uint64_t* stamps_dev);

int xc_set_option(xc_plan_t* plan, int option, int value);

/* xc_correlate -- vis = X-engine(in)  (Eq. 4).  Overwrites all F*NB*8 int32 of vis_dev; old
 *   contents are not read.  in_dev: int8 [T][F][N][2][2]; vis_dev: int32 [F][NB][2][2][2],
 *   16-byte aligned (32-byte alignment gives full-sector stores).  Exact for the whole
 *   int8 range including -128.  Bit-exact to the definition; independent of tile schedule.
 * xc_correlate_acc -- vis += X-engine(in)  ("matrix_d <- X-engine(matrix_d, buffer_d)",
 *   PAPER.md:244; I = N_p * I').  int32 two's-complement addition. */
int xc_correlate(xc_plan_t* plan, const int8_t* in_dev, int32_t* vis_dev, void* cuda_stream);
int xc_correlate_acc(xc_plan_t* plan, const int8_t* in_dev, int32_t* vis_dev, void* cuda_stream);

/* xc_correlate_i4 -- the same operation on 4-bit complex samples ("typically four to eight bits of precision is
 *   sufficient"; two's complement): halves the input bytes that cross PCIe / leave HBM.
 *   in4_dev: uint8 [T][F][N][2 pol], ONE byte per complex sample: low nibble = real part, high nibble = imaginary
 *   part, each a two's-complement integer in [-8, 7] (the paper fixes no packing; this is the library's format).
 *   A staging pass unpacks into the int8 workspace (xc_workspace_bytes(); see xc_set_workspace), then the tensor-core
 *   path runs as for int8 input; exact.  accumulate != 0 adds to vis_dev.  Errors as xc_correlate; UNSUPPORTED with
 *   the SIMT kernel selected. */
int xc_correlate_i4(xc_plan_t* plan, const uint8_t* in4_dev, int32_t* vis_dev, int accumulate, void* cuda_stream);

/* xc_correlate_i4_noalloc -- xc_correlate_i4 for callers that must not (or cannot) allocate device memory.
 *   Who: a real-time capture loop that cannot take cudaMalloc's device-wide stall in the middle of an observation; a
 *   plug-in whose host application owns every byte of device memory and forbids plug-ins to allocate; a process in which
 *   a framework's caching allocator or a memory pool has already taken the HBM that was left, so that an allocation by this
 *   library would fail.  xc_correlate_i4 needs an int8 workspace for its unpacking pass (the tensor-core kernel reads
 *   int8 through TMA) and a plan with small device tables; this call needs neither.  It takes the shape directly (no
 *   plan), keeps the tile table in the kernel parameters, and unpacks into a fixed array of XC_NOALLOC_SCRATCH_BYTES
 *   that is part of the library's device image: every GPU on which the library's image is loaded holds those 16 MiB until
 *   the process exits, whether or not this function is ever called.  The call itself issues no cudaMalloc, cudaFree,
 *   stream/event creation or other allocating CUDA routine, on its first use or later.
 *   Same operation, formats and result as xc_correlate_i4 (Eq. 4; 4-bit samples PAPER.md:45, 96):
 *   in4_dev: uint8 [T][F][N][2 pol] DEVICE memory, low nibble = real, high nibble = imaginary, two's complement;
 *   vis_dev: int32 [F][NB][2][2][2] DEVICE memory, 16-byte aligned, overwritten (accumulate == 0) or added to
 *   (accumulate != 0); both caller-owned.  Two launches (unpack, X-engine) on cuda_stream, asynchronous.
 *   Limits: N <= XC_NOALLOC_MAX_N (the tile table must fit the kernel parameters) and
 *   ((4N rounded up to 128) * F * T) <= XC_NOALLOC_SCRATCH_BYTES (the unpacked block must fit the array), T <= XC_MAX_T.
 *   Errors: INVALID_ARG (null pointer, N/F/T < 1), OVERFLOW (T > XC_MAX_T), UNSUPPORTED (N > XC_NOALLOC_MAX_N, device
 *   not sm_100), NO_WORKSPACE (the unpacked block is larger than XC_NOALLOC_SCRATCH_BYTES: use xc_correlate_i4 with
 *   xc_set_workspace, or cut the block in time and accumulate), ALIGNMENT (vis_dev), CUDA.  Nothing is launched on error.
 *   First call on a device: it looks up the array's device address (the array's name means nothing to a kernel when it
 *   comes from host code), the tensor-map encoder and the kernels' shared-memory opt-in, with that device current; make
 *   that first call outside any stream capture.  Later calls on that device only launch.
 *   Sharing: there is one array per device and every call on that device uses it, whatever its shape or stream.  Calls
 *   that may overlap on the GPU (different streams, no event between them) race on it and give garbage; calls on one
 *   stream, or ordered by events, are safe.  The array keeps the previous call's bytes; nothing has to be cleared by the
 *   caller: every byte a call's X-engine reads was written by that call's own unpacking pass (row bytes beyond 4N are never
 *   read: the tensor map ends there).  Host side: thread-safe. */
#define XC_NOALLOC_SCRATCH_BYTES (16u * 1024u * 1024u)
#define XC_NOALLOC_MAX_N 576
int xc_correlate_i4_noalloc(int N, int F, int T, const uint8_t* in4_dev, int32_t* vis_dev, int accumulate, void* cuda_stream);

/* xc_correlate_f32 -- same operation on float samples.  in_dev: float [T][F][N][2][2] (16-byte aligned; dense, or rows
 *   xc_in_pitch_f32() bytes apart after xc_set_in_pitch_f32);
 *   vis_dev: float [F][NB][2][2][2].  accumulate != 0 adds to vis_dev.  Two kernels (XC_OPT_F32_KERNEL):
 *   - CUDA cores: fp32 FMA arithmetic (the paper's own: PAPER.md:75, 16 FMAs per station pair per sample; warp-level
 *     register tiling as in PAPER.md:130-147).  One accumulator per output, ascending t: deterministic, about T * 2^-24
 *     relative to sqrt(V_ii V_jj) from an fp64 evaluation.
 *   - tensor cores (default): x x^H is a dense contraction; every sample is split into two TF32 numbers
 *     (hi = nearest TF32, lo = a - hi) and every product taken as lo hi + hi lo + hi hi into an fp32 accumulator.  The
 *     dropped parts are below 2^-21 of each product.  The tensor core's fp32 accumulator adds by truncation, so it only
 *     sums 128 samples at a time; the 128-sample partial sums are added in registers (round to nearest).  Deterministic
 *     (fixed schedule); error against an fp64 evaluation ~1e-6 sqrt(V_ii V_jj) whatever T is (tested up to T = 8192);
 *     integer-valued samples below 2^11 with sums below 2^24 give exact results.
 *     Precondition: finite samples with |a| < 2^127.  A sample at or above 0x7F7FF000 (3.4e38), an infinity or a NaN rounds to
 *     a non-finite hi part, lo = a - hi is then NaN, and every visibility of THAT STATION in that channel comes out NaN (the
 *     CUDA-core kernel gives Inf or NaN there by ordinary fp32 rules); visibilities of other stations are unaffected.
 *   Errors as xc_correlate. */
int xc_correlate_f32(xc_plan_t* plan, const float* in_dev, float* vis_dev, int accumulate, void* cuda_stream);

/* xc_correlate_f32_channels -- xc_correlate_f32 on channels [f0, f0 + nf) of the block: the float counterpart of
 *   xc_correlate_channels (channels are independent; one channel range per GPU or stream).
 *   in_dev and vis_dev are the WHOLE block and cube; only the range's visibilities are written.  A proper sub-range runs on
 *   the tensor-core kernel only (XC_ERR_UNSUPPORTED with XC_F32_KERNEL_CUDA_CORES selected). */
int xc_correlate_f32_channels(xc_plan_t* plan, const float* in_dev, float* vis_dev, int f0, int nf, int accumulate,
                              void* cuda_stream);

/* xc_correlate_pipelined -- Algorithm 1 read as textbook double
 *   buffering: n_blocks input blocks lie back to back in PINNED host memory at in_host, always DENSE, 4*N*F*T bytes
 *   each whatever xc_set_in_pitch says (xc_in_bytes() follows the device pitch: do not size host blocks with it); block p+1 is copied host->device on copy_stream into one half of
 *   dev_buf2 (2 * xc_scratch_in_bytes() bytes of device memory, 128-byte aligned) while block p is
 *   correlated on compute_stream from the other half; events order the two streams (no host
 *   synchronisation inside).  vis_dev = sum over blocks (first block overwrites).  The result
 *   stays on the device.  Returns after enqueueing; the caller synchronises
 *   compute_stream.  compute_stream and copy_stream must differ for any overlap to happen. */
int xc_correlate_pipelined(xc_plan_t* plan, const int8_t* in_host_pinned, int n_blocks, int8_t* dev_buf2,
                           int32_t* vis_dev, void* compute_stream, void* copy_stream);

/* xc_integrate -- long integration I = n_blocks * T ("I = N_p I'"; the integrated run of Sec. 6 / Fig. 7,
 *   PAPER.md:283): Algorithm 1 over n_blocks pinned host blocks as in xc_correlate_pipelined, with the int32 partial sums
 *   (exact for at most XC_MAX_T samples) added into an int64 cube after every floor(XC_MAX_T / T) blocks, so the result is
 *   exact for ANY integration length.  vis32_dev: scratch cube of xc_vis_bytes(); vis64_dev: int64 [F][NB][2][2][2]
 *   (2 * xc_vis_bytes(), 16-byte aligned), overwritten with the sum over all blocks; vis64_host: if not NULL the result is
 *   also copied there (the paper's "matrix_h <- matrix_d"), asynchronously on compute_stream.  Returns after
 *   enqueueing; the caller synchronises compute_stream. */
int xc_integrate(xc_plan_t* plan, const int8_t* in_host_pinned, int n_blocks, int8_t* dev_buf2, int32_t* vis32_dev,
                 int64_t* vis64_dev, int64_t* vis64_host, void* compute_stream, void* copy_stream);

/* xc_correlate_channels -- the same operation restricted to channels [f0, f0 + nf) of the plan's F ("evaluated
 *   independently for every frequency"; the paper's multi-GPU plan hands different channels to
 *   different devices).  in_dev / vis_dev are the FULL block and cube of the plan (the range is
 *   addressed inside them with the plan's F as channel pitch); only vis[f0 .. f0+nf) is written.  accumulate != 0
 *   adds.  Ranges of one block may run concurrently on different streams.  A block that needs the staging pass (N % 4
 *   != 0, misaligned pointer) is staged range by range: each call copies its own channels' rows into their place in the
 *   plan-wide workspace (calls on different streams are ordered against each other by the workspace event, so such ranges
 *   do not overlap on the GPU).  Errors: INVALID_ARG for a range outside [0, F); UNSUPPORTED with the SIMT kernel selected
 *   (whole blocks only). */
int xc_correlate_channels(xc_plan_t* plan, const int8_t* in_dev, int32_t* vis_dev, int f0, int nf, int accumulate,
                          void* cuda_stream);

/* xc_correlate_host -- the integrated run with HOST buffers (Fig. 7: host->device copy,
 *   X-engine, device->host copy of the result): copies in_host (dense, 4*N*F*T bytes, pinned for full speed) to
 *   in_dev_scratch (xc_scratch_in_bytes(), 16-byte aligned; rows are re-pitched to 128-byte multiples on the device, so any N -- N % 4 != 0
 *   included -- goes through the channel-range pipeline), correlates, copies the result into vis_host (xc_vis_bytes(), pinned for full speed) and
 *   synchronises the stream before returning.  Blocks of 8 MiB and more are cut into up to 16 channel ranges so
 *   that the copy-in of range c+1, the X-engine on range c and the copy-out of range c-1 overlap; the copies then
 *   run on two plan-owned streams ordered against cuda_stream by events (the only place the library uses streams
 *   of its own).  in_dev_scratch / vis_dev_scratch are caller-owned device buffers of the plan's sizes. */
int xc_correlate_host(xc_plan_t* plan, const int8_t* in_host, int32_t* vis_host, int8_t* in_dev_scratch,
                      int32_t* vis_dev_scratch, void* cuda_stream);

/* xc_correlate_host_i4 -- xc_correlate_host for 4-bit samples (format of xc_correlate_i4): in4_host / in4_dev_scratch hold
 *   xc_in_bytes_i4() bytes; half the host->device bytes of the int8 call, same result cube. */
int xc_correlate_host_i4(xc_plan_t* plan, const uint8_t* in4_host, int32_t* vis_host, uint8_t* in4_dev_scratch,
                         int32_t* vis_dev_scratch, void* cuda_stream);

/* ---- F-engine + corner turn in front of the X-engine ("the next step is to develop
 * this into a full FX correlator") ------------------------------------------------------------------------------------
 * xc_fengine -- for every station s, polarisation p and time block t < T the F-point Fourier transform
 *        X[t][f][s][p] = sum_{k<F} volt[s][p][t*F + k] * exp(-2 pi i f k / F)       ("X_i(nu) = int A_i(tau)
 *   e^{-i 2 pi nu tau}"; "N (fast) Fourier transforms of length F ... once every F samples"),
 *   quantised to int8 as q = clip(rint(X * scale), -127, 127) per real component (round-half-even, decided in fp32;
 *   four to eight bits suffice) and written in the X-engine's input order [t][f][station][pol][re,im]
 *    -- the corner turn is this kernel's store pattern.
 *   volt_dev: int8 [N][2 pol][T*F samples][2 re,im], station-major time series (2-byte aligned); xc_volt_bytes().
 *   cube_dev: int8 rows (t, f) of 4N valid bytes, cube_pitch bytes apart (a multiple of 4, >= 4N; 0 = xc_scratch_pitch(),
 *   the 128-byte multiple the X-engine reads fastest; xc_cube_bytes() is the size at that pitch); 4-byte aligned.
 *   F must be a power of two <= 4096, else XC_ERR_UNSUPPORTED.  fp32 arithmetic (Stockham FFT, radix <= 32): the
 *   spectrum agrees with an fp64 DFT to about 1e-6 relative to sqrt(F) * max|volt|, so a quantised sample can differ by one
 *   step from an exact evaluation only where X * scale lies within that distance of a rounding boundary k + 1/2; the
 *   bins f = 0, F/4, F/2, 3F/4 of integer input are exact, ties included.
 * xc_fengine_f32 -- the same spectra unquantised and unscaled, float [T][F][N][2][2] (dense; 8-byte aligned): for checking
 *   the transform itself against an fp64 DFT.  Strided stores: a testing aid, not a fast path.
 * xc_fx -- the FX correlator: xc_fengine into cube_scratch_dev (xc_cube_bytes(), 16-byte aligned, pitch
 *   xc_scratch_pitch()), then the X-engine on it: vis (+)= sum_t X X^H.  Two launches on the caller's stream; the
 *   X-engine's prologue overlaps the F-engine's tail (programmatic dependent launch). */
/* xc_fengine_channels / xc_fx_channels -- the F-engine and the FX chain for ONE channel range [f0, f0 + nf) of the plan's F
 *   ("evaluated independently for every frequency"; one channel range per GPU, PAPER.md:285 -- every GPU
 *   receives the station time series, and keeps only its own channels of the corner turn).  The transforms
 *   are the full F-point ones (same arithmetic, hence the same quantised samples as xc_fengine), but only the range's
 *   channels are stored: cube_dev / cube_scratch_dev is a PRUNED cube, rows (t, f - f0), nf rows per time block,
 *   xc_scratch_pitch() (or cube_pitch) bytes apart -- xc_scratch_pitch() * nf * T bytes instead of xc_cube_bytes().
 *   xc_fx_channels then runs the X-engine on that cube and writes (accumulate: adds to) vis[f0 .. f0 + nf) of the FULL
 *   visibility cube vis_dev, like xc_correlate_channels.  Errors as xc_fengine / xc_fx; INVALID_ARG for a range outside
 *   [0, F); UNSUPPORTED with the SIMT kernel or XC_OPT_FORCE_STAGE selected. */
int xc_fengine_channels(xc_plan_t* plan, const int8_t* volt_dev, float scale, int8_t* cube_dev, size_t cube_pitch, int f0, int nf,
                        void* cuda_stream);
int xc_fx_channels(xc_plan_t* plan, const int8_t* volt_dev, float scale, int8_t* cube_scratch_dev, int32_t* vis_dev, int f0, int nf,
                   int accumulate, void* cuda_stream);
size_t xc_volt_bytes(const xc_plan_t* plan);   /* 4*N*F*T */
size_t xc_cube_bytes(const xc_plan_t* plan);   /* xc_scratch_pitch()*F*T */
int xc_fengine(xc_plan_t* plan, const int8_t* volt_dev, float scale, int8_t* cube_dev, size_t cube_pitch, void* cuda_stream);
int xc_fengine_f32(xc_plan_t* plan, const int8_t* volt_dev, float* spec_dev, void* cuda_stream);
int xc_fx(xc_plan_t* plan, const int8_t* volt_dev, float scale, int8_t* cube_scratch_dev, int32_t* vis_dev, int accumulate,
          void* cuda_stream);

#ifdef XC_PROFILE
/* PROFILING BUILD ONLY (-DXC_PROFILE; libxc_profile.so): trace_dev = device buffer of 3*256*4 int64 (or NULL to switch
 * off); CTA 0 of the tensor-core kernel writes clock64() stamps of its first 256 pipeline iterations per warp role
 * (0 = TMA producer, 1 = MMA issuer, 2 = epilogue) into it. */
int xc_debug_set_trace(xc_plan_t* plan, void* trace_dev);
#endif

/* Tile schedule introspection (for tests of the triangular map).
 *   xc_tile_count: number of scheduled tiles per channel for the integer path.
 *   xc_tile_get:   tile k -> (block row bi on the i side, block column bj on the j side) and
 *                  the tile's extent in stations (si stations on the i side, sj on the j side). */
int xc_tile_count(const xc_plan_t* plan);
int xc_tile_get(const xc_plan_t* plan, int k, int* bi, int* bj, int* si, int* sj);
/* T-split factor (1 or 2) used by the last integer compute call on this plan (see XC_OPT_TSPLIT). */
int xc_t_split(const xc_plan_t* plan);
/* Kernel (XC_F32_KERNEL_CUDA_CORES or XC_F32_KERNEL_TC) that the last xc_correlate_f32 call on this plan ran; 0 before. */
int xc_f32_kernel_used(const xc_plan_t* plan);
/* Origin shift used by the last integer compute call on this plan (see XC_OPT_ORIGIN_SHIFT): returns the period P (1, 2,
 * 4 or 8 channels; 0 for a null plan) and fills, for c < P, shift_bytes[c] (grid of channels f = c mod P moved left by so
 * many bytes = 4 x stations; 0 = not moved) and tiles[c] (tiles scheduled for such a channel).  Either array may be NULL,
 * else it holds 8 ints. */
int xc_origin_shift(const xc_plan_t* plan, int* shift_bytes, int* tiles);
/* The same decision for a block at device address base_addr (16-byte aligned) with rows row_pitch_bytes apart (a multiple of
 * 16, >= 4N), without touching the device: host logic only (used by the tests of the schedule).  Returns the period, 0 on bad
 * arguments; it also becomes what xc_origin_shift reports until the next compute call.  Tile k of a shifted channel is entry
 * k of the triangular list (bj = 0, 1, ...; bi = 0 .. bj) in units of the tile's stations, its first station bi * si - shift / 4. */
int xc_origin_shift_plan(xc_plan_t* plan, uint64_t base_addr, size_t row_pitch_bytes, int* shift_bytes, int* tiles);

/* The paper's closed-form triangular map and its inverse:
 *   g = by(by+1)/2 + bx,  by = floor(-1/2 + sqrt(1/4 + 2g)),  bx = g - by(by+1)/2,
 *   with an integer fix-up so it is exact for every g (SURVEY 8(c) reading 12). */
int64_t xc_tri_index(int64_t bx, int64_t by);
void xc_tri_inverse(int64_t g, int64_t* bx, int64_t* by);

/* Number of launches of this library's own kernels enqueued by the last compute call on this
 * plan (staging + X-engine), for bench accounting. */
int xc_last_launches(const xc_plan_t* plan);

const char* xc_status_string(int status);
/* Text of the last CUDA error seen by this plan ("" if none). */
const char* xc_last_cuda_error(const xc_plan_t* plan);
/* Library version string. */
const char* xc_version(void);

#ifdef __cplusplus
}
#endif
#endif /* XC_H_ */
