"""paper_1107_4264_b200 -- a B200-native X-engine (FX-correlator cross-multiply stage).

Thin Python binding over the C-ABI library `libxc.so` (see include/xc.h): argument marshalling
only; every step of the path runs in the library's own CUDA kernels.  PyTorch is used for
device memory and streams.  There is no CPU fallback: if the library cannot be loaded, or no
sm_100 GPU is present, calls raise.
"""
from .binding import (XcError, Plan, correlate_i4_noalloc, NOALLOC_SCRATCH_BYTES, NOALLOC_MAX_N, lib, load_library, tri_index, tri_inverse, version,  # noqa: F401
                      I8_KERNEL_AUTO, I8_KERNEL_TC, I8_KERNEL_SIMT, OPT_I8_KERNEL, OPT_MAX_CTAS,
                      OPT_FORCE_STAGE, OPT_DEBUG_SKIP, OPT_TILE, OPT_PDL, OPT_TSPLIT, OPT_ORIGIN_SHIFT, OPT_F32_KERNEL, F32_KERNEL_AUTO, F32_KERNEL_CUDA_CORES, F32_KERNEL_TC, TILE_AUTO, TILE_1CTA_128x128,
                      TILE_2CTA_256x256, MAX_T, TIMING_WORDS, TRACE_WORDS, EXPORTED_SYMBOLS, PROFILE_SYMBOLS,
                      LIB_PATH, LIB_PROFILE_PATH, shard_channels)
