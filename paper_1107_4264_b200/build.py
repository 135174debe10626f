"""Builds libxc.so (the C-ABI X-engine library) in-tree with nvcc for sm_100a.

    python -m paper_1107_4264_b200.build [--force] [-v] [--profile]

--profile builds libxc_profile.so with -DXC_PROFILE: the same library plus the profiling hooks
(xc_debug_set_trace, XC_OPT_DEBUG_SKIP) that the product build does not contain.

nvcc cross-compiles without a GPU.  The .so is git-ignored (history stays source-only) but
travels to the GPU box with the gpurun snapshot.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libxc.so")
LIB_PROFILE = os.path.join(HERE, "libxc_profile.so")
SOURCES = ["xc_api.cu", "xc_noalloc.cu"]
HEADERS = ["xc_ptx.cuh", "xc_i8_tc.cuh", "xc_f32.cuh", "xc_f32_tc.cuh", "xc_fengine.cuh", "xc_simt.cuh", os.path.join("..", "..", "include", "xc.h")]
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-shared", "-Xcompiler", "-fPIC"]


def _nvcc() -> str:
    cand = os.path.join(os.environ.get("CUDA_HOME", "/usr/local/cuda"), "bin", "nvcc")
    return cand if os.path.exists(cand) else "nvcc"


def stale(lib: str = LIB) -> bool:
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False, profile: bool = False) -> str:
    lib = LIB_PROFILE if profile else LIB
    if not force and not stale(lib):
        return lib
    tmp = lib + f".tmp{os.getpid()}"
    cmd = [_nvcc()] + NVCC_FLAGS + os.environ.get("XC_NVCC_EXTRA", "").split() + (["-DXC_PROFILE"] if profile else []) + \
          (["-Xptxas", "-v"] if verbose else []) + \
          ["-o", tmp] + [os.path.join(CSRC, s) for s in SOURCES]
    subprocess.check_call(cmd, cwd=CSRC)
    os.replace(tmp, lib)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, profile="--profile" in sys.argv))
