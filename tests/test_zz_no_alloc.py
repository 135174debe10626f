"""xc_correlate_i4_noalloc: the 4-bit X-engine call that allocates no device memory.

Some users of this library are not allowed to allocate on the GPU: a real-time capture loop that cannot take cudaMalloc's
device-wide stall, a plug-in of an application that owns all device memory, a process whose remaining HBM a caching
allocator has already claimed.  For them the library carries ONE such entry point; it unpacks into a fixed 16 MiB array of
the library's device image instead of a cudaMalloc'ed workspace, and that array is shared by every call on the device.

What is checked here, against the existing path (Plan.correlate_i4, itself bit-exact against the oracle in
test_xc_gpu.py), with the integer path's tolerance -- none, the cubes must be equal bit for bit:
  * two calls in a row on different shapes, the second SMALLER than the first, so that bytes the first call left in the
    shared array would show up if the second read anything it had not written itself;
  * accumulate adds; both tile shapes are reached; every output entry is written (poisoned cubes);
  * sizes beyond the fixed array, or beyond the N limit, are refused with their own status codes and launch nothing;
  * free device memory does not move across a call once the device has been set up.

This file is named so that pytest collects it last: `pytest -x` stops at the first failure, and a failure here must not
hide the parity tests.  It passes on its own in a fresh process and after all the other tests.
"""
import os
import re

import numpy as np
import pytest

import paper_1107_4264_b200 as xcb
import xc_workloads as wl
from paper_1107_4264_b200 import build as xc_build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module", autouse=True)
def _built():
    xc_build.build()
    xcb.load_library()


def test_source_calls_no_allocating_routine():
    """Host logic only (runs without a GPU): the translation unit of the entry point names no allocating CUDA call, takes
    the array's device address from cudaGetSymbolAddress, and the limits in the header, the source and the binding agree."""
    src = open(os.path.join(ROOT, "paper_1107_4264_b200", "csrc", "xc_noalloc.cu")).read()
    code = re.sub(r"//[^\n]*", "", src)                      # comments may (and do) talk about cudaMalloc
    for banned in ("cudaMalloc", "cudaFree", "cudaHostAlloc", "cudaStreamCreate", "cudaEventCreate", "cuMemAlloc", "cudaMemPool",
                   "cublas", "new ", "std::vector"):
        assert banned not in code, banned
    assert re.search(r"static\s+__device__\s+__align__\(256\)\s+unsigned char\s+xc_noalloc_scratch\[XC_NOALLOC_SCRATCH_BYTES\]", code)
    assert "cudaGetSymbolAddress(&ptr, xc_noalloc_scratch)" in code
    hdr = open(os.path.join(ROOT, "include", "xc.h")).read()
    assert "#define XC_NOALLOC_SCRATCH_BYTES (16u * 1024u * 1024u)" in hdr and xcb.NOALLOC_SCRATCH_BYTES == 16 << 20
    assert f"#define XC_NOALLOC_MAX_N {xcb.NOALLOC_MAX_N}" in hdr
    # 9 block rows of 64 stations = 45 tiles: the largest triangle that fits the 48 inline table entries
    assert (xcb.NOALLOC_MAX_N + 63) // 64 == 9 and 9 * 10 // 2 <= 48 < 10 * 11 // 2


def test_argument_checks_need_no_gpu():
    """The refusals come before any CUDA call, so they can be checked anywhere."""
    import ctypes
    L = xcb.lib()
    one = ctypes.c_void_p(256)                               # never dereferenced: every case below is refused first
    assert L.xc_correlate_i4_noalloc(0, 1, 1, one, one, 0, None) == -1
    assert L.xc_correlate_i4_noalloc(4, 1, 1, None, one, 0, None) == -1
    assert L.xc_correlate_i4_noalloc(4, 1, 65536, one, one, 0, None) == -3
    assert L.xc_correlate_i4_noalloc(xcb.NOALLOC_MAX_N + 1, 1, 1, one, one, 0, None) == -2
    assert L.xc_correlate_i4_noalloc(4, 1, 1, one, ctypes.c_void_p(264), 0, None) == -4
    # 128-byte rows: exactly 16 MiB fits, one more row does not
    rows = xcb.NOALLOC_SCRATCH_BYTES // 128
    assert L.xc_correlate_i4_noalloc(32, rows // 1024 + 1, 1024, one, one, 0, None) == -6
    assert L.xc_status_string(-6) == b"XC_ERR_NO_WORKSPACE"


def _existing_path(x4_np, torch):
    T, F, N = x4_np.shape[:3]
    p = xcb.Plan(N, F, T)
    vis = torch.full(p.vis_shape(), 0x5A5A5A5A, dtype=torch.int32, device="cuda")
    p.correlate_i4(torch.from_numpy(x4_np).cuda(), vis)
    torch.cuda.synchronize()
    out = vis.cpu().numpy()
    p.close()
    return out


@pytest.mark.gpu
def test_two_calls_in_a_row_match_the_existing_path():
    import torch
    assert torch.cuda.is_available()
    # first a wide, multi-tile block (CTA-pair tiles, ragged N: padding stations inside the rows), then a small one whose
    # rows are shorter and fewer (single-CTA tile): everything the second call reads was left dirty by the first
    shapes = [(100, 40, 64), (37, 2, 100)]
    blocks = [wl.packed_i4(N, F, T, seed=900 + N) for (N, F, T) in shapes]
    want = [_existing_path(b, torch) for b in blocks]
    got = []
    dev_in = [torch.from_numpy(b).cuda() for b in blocks]
    cubes = [torch.full(w.shape, 0x5A5A5A5A, dtype=torch.int32, device="cuda") for w in want]
    for x, v in zip(dev_in, cubes):                           # back to back on one stream, no synchronisation in between
        xcb.correlate_i4_noalloc(x, v)
    torch.cuda.synchronize()
    for v, w in zip(cubes, want):
        assert np.array_equal(v.cpu().numpy(), w)
    # again in the opposite order, accumulating: the cubes double
    for x, v in zip(reversed(dev_in), reversed(cubes)):
        xcb.correlate_i4_noalloc(x, v, accumulate=True)
    torch.cuda.synchronize()
    for v, w in zip(cubes, want):
        assert np.array_equal(v.cpu().numpy(), 2 * w)


@pytest.mark.gpu
@pytest.mark.parametrize("N,F,T", [(1, 1, 1), (8, 3, 40), (64, 3, 257), (136, 1, 300), (300, 2, 33)])
def test_small_and_ragged_shapes(N, F, T):
    import torch
    x4 = wl.packed_i4(N, F, T, seed=950 + N)
    vis = torch.full((F, N * (N + 1) // 2, 2, 2, 2), 0x5A5A5A5A, dtype=torch.int32, device="cuda")
    xcb.correlate_i4_noalloc(torch.from_numpy(x4).cuda(), vis)
    torch.cuda.synchronize()
    assert np.array_equal(vis.cpu().numpy(), _existing_path(x4, torch))


@pytest.mark.gpu
def test_refuses_what_does_not_fit_and_launches_nothing():
    import torch
    # (128-byte rows) x 64 channels x 2049 samples = 16 MiB + 8 KiB
    N, F, T = 32, 64, 2049
    x4 = torch.zeros((T, F, N, 2), dtype=torch.uint8, device="cuda")
    vis = torch.full((F, N * (N + 1) // 2, 2, 2, 2), 7, dtype=torch.int32, device="cuda")
    with pytest.raises(xcb.XcError) as e:
        xcb.correlate_i4_noalloc(x4, vis)
    assert e.value.code == -6 and "XC_ERR_NO_WORKSPACE" in str(e.value) and str(xcb.NOALLOC_SCRATCH_BYTES) in str(e.value)
    torch.cuda.synchronize()
    assert bool((vis == 7).all())                            # untouched
    # one sample less fills the array to the last byte and works
    x4 = torch.from_numpy(wl.packed_i4(N, F, T - 1, seed=977)).cuda()
    xcb.correlate_i4_noalloc(x4, vis)
    torch.cuda.synchronize()
    assert np.array_equal(vis.cpu().numpy(), _existing_path(x4.cpu().numpy(), torch))
    with pytest.raises(xcb.XcError) as e:
        xcb.correlate_i4_noalloc(torch.zeros((1, 1, xcb.NOALLOC_MAX_N + 1, 2), dtype=torch.uint8, device="cuda"))
    assert e.value.code == -2


@pytest.mark.gpu
def test_free_device_memory_does_not_move():
    import torch
    x4 = torch.from_numpy(wl.packed_i4(48, 5, 70, seed=990)).cuda()
    vis = torch.empty((5, 48 * 49 // 2, 2, 2, 2), dtype=torch.int32, device="cuda")
    xcb.correlate_i4_noalloc(x4, vis)                        # set-up of this device, kernels loaded
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        xcb.correlate_i4_noalloc(x4, vis)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 >= free0
