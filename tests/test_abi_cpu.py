"""CPU-side checks of the C-ABI library (no compute calls): it loads, exports every symbol
include/xc.h declares, validates arguments, and its triangular tile schedule
covers every stored station pair exactly once."""
import ctypes
import os
import re

import numpy as np
import pytest

import paper_1107_4264_b200 as xcb
from paper_1107_4264_b200 import build as xc_build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module", autouse=True)
def _built():
    xc_build.build()
    xcb.load_library()


def test_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "xc.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    # declarations inside #ifdef XC_PROFILE belong to the profiling build only
    prof = "".join(re.findall(r"#ifdef XC_PROFILE(.*?)#endif", hdr, flags=re.S))
    hdr = re.sub(r"#ifdef XC_PROFILE.*?#endif", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(xc_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(xcb.EXPORTED_SYMBOLS)
    assert set(re.findall(r"\b(xc_[a-z0-9_]+)\s*\(", prof)) == set(xcb.PROFILE_SYMBOLS)
    L = ctypes.CDLL(xcb.binding.LIB_PATH)
    for name in declared:
        assert hasattr(L, name), name
    for name in xcb.PROFILE_SYMBOLS:                        # the product build carries no profiling hooks
        assert not hasattr(L, name), name
    assert L.xc_set_option(xcb.Plan(8, 2, 16)._h, xcb.OPT_DEBUG_SKIP, 1) == -1


def test_no_oracle_or_cpu_path_in_product():
    """The product package never imports the oracle (or numpy compute) -- parity would be void."""
    pkg = os.path.join(ROOT, "paper_1107_4264_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, fn)).read()
                assert "oracle" not in src.replace("no oracle", ""), fn
                assert "xo_" not in src, fn


def test_plan_argument_validation():
    L = xcb.lib()
    h = ctypes.c_void_p()
    assert L.xc_plan(ctypes.byref(h), 16, 2, 4, 256, 0) == 0 and h.value
    assert L.xc_in_bytes(h) == 4 * 16 * 4 * 256
    assert L.xc_in_bytes_f32(h) == 16 * 16 * 4 * 256
    assert L.xc_n_baselines(h) == 136                      # BASELINE.json configs[0]
    assert L.xc_vis_bytes(h) == 32 * 136 * 4
    assert L.xc_in_pitch(h) == 64 and L.xc_scratch_pitch(h) == 128 and L.xc_scratch_in_bytes(h) == (128 + 64) * 4 * 256 and L.xc_workspace_bytes(h) == 128 * 4 * 256
    assert L.xc_set_in_pitch(h, 63) == -1 and L.xc_set_in_pitch(h, 256) == 0
    assert L.xc_in_pitch(h) == 256 and L.xc_in_bytes(h) == 256 * 4 * 256
    assert L.xc_set_in_pitch(h, 0) == 0 and L.xc_in_pitch(h) == 64
    L.xc_destroy(h)
    for args, code in [((0, 2, 4, 8, 0), -1), ((4, 2, 0, 8, 0), -1), ((4, 2, 4, 0, 0), -1),
                       ((4, 1, 4, 8, 0), -2), ((4, 2, 4, 8, 7), -2), ((4, 2, 4, 65536, 0), -3)]:
        h = ctypes.c_void_p()
        assert L.xc_plan(ctypes.byref(h), *args) == code, args
        assert not h.value
    assert L.xc_plan(None, 4, 2, 4, 8, 0) == -1
    assert L.xc_status_string(-3) == b"XC_ERR_OVERFLOW" and L.xc_status_string(-7) == b"XC_ERR_NO_MEMORY"
    assert L.xc_status_string(-8) == b"XC_ERR_UNKNOWN"
    L.xc_destroy(None)
    # 2 * 128^2 * XC_MAX_T still fits int32, one more sample does not (PAPER.md:96 reading 7)
    assert 2 * 128 * 128 * xcb.MAX_T < 2 ** 31 <= 2 * 128 * 128 * (xcb.MAX_T + 1)


def test_compute_without_gpu_fails_loudly():
    import torch
    if torch.cuda.is_available():
        pytest.skip("has a GPU")
    p = xcb.Plan(8, 2, 16)
    fake = ctypes.c_void_p(0x1000)
    rc = xcb.lib().xc_correlate(p._h, fake, fake, None)
    assert rc in (-5, -2)                                  # XC_ERR_CUDA / UNSUPPORTED: never a CPU fallback
    rc = xcb.lib().xc_correlate_f32(p._h, fake, fake, 0, None)
    assert rc in (-5, -2)


@pytest.mark.parametrize("mode", [0, 1, 3])
@pytest.mark.parametrize("N", [1, 2, 3, 5, 16, 31, 32, 33, 64, 65, 100, 128, 129, 256, 500, 512, 1024])
def test_tile_schedule_covers_triangle_exactly_once(N, mode):
    p = xcb.Plan(N, 1, 8)
    p.set_option(xcb.OPT_TILE, mode)
    tiles = p.tiles()
    cover = np.zeros((N, N), np.int32)
    for bi, bj, si, sj in tiles:
        i0, j0 = bi * si, bj * sj
        assert i0 < N and j0 < N
        ii = np.arange(i0, min(i0 + si, N))[:, None]
        jj = np.arange(j0, min(j0 + sj, N))[None, :]
        assert (ii <= jj).any(), "a scheduled tile holds no stored pair"
        cover[i0:i0 + si, j0:j0 + sj] += 1
    iu = np.triu_indices(N)                                # i <= j
    assert (cover[iu] == 1).all()
    assert len(set((t[0], t[1]) for t in tiles)) == len(tiles)
    # raw/useful area as in the paper's wasted-work model: never worse than 3x at N >= 64
    if N >= 64 and mode == 0:
        raw = sum(si * sj for _, _, si, sj in tiles)
        assert raw <= 4.0 * (N * (N + 1) // 2)


def test_tile_counts_match_survey_table():
    """S1: nb(nb+1)/2 square 256x256 tiles per channel, nb = ceil(4N/256) -> 1, 3, 10, 36, 136
    for N = 64 ... 1024 (CTA-pair tiles); the same formula with nb = ceil(4N/128) for single-CTA 128x128 tiles."""
    for N, n2, n1 in [(64, 1, 3), (128, 3, 10), (256, 10, 36), (512, 36, 136), (1024, 136, 528)]:
        p = xcb.Plan(N, 1, 8)
        p.set_option(xcb.OPT_TILE, xcb.TILE_2CTA_256x256)
        assert len(p.tiles()) == n2
        p.set_option(xcb.OPT_TILE, xcb.TILE_1CTA_128x128)
        assert len(p.tiles()) == n1


def test_triangular_map_round_trip():
    """g = by(by+1)/2 + bx and its inverse."""
    g = 0
    for by in range(0, 300):
        for bx in range(0, by + 1):
            assert xcb.tri_index(bx, by) == g
            assert xcb.tri_inverse(g) == (bx, by)
            g += 1
    for by in [10 ** 6, 94906265, 94906266, 2 ** 31 - 1, 3 * 10 ** 9]:   # around 2g ~ 2^53: float sqrt is inexact
        for bx in (0, 1, by // 2, by - 1, by):
            g = by * (by + 1) // 2 + bx
            assert xcb.tri_inverse(g) == (bx, by)


def test_shard_channels_partition():
    for F in (1, 7, 64, 1024):
        for ws in (1, 2, 3, 8):
            parts = [xcb.shard_channels(F, ws, r) for r in range(ws)]
            assert parts[0][0] == 0 and parts[-1][1] == F
            assert all(parts[k][1] == parts[k + 1][0] for k in range(ws - 1))
            sizes = [hi - lo for lo, hi in parts]
            assert max(sizes) - min(sizes) <= 1


def test_option_validation():
    """xc_set_option rejects values outside each option's range and unknown options (no device needed)."""
    p = xcb.Plan(64, 4, 128)
    L, h = xcb.lib(), p._h
    ok = [(xcb.OPT_I8_KERNEL, 2), (xcb.OPT_MAX_CTAS, 0), (xcb.OPT_MAX_CTAS, 37), (xcb.OPT_FORCE_STAGE, 1), (xcb.OPT_TILE, 3),
          (xcb.OPT_TILE, 0), (xcb.OPT_TSPLIT, 2), (xcb.OPT_TSPLIT, 0), (xcb.OPT_PDL, 0), (xcb.OPT_PDL, 1)]
    bad = [(xcb.OPT_I8_KERNEL, 3), (xcb.OPT_MAX_CTAS, -1), (xcb.OPT_TILE, 2), (xcb.OPT_TILE, 4), (xcb.OPT_TILE, -1),
           (xcb.OPT_TSPLIT, 3), (5, 0), (6, 0), (99, 0)]   # 5 / 6: round 1's epilogue / stage-size options are gone
    for opt, val in ok:
        assert L.xc_set_option(h, opt, val) == 0, (opt, val)
    for opt, val in bad:
        assert L.xc_set_option(h, opt, val) == -1, (opt, val)
    assert L.xc_set_option(None, xcb.OPT_TILE, 0) == -1
    # every tile mode keeps an exact-cover schedule after switching back and forth
    for mode in (3, 1, 0):
        p.set_option(xcb.OPT_TILE, mode)
        assert len(p.tiles()) >= 1


def test_tracked_ncu_exports_feed_the_bench_roofline():
    """bench.py reads `roofline.traffic` and the tensor-pipe figure from the tracked ncu exports under profiles/ (nothing is
    hard-coded in bench.py): every export of this round parses, names the X-engine kernel, and its DRAM traffic is within 12 %
    of the algorithmic bytes of its workload (input read once, output written once -- no wasted re-reads)."""
    import sys
    sys.path.insert(0, ROOT)
    import bench
    import xc_workloads as wl
    seen = 0
    for name in ("cfg2", "cfg3", "cfg4", "cfg5_N500", "cfg5_N1024"):
        prof = bench.ncu_profile(name)
        assert prof and prof["launches"] >= 1, name
        w = wl.CONFIGS[name]
        assert 0.88 <= prof["dram_bytes"] / (w.in_bytes + w.vis_bytes) <= 1.12, (name, prof["dram_bytes"])
        assert 40.0 < prof["tensor_pipe_active_pct"] <= 100.0
        seen += 1
    assert seen == 5
    assert bench.ncu_profile("no_such_workload") == {}


@pytest.mark.parametrize("mode", [xcb.TILE_2CTA_256x256, xcb.TILE_1CTA_128x128])
@pytest.mark.parametrize("N,F", [(500, 64), (100, 64), (36, 16), (68, 32), (12, 8), (1000, 8), (132, 32), (96, 3), (500, 3)])
def test_origin_shift_schedule_covers_triangle_exactly_once(N, F, mode):
    """DESIGN.md 4 (XC_OPT_ORIGIN_SHIFT; PAPER.md:112, 149 line-aligned rows): for every channel class the tile grid moved
    left by shift / 4 stations still covers every pair i <= j < N exactly once; shifts are what the addresses say; a class
    keeps the unshifted grid when the shift would cost more than a quarter more tiles; no shift at all unless pitch x F is a
    multiple of 128 bytes."""
    p = xcb.Plan(N, F, 64)
    p.set_option(xcb.OPT_TILE, mode)
    si = p.tiles()[0][2]
    n0 = -(-N // si)
    pitch = 4 * N
    for base in (0x7F0000000000, 0x7F0000000000 + 48):
        cls = p.origin_shift_plan(base, pitch)
        if (pitch * F) % 128:
            assert cls == [(0, n0 * (n0 + 1) // 2)]
            continue
        period = len(cls)
        assert period in (1, 2, 4, 8) and (pitch * period) % 128 == 0 and (period == 1 or (pitch * (period // 2)) % 128 != 0)
        for c, (shift, tiles) in enumerate(cls):
            want = (base + c * pitch) % 128
            n = -(-(4 * N + shift) // (4 * si))
            assert tiles == n * (n + 1) // 2
            assert shift in (0, want) and shift % 16 == 0
            if shift == 0 and want != 0:        # declined: the shifted grid would need more than 1.25 x the tiles
                nw = -(-(4 * N + want) // (4 * si))
                assert 4 * nw * (nw + 1) > 5 * n0 * (n0 + 1)
            cover = np.zeros((N, N), dtype=np.int32)
            k = 0
            for bj in range(n):
                for bi in range(bj + 1):
                    i0, j0 = bi * si - shift // 4, bj * si - shift // 4
                    ii = np.arange(max(i0, 0), min(i0 + si, N))[:, None]
                    jj = np.arange(max(j0, 0), min(j0 + si, N))[None, :]
                    cover[max(i0, 0):min(i0 + si, N), max(j0, 0):min(j0 + si, N)] += (ii <= jj)
                    k += 1
            assert k == tiles
            iu = np.triu_indices(N)
            assert (cover[iu] == 1).all() and cover.sum() == N * (N + 1) // 2
    p.close()
