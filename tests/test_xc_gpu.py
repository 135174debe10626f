"""GPU parity tests: the CUDA path (through the C ABI) against the CPU oracle, element by element.

int8 path: bit-exact.  fp32 path: |V - V64| <= 1e-5 * sqrt(V64_ii * V64_jj) (north_star; SURVEY 8(c)
reading 13), and exactly equal to the int8 result for integer-valued input whose sums stay below 2^24.
At BASELINE.json's full sizes the oracle covers a sample of channels (always f = 0 and F-1, all
baselines) and an independent exact fp64 matmul on the GPU (torch, no code shared with the kernels:
every partial sum is < 2^53) covers every output.
"""
import numpy as np
import pytest
import torch

import paper_1107_4264_b200 as xcb
import xc_workloads as wl
from oracle import xo
from paper_1107_4264_b200 import build as xc_build

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _built():
    xc_build.build()
    xcb.load_library()
    assert torch.cuda.is_available()


# (tile shape, T-split option): the two built tile shapes; the single-CTA tile without and with the T-split forced
MODES = [(xcb.TILE_1CTA_128x128, 1), (xcb.TILE_1CTA_128x128, 2), (xcb.TILE_2CTA_256x256, 0)]
MODE_IDS = ["solo128", "solo128-tsplit", "pair256"]


def run_i8(x_np, kernel=xcb.I8_KERNEL_AUTO, force_stage=False, max_ctas=0, tile=xcb.TILE_AUTO, tsplit=0):
    T, F, N = x_np.shape[:3]
    p = xcb.Plan(N, F, T)
    p.set_option(xcb.OPT_TILE, tile)
    p.set_option(xcb.OPT_TSPLIT, tsplit)
    p.set_option(xcb.OPT_I8_KERNEL, kernel)
    p.set_option(xcb.OPT_FORCE_STAGE, int(force_stage))
    p.set_option(xcb.OPT_MAX_CTAS, max_ctas)
    x = torch.from_numpy(x_np).cuda()
    vis = torch.full(p.vis_shape(), 0x5A5A5A5A, dtype=torch.int32, device="cuda")  # poison: every entry must be written
    p.correlate(x, vis)
    torch.cuda.synchronize()
    out = vis.cpu().numpy()
    p.close()
    return out


def gram_check_fp64(x_gpu, vis_gpu, f_chunk=8):
    """Independent exact check of EVERY output: fp64 matmul of the real 4N x T matrix per channel."""
    T, F, N = x_gpu.shape[:3]
    iu = torch.triu_indices(N, N, device="cuda")            # (i, j) with i <= j
    order = torch.argsort(iu[1] * (iu[1] + 1) // 2 + iu[0])
    ii, jj = iu[0][order], iu[1][order]
    for f0 in range(0, F, f_chunk):
        f1 = min(F, f0 + f_chunk)
        z = x_gpu[:, f0:f1].reshape(T, f1 - f0, 2 * N, 2).to(torch.float64)
        zc = torch.complex(z[..., 0], z[..., 1]).permute(1, 2, 0)            # [f][2N][T]
        full = zc @ zc.conj().transpose(1, 2)                                  # x x^H, [f][2N][2N]
        full = full.reshape(f1 - f0, N, 2, N, 2)
        ref = full[:, ii, :, jj, :]                                            # [nb][f][pi][pj] (advanced idx first)
        ref = ref.permute(1, 0, 2, 3)
        ref = torch.stack([ref.real, ref.imag], dim=-1).round().to(torch.int64)
        got = vis_gpu[f0:f1].to(torch.int64)
        if not torch.equal(ref, got):
            bad = (ref != got).nonzero()[0].tolist()
            raise AssertionError(f"mismatch at f={f0 + bad[0]} b={bad[1]} idx={bad[2:]}: "
                                 f"ref={ref[tuple(bad)].item()} got={got[tuple(bad)].item()}")


# ---------------------------------------------------------------------------------------------
# config 1 in full, both kernels
# ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("kernel", [xcb.I8_KERNEL_TC, xcb.I8_KERNEL_SIMT])
def test_config1_full(kernel):
    w = wl.CONFIGS["cfg1"]
    x = wl.make_input(w)
    ref = xo.correlate_i8(x)
    got = run_i8(x, kernel)
    assert got.shape == (4, 136, 2, 2, 2)
    assert np.array_equal(got, ref)


# ---------------------------------------------------------------------------------------------
# small shapes: several tiles, ragged tails in N and T, degenerate sizes
# ---------------------------------------------------------------------------------------------

SMALL = [(1, 1, 1), (2, 3, 5), (3, 2, 31), (5, 2, 33), (16, 3, 64), (31, 2, 65), (32, 2, 100), (33, 2, 129),
         (40, 3, 1000), (64, 2, 200), (65, 2, 96), (100, 2, 257), (128, 2, 300), (132, 1, 130), (200, 1, 70),
         (257, 1, 64), (300, 1, 33)]


@pytest.mark.parametrize("mode", MODES, ids=MODE_IDS)
@pytest.mark.parametrize("N,F,T", SMALL)
def test_small_shapes_tc(N, F, T, mode):
    x = wl.full_range(N, F, T, seed=N * 1000 + T)            # whole int8 range incl. -128 (reading 6)
    ref = xo.correlate_i8(x)
    assert np.array_equal(run_i8(x, xcb.I8_KERNEL_TC, tile=mode[0], tsplit=mode[1]), ref)


@pytest.mark.parametrize("N,F,T", [(1, 1, 1), (5, 2, 33), (33, 2, 129), (100, 2, 57)])
def test_small_shapes_simt(N, F, T):
    x = wl.full_range(N, F, T, seed=7 + N)
    assert np.array_equal(run_i8(x, xcb.I8_KERNEL_SIMT), xo.correlate_i8(x))


def test_all_minus_128():
    """Worst case magnitude: every component -128; V = 2 * 128^2 * T on every real part."""
    N, F, T = 36, 2, 96
    x = np.full((T, F, N, 2, 2), -128, np.int8)
    got = run_i8(x)
    assert np.array_equal(got, xo.correlate_i8(x))
    assert (got[..., 0] == 2 * 128 * 128 * T).all() and (got[..., 1] == 0).all()


def test_max_T_no_overflow():
    """T = XC_MAX_T with all -128: 2 * 128^2 * 65535 = 2147450880 < 2^31 (reading 7)."""
    N, F, T = 4, 1, xcb.MAX_T
    x = np.full((T, F, N, 2, 2), -128, np.int8)
    got = run_i8(x)
    assert (got[..., 0] == 2 * 128 * 128 * T).all() and (got[..., 1] == 0).all()


def test_forced_staging_and_unaligned_pointer():
    N, F, T = 64, 3, 150
    x = wl.full_range(N, F, T, seed=5)
    ref = xo.correlate_i8(x)
    assert np.array_equal(run_i8(x, force_stage=True), ref)
    # input pointer off by 4 bytes: not 16-byte aligned -> S0 staging path is taken by the library itself
    p = xcb.Plan(N, F, T)
    buf = torch.zeros(x.size + 64, dtype=torch.int8, device="cuda")
    xs = buf[4:4 + x.size].view(T, F, N, 2, 2)
    assert xs.data_ptr() % 16 == 4
    xs.copy_(torch.from_numpy(x))
    ws = torch.empty(p.workspace_bytes, dtype=torch.int8, device="cuda")
    p.set_workspace(ws)
    vis = p.correlate(xs)
    assert p.last_launches == 2
    torch.cuda.synchronize()
    assert np.array_equal(vis.cpu().numpy(), ref)


def test_error_paths_on_device():
    """Status codes promised by include/xc.h: misaligned vis, workspace too small / misaligned, null pointers; and a
    failed call leaves the plan usable."""
    import ctypes
    N, F, T = 10, 2, 40                                       # N % 4 != 0 -> staging needed
    x = wl.full_range(N, F, T, seed=1)
    p = xcb.Plan(N, F, T)
    L, h = xcb.lib(), p._h
    xd = torch.from_numpy(x).cuda()
    vbuf = torch.zeros(p.vis_bytes // 4 + 16, dtype=torch.int32, device="cuda")
    st = ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)
    assert L.xc_correlate(h, ctypes.c_void_p(xd.data_ptr()), ctypes.c_void_p(vbuf.data_ptr() + 4), st) == -4   # XC_ERR_ALIGNMENT
    assert L.xc_correlate(h, None, ctypes.c_void_p(vbuf.data_ptr()), st) == -1
    assert L.xc_correlate(h, ctypes.c_void_p(xd.data_ptr()), None, st) == -1
    small = torch.zeros(256, dtype=torch.int8, device="cuda")
    assert L.xc_set_workspace(h, ctypes.c_void_p(small.data_ptr()), 256) == -6            # XC_ERR_NO_WORKSPACE
    big = torch.zeros(p.workspace_bytes + 256, dtype=torch.int8, device="cuda")
    assert L.xc_set_workspace(h, ctypes.c_void_p(big.data_ptr() + 8), p.workspace_bytes) == -4
    assert L.xc_set_workspace(h, ctypes.c_void_p(big.data_ptr()), p.workspace_bytes) == 0
    vis = p.correlate(xd)
    assert np.array_equal(vis.cpu().numpy(), xo.correlate_i8(x))
    assert L.xc_set_workspace(h, None, 0) == 0                                             # back to a library-owned one
    assert np.array_equal(p.correlate(xd).cpu().numpy(), xo.correlate_i8(x))
    assert L.xc_integrate(h, None, 1, None, None, None, None, st, st) == -1
    assert L.xc_correlate_pipelined(h, ctypes.c_void_p(1 << 20), 0, ctypes.c_void_p(1 << 20), ctypes.c_void_p(vbuf.data_ptr()), st, st) == -1


def test_persistent_schedule_independent_of_cta_count():
    N, F, T = 100, 5, 200
    x = wl.gaussian(N, F, T, seed=11, sigma=30.0)
    ref = xo.correlate_i8(x)
    for tile, ts in MODES:
        for ctas in (1, 2, 7, 0):
            assert np.array_equal(run_i8(x, max_ctas=ctas, tile=tile, tsplit=ts), ref), (tile, ts, ctas)


def test_accumulate_is_linear_in_time():
    """I = N_p * I': three blocks accumulated == one long integration, exactly."""
    N, F, T = 48, 4, 96
    blocks = [wl.gaussian(N, F, T, seed=20 + k, sigma=20.0) for k in range(3)]
    ref = xo.correlate_i8(np.concatenate(blocks, axis=0))
    for tile, ts in MODES:
        p = xcb.Plan(N, F, T)
        p.set_option(xcb.OPT_TILE, tile)
        p.set_option(xcb.OPT_TSPLIT, ts)
        vis = p.correlate(torch.from_numpy(blocks[0]).cuda())
        for b in blocks[1:]:
            p.correlate_acc(torch.from_numpy(b).cuda(), vis)
        torch.cuda.synchronize()
        assert np.array_equal(vis.cpu().numpy(), ref), (tile, ts)
        assert p.t_split == (2 if ts == 2 else 1)


def test_common_tone_phases_on_gpu():
    """Rank-1 input: V_ij = T A^2 w_i conj(w_j) (fixes which factor is conjugated, reading 1)."""
    N, F, T, A = 40, 2, 64, 3
    x, wq = wl.common_tone(N, F, T, seed=3, A=A)
    got = run_i8(x)
    w = np.exp(1j * np.pi / 2 * wq)                          # [f][s][p]
    for f in range(F):
        for (i, j) in [(0, 0), (0, 1), (3, 17), (39, 39), (12, 38)]:
            b = j * (j + 1) // 2 + i
            v = got[f, b, ..., 0] + 1j * got[f, b, ..., 1]
            exp = T * A * A * w[f, i][:, None] * np.conj(w[f, j])[None, :]
            assert np.allclose(v, exp)


# ---------------------------------------------------------------------------------------------
# two-stream pipeline (Algorithm 1) and the host end-to-end call
# ---------------------------------------------------------------------------------------------

def test_pipelined_matches_long_integration():
    N, F, T, nblk = 64, 8, 128, 5
    w = wl.Workload("pipe", N, F, T, "gauss", 8.0, 0)
    blocks = wl.make_blocks(w, nblk)
    ref = xo.correlate_i8(np.concatenate(blocks, axis=0))
    p = xcb.Plan(N, F, T)
    host = torch.from_numpy(np.stack(blocks)).pin_memory()
    dev2 = p.new_scratch(2)
    vis = torch.full(p.vis_shape(), -1, dtype=torch.int32, device="cuda")
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    torch.cuda.synchronize()
    p.correlate_pipelined(host, dev2, vis, s1, s2)
    s1.synchronize()
    assert p.last_launches == nblk
    assert np.array_equal(vis.cpu().numpy(), ref)
    # again into the same buffers: entry ordering against earlier work on the compute stream
    p.correlate_pipelined(host, dev2, vis, s1, s2)
    s1.synchronize()
    assert np.array_equal(vis.cpu().numpy(), ref)


def test_host_end_to_end_call():
    w = wl.CONFIGS["cfg1"]
    x = wl.make_input(w)
    p = xcb.Plan(w.N, w.F, w.T)
    xh = torch.from_numpy(x).pin_memory()
    vh = torch.empty(p.vis_shape(), dtype=torch.int32).pin_memory()
    xd = p.new_scratch()
    vd = p.new_vis()
    p.correlate_host(xh, vh, xd, vd)
    assert np.array_equal(vh.numpy(), xo.correlate_i8(x))


@pytest.mark.parametrize("N,F,T", [(1, 2, 9), (33, 3, 100), (50, 2, 64), (100, 43, 600)])
def test_host_paths_repitch_ragged_N(N, F, T):
    """The host-buffer calls give the X-engine a device block whose rows are 128-byte multiples (dense H2D copy + a small
    re-pitch kernel when 4N is not one already): any N -- N % 4 != 0 included -- works there, and blocks >= 8 MiB still go
    through the channel-range pipeline.  Same bits as the oracle through xc_correlate_host and xc_correlate_pipelined."""
    x = wl.full_range(N, F, T, seed=900 + N)
    ref = xo.correlate_i8(x)
    p = xcb.Plan(N, F, T)
    assert p.scratch_pitch % 128 == 0 and p.scratch_pitch >= 4 * N
    assert p.scratch_in_bytes == p.scratch_pitch * F * T + -(-4 * N * F * T // 128) * 128     # (no 4N here is a multiple of 128)
    xh = torch.from_numpy(x).pin_memory()
    vh = torch.full(p.vis_shape(), 0x5A5A5A5A, dtype=torch.int32).pin_memory()
    xd = p.new_scratch()
    xd.fill_(0x55)                                            # bytes between 4N and the pitch are never read as data
    vd = torch.full(p.vis_shape(), 0x5A5A5A5A, dtype=torch.int32, device="cuda")
    p.correlate_host(xh, vh, xd, vd)
    big = 4 * N * F * T >= (8 << 20)
    assert p.last_launches == (32 if big else 2)              # per channel range: re-pitch + X-engine
    assert np.array_equal(vh.numpy(), ref)
    host = torch.from_numpy(np.stack([x, x, x])).pin_memory()
    dev2 = p.new_scratch(2)
    dev2.fill_(0x55)
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    torch.cuda.synchronize()
    p.correlate_pipelined(host, dev2, vd, s1, s2)
    s1.synchronize()
    assert p.last_launches == 6
    assert np.array_equal(vd.cpu().numpy().astype(np.int64), 3 * ref.astype(np.int64))


def test_host_call_chunked_overlap():
    """Blocks of 8 MiB and more go through xc_correlate_host's channel-range pipeline (copy-in, X-engine and copy-out
    of different ranges overlap): same bits as the oracle, every output written, repeatable into the same buffers."""
    N, F, T = 64, 43, 1000                                   # 11 MB; F not a multiple of the 16 ranges
    x = wl.gaussian(N, F, T, seed=77, sigma=4.0)
    p = xcb.Plan(N, F, T)
    xh = torch.from_numpy(x).pin_memory()
    vh = torch.full(p.vis_shape(), 0x5A5A5A5A, dtype=torch.int32).pin_memory()
    xd = p.new_scratch()
    vd = torch.full(p.vis_shape(), 0x5A5A5A5A, dtype=torch.int32, device="cuda")
    p.correlate_host(xh, vh, xd, vd)
    assert p.last_launches == 16
    ref = xo.correlate_i8(x)
    assert np.array_equal(vh.numpy(), ref)
    vh.fill_(0)
    s = torch.cuda.Stream()
    p.correlate_host(xh, vh, xd, vd, stream=s)
    assert np.array_equal(vh.numpy(), ref)


def test_random_shapes_auto_mode():
    """Seeded sweep of ragged shapes through the launch configuration xc_plan picks by itself (AUTO), overwrite and
    accumulate, against the oracle -- bit-exact, every output written (poison check via the accumulate identity)."""
    rng = np.random.default_rng(20261104)
    shapes = [(int(rng.integers(1, 301)), int(rng.integers(1, 6)), int(rng.integers(1, 701))) for _ in range(36)]
    shapes += [(256, 2, 129), (255, 1, 128), (260, 1, 127), (64, 5, 1), (129, 2, 256)]
    for N, F, T in shapes:
        x = wl.full_range(N, F, T, seed=7 * N + T)
        ref = xo.correlate_i8(x)
        p = xcb.Plan(N, F, T)
        xd = torch.from_numpy(x).cuda()
        vis = torch.full(p.vis_shape(), 0x5A5A5A5A, dtype=torch.int32, device="cuda")
        p.correlate(xd, vis)
        got = vis.cpu().numpy()
        assert np.array_equal(got, ref), (N, F, T)
        p.correlate_acc(xd, vis)
        assert np.array_equal(vis.cpu().numpy(), 2 * ref), (N, F, T, "acc")
        p.close()


@pytest.mark.parametrize("N,F,T", [(100, 8, 200), (500, 8, 150), (36, 16, 300), (68, 32, 64), (12, 8, 33), (500, 16, 40)])
def test_origin_shift_unaligned_pitch(N, F, T):
    """Dense blocks whose rows are not 128 bytes apart while pitch x F is (XC_OPT_ORIGIN_SHIFT; PAPER.md:112,
    149): every channel's tile grid is moved left by the offset of its rows inside their 128-byte line.  Bit-exact against
    the oracle in both tile shapes, with and without T-split, overwrite and accumulate, on a channel sub-range (whose base
    address changes the shifts), every output written; the unshifted schedule gives the same cube."""
    assert (4 * N) % 128 != 0 and (4 * N * F) % 128 == 0
    x = wl.full_range(N, F, T, seed=3 * N + F)
    ref = xo.correlate_i8(x)
    xd = torch.from_numpy(x).cuda()
    for tile, ts in [(xcb.TILE_AUTO, 0), (xcb.TILE_2CTA_256x256, 0), (xcb.TILE_1CTA_128x128, 1), (xcb.TILE_1CTA_128x128, 2)]:
        p = xcb.Plan(N, F, T)
        p.set_option(xcb.OPT_TILE, tile)
        p.set_option(xcb.OPT_TSPLIT, ts)
        vis = torch.full(p.vis_shape(), 0x5A5A5A5A, dtype=torch.int32, device="cuda")
        p.correlate(xd, vis)
        used = p.origin_shift
        assert len(used) > 1 and any(sh for sh, _ in used), used             # the shifted schedule really ran
        assert all(sh % 16 == 0 and 0 <= sh < 128 for sh, _ in used)
        assert np.array_equal(vis.cpu().numpy(), ref), (tile, ts)
        p.correlate_acc(xd, vis)
        assert np.array_equal(vis.cpu().numpy(), 2 * ref), (tile, ts, "acc")
        # a channel sub-range starts at another address: other shifts, same numbers
        if F >= 8:
            vis.fill_(0x5A5A5A5A)
            p.correlate_channels(xd, vis, 3, F - 4)
            got = vis.cpu().numpy()
            assert np.array_equal(got[3:F - 1], ref[3:F - 1]), (tile, ts, "sub-range")
            assert (got[:3] == 0x5A5A5A5A).all() and (got[F - 1:] == 0x5A5A5A5A).all()
        # origin shift off: the round-1 schedule, same cube
        p.set_option(xcb.OPT_ORIGIN_SHIFT, 0)
        v0 = p.correlate(xd)
        assert p.origin_shift == [(0, len(p.tiles()))]
        assert np.array_equal(v0.cpu().numpy(), ref)
        p.close()


def test_origin_shift_random_shapes():
    """Seeded sweep of dense blocks with N % 4 == 0, N % 32 != 0 and F % 8 == 0 (so pitch x F is a multiple of 128 bytes and the
    shifted schedule runs) through the launch configuration xc_plan picks by itself: bit-exact, overwrite and accumulate."""
    rng = np.random.default_rng(20261105)
    done = 0
    while done < 14:
        N, F, T = 4 * int(rng.integers(1, 90)), 8 * int(rng.integers(1, 3)), int(rng.integers(1, 500))
        if N % 32 == 0:
            continue
        done += 1
        x = wl.full_range(N, F, T, seed=11 * N + T)
        ref = xo.correlate_i8(x)
        p = xcb.Plan(N, F, T)
        xd = torch.from_numpy(x).cuda()
        vis = torch.full(p.vis_shape(), 0x5A5A5A5A, dtype=torch.int32, device="cuda")
        p.correlate(xd, vis)
        assert len(p.origin_shift) > 1, (N, F, T)
        assert np.array_equal(vis.cpu().numpy(), ref), (N, F, T, p.origin_shift)
        p.correlate_acc(xd, vis)
        assert np.array_equal(vis.cpu().numpy(), 2 * ref), (N, F, T, "acc")
        p.close()


def test_origin_shift_misaligned_base_pointer():
    """A block whose rows ARE 128 bytes apart but whose base address is not line-aligned: one shift for all channels."""
    N, F, T = 96, 3, 200         # 384-byte rows: 384 + 112 still fits the pair tile's two block rows
    x = wl.full_range(N, F, T, seed=77)
    ref = xo.correlate_i8(x)
    buf = torch.zeros(x.size + 256, dtype=torch.int8, device="cuda")
    for off in (16, 48, 112):
        base = (-buf.data_ptr()) % 128 + off
        xd = buf[base:base + x.size].view(T, F, N, 2, 2)
        xd.copy_(torch.from_numpy(x))
        p = xcb.Plan(N, F, T)
        p.set_option(xcb.OPT_TILE, xcb.TILE_2CTA_256x256)
        vis = torch.full(p.vis_shape(), 0x5A5A5A5A, dtype=torch.int32, device="cuda")
        p.correlate(xd, vis)
        assert p.origin_shift == [(off, 3)]
        assert np.array_equal(vis.cpu().numpy(), ref), off
        p.close()


@pytest.mark.parametrize("N,F,T", [(1, 1, 1), (3, 2, 17), (8, 3, 40), (16, 2, 129), (37, 2, 100), (64, 3, 257), (100, 2, 130),
                                   (136, 1, 300)])
def test_i4_small_shapes(N, F, T):
    """4-bit samples (DESIGN reading 17) against the oracle's own nibble decoding: bit-exact, every
    output written, accumulate adds; both unpack kernels (N % 8 == 0 fast path and the general one) are covered."""
    x4 = wl.packed_i4(N, F, T, seed=50 + N)
    ref = xo.correlate_i4(x4)
    p = xcb.Plan(N, F, T)
    xd = torch.from_numpy(x4).cuda()
    vis = torch.full(p.vis_shape(), 0x5A5A5A5A, dtype=torch.int32, device="cuda")
    p.correlate_i4(xd, vis)
    assert np.array_equal(vis.cpu().numpy(), ref)
    p.correlate_i4(xd, vis, accumulate=True)
    assert np.array_equal(vis.cpu().numpy(), 2 * ref)
    # the same values as int8 through xc_correlate give the same cube
    v8 = p.correlate(torch.from_numpy(xo.unpack_i4(x4)).cuda())
    assert np.array_equal(v8.cpu().numpy(), ref)


def test_i4_host_call_chunked():
    """xc_correlate_host_i4 on a block large enough for the channel-range pipeline (unpack and X-engine per range):
    same cube as the oracle; and xc_correlate_channels stays whole-block-only for int8 input that needs staging."""
    N, F, T = 64, 70, 1000                                   # 8.96 MB packed
    x4 = wl.packed_i4(N, F, T, seed=71)
    p = xcb.Plan(N, F, T)
    xh = torch.from_numpy(x4).pin_memory()
    vh = torch.full(p.vis_shape(), 0x5A5A5A5A, dtype=torch.int32).pin_memory()
    xd = torch.zeros((T, F, N, 2), dtype=torch.uint8, device="cuda")
    vd = torch.full(p.vis_shape(), 0x5A5A5A5A, dtype=torch.int32, device="cuda")
    p.correlate_host_i4(xh, vh, xd, vd)
    assert p.last_launches == 32                              # 16 ranges x (unpack + X-engine)
    assert np.array_equal(vh.numpy(), xo.correlate_i4(x4))
    # ragged N (general unpack kernel, padded workspace rows), small block -> unchunked
    x4 = wl.packed_i4(13, 3, 50, seed=72)
    p = xcb.Plan(13, 3, 50)
    xh = torch.from_numpy(x4).pin_memory()
    vh = torch.zeros(p.vis_shape(), dtype=torch.int32).pin_memory()
    p.correlate_host_i4(xh, vh, torch.zeros((50, 3, 13, 2), dtype=torch.uint8, device="cuda"), p.new_vis())
    assert np.array_equal(vh.numpy(), xo.correlate_i4(x4))


def test_i4_config2_shape_sampled():
    """Config 2's shape with 4-bit samples: sampled channels against the oracle, every output against xc_correlate on the
    unpacked values (itself parity-tested at this size)."""
    w = wl.CONFIGS["cfg2"]
    x4 = wl.packed_i4(w.N, w.F, w.T, seed=2002)
    p = xcb.Plan(w.N, w.F, w.T)
    xd = torch.from_numpy(x4).cuda()
    vis = torch.full(p.vis_shape(), 0x5A5A5A5A, dtype=torch.int32, device="cuda")
    p.correlate_i4(xd, vis)
    assert p.last_launches == 2
    fsel = [0, 511, 1023]
    ref = xo.correlate_i4(np.ascontiguousarray(x4[:, fsel]))
    assert np.array_equal(vis[torch.tensor(fsel, device="cuda")].cpu().numpy(), ref)
    x8 = torch.from_numpy(xo.unpack_i4(x4)).cuda()
    assert torch.equal(p.correlate(x8), vis)


def test_integrate_long_integration_int64():
    """xc_integrate: Algorithm 1 with int64 widening.  (a) all -128 over 3 x 30000 samples leaves
    int32 (2 * 128^2 * 90000 > 2^31) and must hit the closed form; (b) random full-range blocks against the oracle's
    int64 sums over the concatenated integration, with a widening period of 2 blocks and a ragged last group; the host
    copy of the result is the same cube."""
    N, F, T, nblk = 8, 2, 30000, 3
    p = xcb.Plan(N, F, T)
    host = torch.full((nblk,) + p.in_shape(), -128, dtype=torch.int8).pin_memory()
    dev2 = p.new_scratch(2)
    v32 = p.new_vis()
    v64 = torch.full(p.vis_shape(), -7, dtype=torch.int64, device="cuda")
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    torch.cuda.synchronize()
    p.integrate(host, dev2, v32, v64, s1, s2)
    s1.synchronize()
    got = v64.cpu().numpy()
    assert (got[..., 0] == 2 * 128 * 128 * T * nblk).all() and (got[..., 1] == 0).all()
    assert 2 * 128 * 128 * T * nblk > 2 ** 31

    N, F, T, nblk = 40, 3, 30000, 7                          # group = 65535 // 30000 = 2 blocks -> widenings after 2, 4, 6, 7
    blocks = [wl.full_range(N, F, T, seed=300 + k) for k in range(nblk)]
    p = xcb.Plan(N, F, T)
    host = torch.from_numpy(np.stack(blocks)).pin_memory()
    dev2 = p.new_scratch(2)
    v32 = p.new_vis()
    v64 = torch.full(p.vis_shape(), -7, dtype=torch.int64, device="cuda")
    v64h = torch.zeros(p.vis_shape(), dtype=torch.int64).pin_memory()
    p.integrate(host, dev2, v32, v64, s1, s2, vis64_host=v64h)
    s1.synchronize()
    assert p.last_launches == 2 * nblk + 4                   # per block: re-pitch (4N = 160 -> 256) + X-engine; 4 widenings
    ref = xo.channels_i8_wide(np.concatenate(blocks, axis=0))
    assert np.array_equal(v64.cpu().numpy(), ref)
    assert np.array_equal(v64h.numpy(), ref)
    assert np.abs(ref).max() > 2 ** 31                       # the case really needs the widening


def test_cuda_graph_capture_and_pdl_chain():
    """xc_correlate / xc_correlate_acc are plain stream work (after the first call has created the plan's device
    state): they can be captured into a CUDA graph and replayed, and a chain of accumulate calls keeps its
    read-after-write order although the kernels are launched with programmatic stream serialization (each kernel
    waits for its predecessor before its first global access)."""
    N, F, T = 64, 6, 300
    x = wl.full_range(N, F, T, seed=11)
    ref = xo.correlate_i8(x).astype(np.int64)
    p = xcb.Plan(N, F, T)
    xd = torch.from_numpy(x).cuda()
    vis = p.new_vis()
    p.correlate(xd, vis)                                      # warm-up outside capture (tile table upload, attributes)
    s = torch.cuda.Stream()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=s):
        cur = torch.cuda.current_stream()
        p.correlate(xd, vis, stream=cur)
        for _ in range(6):
            p.correlate_acc(xd, vis, stream=cur)
    vis.fill_(-1)
    g.replay()
    torch.cuda.synchronize()
    assert np.array_equal(vis.cpu().numpy().astype(np.int64), 7 * ref)
    vis.fill_(3)
    g.replay()
    torch.cuda.synchronize()
    assert np.array_equal(vis.cpu().numpy().astype(np.int64), 7 * ref)
    # the same chain without PDL gives the same bits
    p.set_option(xcb.OPT_PDL, 0)
    p.correlate(xd, vis)
    for _ in range(6):
        p.correlate_acc(xd, vis)
    torch.cuda.synchronize()
    assert np.array_equal(vis.cpu().numpy().astype(np.int64), 7 * ref)


def test_correlate_channels_ranges():
    """xc_correlate_channels: ranges of one block, processed separately (here on two streams),
    write exactly their own slice of the cube; accumulate adds to that slice only."""
    N, F, T = 96, 11, 150
    x = wl.full_range(N, F, T, seed=5)
    ref = xo.correlate_i8(x)
    p = xcb.Plan(N, F, T)
    xd = torch.from_numpy(x).cuda()
    poison = 0x5A5A5A5A
    vis = torch.full(p.vis_shape(), poison, dtype=torch.int32, device="cuda")
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    torch.cuda.synchronize()
    p.correlate_channels(xd, vis, 0, 4, stream=s1)
    p.correlate_channels(xd, vis, 7, 4, stream=s2)
    torch.cuda.synchronize()
    got = vis.cpu().numpy()
    assert np.array_equal(got[0:4], ref[0:4]) and np.array_equal(got[7:11], ref[7:11])
    assert (got[4:7] == poison).all()
    p.correlate_channels(xd, vis, 4, 3)
    p.correlate_channels(xd, vis, 2, 5, accumulate=True)
    torch.cuda.synchronize()
    got = vis.cpu().numpy()
    want = ref.copy()
    want[2:7] *= 2
    assert np.array_equal(got, want)
    for f0, nf in [(-1, 2), (0, 0), (10, 2), (0, 12)]:
        with pytest.raises(xcb.XcError):
            p.correlate_channels(xd, vis, f0, nf)
    # a block that needs the staging pass (N % 4 != 0) is staged range by range; the SIMT kernel takes whole blocks only
    N2, F2, T2 = 45, 7, 90
    x2 = wl.full_range(N2, F2, T2, seed=6)
    ref2 = xo.correlate_i8(x2)
    p2 = xcb.Plan(N2, F2, T2)
    x2d = torch.from_numpy(x2).cuda()
    vis2 = torch.full(p2.vis_shape(), poison, dtype=torch.int32, device="cuda")
    p2.correlate_channels(x2d, vis2, 5, 2, stream=s1)
    p2.correlate_channels(x2d, vis2, 0, 3, stream=s2)
    torch.cuda.synchronize()
    assert p2.last_launches == 2                                  # staging + X-engine
    got2 = vis2.cpu().numpy()
    assert np.array_equal(got2[0:3], ref2[0:3]) and np.array_equal(got2[5:7], ref2[5:7]) and (got2[3:5] == poison).all()
    p2.correlate_channels(x2d, vis2, 3, 2)
    p2.correlate_channels(x2d, vis2, 1, 5, accumulate=True)
    torch.cuda.synchronize()
    want2 = ref2.copy()
    want2[1:6] *= 2
    assert np.array_equal(vis2.cpu().numpy(), want2)
    p2.set_option(xcb.OPT_I8_KERNEL, xcb.I8_KERNEL_SIMT)
    with pytest.raises(xcb.XcError):
        p2.correlate_channels(x2d, vis2, 1, 2)


# ---------------------------------------------------------------------------------------------
# pitched device input, T-split, timing stamps, staging on several streams, channel sharding on devices
# ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("N,F,T,pitch", [(50, 3, 130, 256), (33, 2, 100, 144), (33, 2, 100, 256), (500, 2, 300, 2048),
                                         (7, 2, 40, 30), (64, 2, 64, 256)])
def test_pitched_device_input(N, F, T, pitch):
    """xc_set_in_pitch (line-aligned rows): the same cube from a block whose rows are `pitch` bytes
    apart; the bytes between 4N and the pitch are garbage and must not matter.  A 16-byte-multiple pitch is read in
    place by TMA whatever N is (one launch); any other pitch goes through the staging kernel (two launches)."""
    x = wl.full_range(N, F, T, seed=400 + N + pitch)
    ref = xo.correlate_i8(x)
    for tile, ts in MODES:
        p = xcb.Plan(N, F, T)
        p.set_option(xcb.OPT_TILE, tile)
        p.set_option(xcb.OPT_TSPLIT, ts)
        p.set_in_pitch(pitch)
        assert p.in_pitch == pitch and p.in_bytes == pitch * F * T
        xd = torch.full((T, F, pitch), 0x77, dtype=torch.int8, device="cuda")
        xd[:, :, :4 * N] = torch.from_numpy(x).cuda().view(T, F, 4 * N)
        vis = torch.full(p.vis_shape(), 0x5A5A5A5A, dtype=torch.int32, device="cuda")
        p.correlate(xd, vis)
        assert p.last_launches == (1 if pitch % 16 == 0 else 2)
        assert np.array_equal(vis.cpu().numpy(), ref), (tile, ts)
        p.correlate_acc(xd, vis)
        assert np.array_equal(vis.cpu().numpy(), 2 * ref), (tile, ts)
        if pitch % 16 == 0:
            p.correlate_channels(xd, vis, F - 1, 1)
            assert np.array_equal(vis.cpu().numpy()[F - 1], ref[F - 1])
        p.set_option(xcb.OPT_I8_KERNEL, xcb.I8_KERNEL_SIMT)
        assert np.array_equal(p.correlate(xd).cpu().numpy(), ref)
        p.set_option(xcb.OPT_I8_KERNEL, xcb.I8_KERNEL_AUTO)
        p.set_option(xcb.OPT_FORCE_STAGE, 1)                    # the staging kernels read pitched rows too (any N)
        assert np.array_equal(p.correlate(xd).cpu().numpy(), ref)
        assert p.last_launches == 2
        p.close()


def test_t_split_selection_and_result():
    """T-split: AUTO turns it on for the single-CTA tile when 2 * tiles * F fits the SM
    count and the integration is long enough to pay for the hand-over (T >= 8192); forced, it runs whenever both ranks get
    a sample; the cube is the same bits either way (overwrite and accumulate, several tiles per cluster, ragged T)."""
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    for N, F, T, want in [(32, 8, 2048, 1), (32, 8, 8192, 2), (32, sms, 8200, 1), (16, 4, 256, 1), (8, 2, 1, 1), (8, 2, 32, 1),
                          (8, 2, 33, 1), (40, 3, 9001, 2)]:
        x = wl.full_range(N, F, T, seed=N + F + T)
        ref = xo.correlate_i8(x)
        p = xcb.Plan(N, F, T)
        vis = torch.full(p.vis_shape(), 0x5A5A5A5A, dtype=torch.int32, device="cuda")
        xd = torch.from_numpy(x).cuda()
        p.correlate(xd, vis)
        assert p.t_split == want, (N, F, T, p.t_split)
        assert np.array_equal(vis.cpu().numpy(), ref), (N, F, T)
        p.set_option(xcb.OPT_TILE, xcb.TILE_1CTA_128x128)
        for ts in (1, 2):
            p.set_option(xcb.OPT_TSPLIT, ts)
            for ctas in (0, 2, 6):                            # 1 and 3 clusters: several tiles per cluster
                p.set_option(xcb.OPT_MAX_CTAS, ctas)
                p.correlate(xd, vis)
                assert p.t_split == (2 if ts == 2 and T > 32 else 1)
                p.correlate_acc(xd, vis)
                assert np.array_equal(vis.cpu().numpy(), 2 * ref), (N, F, T, ts, ctas)
        p.close()


def test_timing_buffer():
    """xc_set_timing_buffer: [1] - [0] is the kernel's duration on the global nanosecond timer, CTA 0's cycle stamps give
    the SM clock; switching it off leaves the buffer untouched."""
    w = wl.CONFIGS["cfg5_N100"]
    x = torch.from_numpy(wl.make_input(w)).cuda()
    p = xcb.Plan(w.N, w.F, w.T)
    vis = p.new_vis()
    p.correlate(x, vis)
    st = torch.zeros(xcb.TIMING_WORDS, dtype=torch.int64, device="cuda")
    p.set_timing_buffer(st)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    st[0], st[1] = 2 ** 62, 0
    torch.cuda.synchronize()
    e0.record()
    p.correlate(x, vis)
    e1.record()
    torch.cuda.synchronize()
    t = st.tolist()
    dur_us = (t[1] - t[0]) / 1e3
    assert 1.0 < dur_us <= e0.elapsed_time(e1) * 1e3 + 5.0, (dur_us, e0.elapsed_time(e1))
    mhz = (t[4] - t[2]) / (t[5] - t[3]) * 1e3
    assert 500 < mhz < 2200, mhz
    p.set_timing_buffer(None)
    st.zero_()
    p.correlate(x, vis)
    torch.cuda.synchronize()
    assert (st == 0).all()


def test_staged_calls_on_two_streams_share_the_workspace_safely():
    """Two calls on one plan that both need the staging pass (N % 4 != 0), issued on different streams: the second
    staging kernel must wait for the first X-engine to finish with the plan-wide workspace (an event orders them)."""
    N, F, T = 30, 6, 4000
    xa = wl.full_range(N, F, T, seed=1)
    xb = wl.full_range(N, F, T, seed=2)
    ra, rb = xo.correlate_i8(xa), xo.correlate_i8(xb)
    p = xcb.Plan(N, F, T)
    da, db = torch.from_numpy(xa).cuda(), torch.from_numpy(xb).cuda()
    va, vb = p.new_vis(), p.new_vis()
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    torch.cuda.synchronize()
    for _ in range(4):
        p.correlate(da, va, stream=s1)
        p.correlate(db, vb, stream=s2)
    torch.cuda.synchronize()
    assert np.array_equal(va.cpu().numpy(), ra) and np.array_equal(vb.cpu().numpy(), rb)


def test_channel_sharding_on_devices():
    """PAPER.md:285 "data for different frequency channels can be trivially distributed among different GPUs": every
    shard_channels() range goes through its own plan's xc_correlate_channels into the shared cube; the assembled cube
    equals the oracle.  With two or more GPUs the ranges run on cuda:0 / cuda:1 (each plan binds to its device, the
    input block is replicated, the cube slices are gathered); with one GPU, on two streams of cuda:0."""
    N, F, T, world = 96, 13, 200, 2
    x = wl.full_range(N, F, T, seed=123)
    ref = xo.correlate_i8(x)
    ndev = torch.cuda.device_count()
    out = np.empty_like(ref)
    plans = []
    for r in range(world):
        lo, hi = xcb.shard_channels(F, world, r)
        dev = r % ndev
        with torch.cuda.device(dev):
            p = xcb.Plan(N, F, T)
            xd = torch.from_numpy(x).to(f"cuda:{dev}")
            vis = torch.full(p.vis_shape(), 0x5A5A5A5A, dtype=torch.int32, device=f"cuda:{dev}")
            s = torch.cuda.Stream(device=dev)
            p.correlate_channels(xd, vis, lo, hi - lo, stream=s)
            plans.append((p, vis, s, lo, hi, xd))
    for p, vis, s, lo, hi, xd in plans:
        s.synchronize()
        got = vis.cpu().numpy()
        out[lo:hi] = got[lo:hi]
        mask = np.ones(F, bool)
        mask[lo:hi] = False
        assert (got[mask] == 0x5A5A5A5A).all()                # a rank writes its own channels only
    assert np.array_equal(out, ref)
    if ndev >= 2:                                             # a plan stays on the device of its first compute call
        p0, _, _, lo, hi, xd0 = plans[0]
        with torch.cuda.device(1):
            with pytest.raises(xcb.XcError):
                p0.correlate_channels(xd0, plans[0][1], lo, hi - lo)


# ---------------------------------------------------------------------------------------------
# fp32 path
# ---------------------------------------------------------------------------------------------

def f32_tolerance_check(got, ref64, N):
    """|V - V64| <= 1e-5 sqrt(V64[(i,pi),(i,pi)] V64[(j,pj),(j,pj)]) per complex entry."""
    F = ref64.shape[0]
    diag = np.array([j * (j + 1) // 2 + j for j in range(N)])
    auto = np.stack([ref64[:, diag, 0, 0, 0], ref64[:, diag, 1, 1, 0]], axis=-1)     # [f][s][p]
    jj, ii = np.array([(j, i) for j in range(N) for i in range(j + 1)]).T
    norm = np.sqrt(auto[:, ii][:, :, :, None] * auto[:, jj][:, :, None, :])           # [f][b][pi][pj]
    err = np.abs((got[..., 0] - ref64[..., 0]) + 1j * (got[..., 1] - ref64[..., 1]))
    ratio = err / np.maximum(norm, 1e-30)
    assert ratio.max() <= 1e-5, ratio.max()
    return ratio.max()


F32_KERNELS = [xcb.F32_KERNEL_CUDA_CORES, xcb.F32_KERNEL_TC]     # fp32 FMAs on the CUDA cores / three TF32 MMAs per product


@pytest.mark.parametrize("kern", F32_KERNELS)
@pytest.mark.parametrize("N,F,T", [(1, 1, 1), (3, 2, 17), (33, 2, 100), (64, 3, 257), (100, 2, 130), (130, 1, 1000)])
def test_f32_against_fp64_oracle(N, F, T, kern):
    rng = np.random.default_rng(N + T)
    x = rng.standard_normal((T, F, N, 2, 2)).astype(np.float32) * 4.0
    p = xcb.Plan(N, F, T)
    p.set_option(xcb.OPT_F32_KERNEL, kern)
    vis = torch.full(p.vis_shape(), float("nan"), dtype=torch.float32, device="cuda")
    p.correlate_f32(torch.from_numpy(x).cuda(), vis)
    torch.cuda.synchronize()
    assert p.f32_kernel_used == kern
    got = vis.cpu().numpy().astype(np.float64)
    assert np.isfinite(got).all()
    f32_tolerance_check(got, xo.channels_f64(x), N)


@pytest.mark.parametrize("kern", F32_KERNELS)
def test_f32_long_integration_keeps_the_tolerance(kern):
    """T = 8192 Gaussian floats: sums of like-signed terms (the autocorrelations) must not drift -- the tensor core adds
    into its accumulator by truncation, so the tensor-core kernel sums 128-sample chunks there and the chunks in registers."""
    N, F, T = 70, 1, 8192
    rng = np.random.default_rng(8192)
    x = (rng.standard_normal((T, F, N, 2, 2)) * 3.0).astype(np.float32)
    p = xcb.Plan(N, F, T)
    p.set_option(xcb.OPT_F32_KERNEL, kern)
    vis = torch.full(p.vis_shape(), float("nan"), dtype=torch.float32, device="cuda")
    p.correlate_f32(torch.from_numpy(x).cuda(), vis)
    torch.cuda.synchronize()
    got = vis.cpu().numpy().astype(np.float64)
    worst = f32_tolerance_check(got, xo.channels_f64(x), N)
    if kern == xcb.F32_KERNEL_TC:
        assert worst < 3e-6, worst          # the bias of one 128-sample chunk, not of 8192 samples


def test_f32_tc_graph_capture_accumulate_chain_and_cta_cap():
    """The tensor-core fp32 kernel is plain stream work launched with programmatic stream serialization: an overwrite + 2
    accumulate calls (sums stay below 2^24) captured into a CUDA graph keep their read-after-write order (integer-valued input: exact), and a cap on
    the number of CTAs (XC_OPT_MAX_CTAS) changes the schedule, not the numbers."""
    N, F, T = 136, 5, 300
    x = wl.full_range(N, F, T, seed=31)
    ref = xo.correlate_i8(x).astype(np.float32)
    xf = torch.from_numpy(x).cuda().to(torch.float32)
    p = xcb.Plan(N, F, T)
    vis = p.new_vis(torch.float32)
    p.correlate_f32(xf, vis)
    assert p.f32_kernel_used == xcb.F32_KERNEL_TC
    s = torch.cuda.Stream()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=s):
        cur = torch.cuda.current_stream()
        p.correlate_f32(xf, vis, stream=cur)
        for _ in range(2):
            p.correlate_f32(xf, vis, accumulate=True, stream=cur)
    assert 3 * np.abs(ref).max() < 2 ** 24
    for fill in (float("nan"), 7.0):
        vis.fill_(fill)
        g.replay()
        torch.cuda.synchronize()
        assert np.array_equal(vis.cpu().numpy(), 3 * ref)
    for cap in (2, 7, 30):
        p.set_option(xcb.OPT_MAX_CTAS, cap)
        vis.fill_(float("nan"))
        p.correlate_f32(xf, vis)
        assert np.array_equal(vis.cpu().numpy(), ref), cap
    p.close()


def test_f32_channel_sharding():
    """xc_correlate_f32_channels (PAPER.md:65, 285 for float samples): every shard_channels() range of a 3-way split runs
    through its own plan on its own stream (on its own GPU when several exist) into a poison-filled cube; the assembled cube
    equals the whole-block call bit for bit (same kernel, same per-channel schedule), meets the tolerance against the fp64
    oracle, and no rank writes outside its range; accumulate adds; the CUDA-core kernel refuses proper sub-ranges."""
    N, F, T, world = 100, 11, 190, 3
    rng = np.random.default_rng(5)
    x = (rng.standard_normal((T, F, N, 2, 2)) * 3.0).astype(np.float32)
    ndev = torch.cuda.device_count()
    p_all = xcb.Plan(N, F, T)
    whole = p_all.correlate_f32(torch.from_numpy(x).cuda()).cpu().numpy()
    f32_tolerance_check(whole.astype(np.float64), xo.channels_f64(x), N)
    out = np.empty_like(whole)
    runs = []
    for r in range(world):
        lo, hi = xcb.shard_channels(F, world, r)
        dev = r % ndev
        with torch.cuda.device(dev):
            p = xcb.Plan(N, F, T)
            xd = torch.from_numpy(x).to(f"cuda:{dev}")
            vis = torch.full(p.vis_shape(), -77.0, dtype=torch.float32, device=f"cuda:{dev}")
            st = torch.cuda.Stream(device=dev)
            p.correlate_f32_channels(xd, vis, lo, hi - lo, stream=st)
            runs.append((p, xd, vis, st, lo, hi))
    for p, xd, vis, st, lo, hi in runs:
        st.synchronize()
        got = vis.cpu().numpy()
        out[lo:hi] = got[lo:hi]
        mask = np.ones(F, bool)
        mask[lo:hi] = False
        assert (got[mask] == -77.0).all()
    assert np.array_equal(out, whole)
    p, xd, vis, st, lo, hi = runs[1]
    with torch.cuda.device(vis.device):
        p.correlate_f32_channels(xd, vis, lo, hi - lo, accumulate=True, stream=st)
        st.synchronize()
        assert np.array_equal(vis.cpu().numpy()[lo:hi], 2 * whole[lo:hi])
        p.set_option(xcb.OPT_F32_KERNEL, xcb.F32_KERNEL_CUDA_CORES)
        with pytest.raises(xcb.XcError):
            p.correlate_f32_channels(xd, vis, lo, hi - lo)
        p.correlate_f32_channels(xd, vis, 0, F)              # the whole range is just xc_correlate_f32
        f32_tolerance_check(vis.cpu().numpy().astype(np.float64), xo.channels_f64(x), N)


def test_f32_tc_wide_dynamic_range():
    """The hi/lo split of the tensor-core kernel on samples whose magnitudes span 2^-20 .. 2^20 and whose mantissas are full
    (a single TF32 product would be off by 2^-11): still inside 1e-5 sqrt(V_ii V_jj) of the fp64 oracle; AUTO picks the
    tensor-core kernel at this N."""
    N, F, T = 72, 2, 96
    rng = np.random.default_rng(4711)
    x = (rng.standard_normal((T, F, N, 2, 2)) * np.exp2(rng.integers(-20, 21, size=(1, 1, N, 1, 1)))).astype(np.float32)
    p = xcb.Plan(N, F, T)
    vis = torch.full(p.vis_shape(), float("nan"), dtype=torch.float32, device="cuda")
    p.correlate_f32(torch.from_numpy(x).cuda(), vis)
    torch.cuda.synchronize()
    assert p.f32_kernel_used == xcb.F32_KERNEL_TC
    got = vis.cpu().numpy().astype(np.float64)
    assert np.isfinite(got).all()
    f32_tolerance_check(got, xo.channels_f64(x), N)


@pytest.mark.parametrize("N,F,T", [(100, 3, 130), (37, 2, 64), (500, 2, 96)])
def test_f32_pitched_rows(N, F, T):
    """xc_set_in_pitch_f32 (rows aligned to the memory line): the same float samples in rows padded to a
    multiple of 128 bytes (poisoned padding) give the same bits as the dense block, sub-ranges included, and meet the
    tolerance against the fp64 oracle; the CUDA-core kernel refuses a pitched plan; pitch 0 restores the dense default."""
    x = wl.gaussian(N, F, T, seed=300 + N, sigma=20.0).astype(np.float32) * np.float32(0.37)
    ref = xo.channels_f64(x)
    p = xcb.Plan(N, F, T)
    xd = torch.from_numpy(x).cuda()
    dense = p.correlate_f32(xd).cpu().numpy()
    f32_tolerance_check(dense.astype(np.float64), ref, N)
    pitch = (16 * N + 127) // 128 * 128
    xp = torch.full((T, F, pitch // 4), float("nan"), dtype=torch.float32, device="cuda")
    xp[:, :, :4 * N] = xd.view(T, F, 4 * N)
    with pytest.raises(xcb.XcError):
        p.set_in_pitch_f32(16 * N - 16)
    with pytest.raises(xcb.XcError):
        p.set_in_pitch_f32(pitch + 8)
    p.set_in_pitch_f32(pitch)
    assert p.in_pitch_f32 == pitch and p.in_bytes_f32 == pitch * F * T
    vis = torch.full(p.vis_shape(), float("nan"), dtype=torch.float32, device="cuda")
    p.correlate_f32(xp, vis)
    assert np.array_equal(vis.cpu().numpy(), dense)
    vis.fill_(float("nan"))
    for f0 in range(F):
        p.correlate_f32_channels(xp, vis, f0, 1)
    assert np.array_equal(vis.cpu().numpy(), dense)
    p.set_option(xcb.OPT_F32_KERNEL, xcb.F32_KERNEL_CUDA_CORES)
    with pytest.raises(xcb.XcError) as e:
        p.correlate_f32(xp, vis)
    assert e.value.code == -2
    p.set_option(xcb.OPT_F32_KERNEL, xcb.F32_KERNEL_AUTO)
    p.set_in_pitch_f32(0)
    assert p.in_pitch_f32 == 16 * N
    assert np.array_equal(p.correlate_f32(xd).cpu().numpy(), dense)
    p.close()


@pytest.mark.parametrize("kern", F32_KERNELS)
def test_f32_non_finite_sample_stays_inside_its_station(kern):
    """xc.h's precondition for float samples (finite, |a| < 2^127): one infinite sample and one that rounds to infinity in
    TF32 (0x7F7FF000 and above) spoil only the visibilities of their own station in their own channel -- non-finite there
    with either kernel -- while every other baseline still meets the tolerance against the fp64 oracle; a large but
    admissible sample (1e18: products 1e36) is handled by both kernels."""
    N, F, T = 40, 2, 64
    rng = np.random.default_rng(99)
    x = rng.standard_normal((T, F, N, 2, 2)).astype(np.float32)
    x[5, 0, 7, 0, 0] = 1e18                                     # admissible
    ref = xo.channels_f64(x)
    bad = x.copy()
    bad[3, 0, 11, 1, 0] = np.inf
    bad[9, 1, 30, 0, 1] = np.float32(3.4028e38)                 # finite, but rounds to infinity as TF32
    p = xcb.Plan(N, F, T)
    p.set_option(xcb.OPT_F32_KERNEL, kern)
    good = p.correlate_f32(torch.from_numpy(x).cuda()).cpu().numpy().astype(np.float64)
    f32_tolerance_check(good, ref, N)
    got = p.correlate_f32(torch.from_numpy(bad).cuda()).cpu().numpy().astype(np.float64)
    p.close()
    jj, ii = np.array([(j, i) for j in range(N) for i in range(j + 1)]).T
    for f, s in [(0, 11), (1, 30)]:
        touched = (ii == s) | (jj == s)
        assert not np.isfinite(got[f, s * (s + 1) // 2 + s]).all()               # the station's own autocorrelation is spoilt
        assert np.isfinite(got[f, ~touched]).all()
        got[f, touched] = ref[f, touched]                                        # everything else must be as if nothing happened
    f32_tolerance_check(got, ref, N)


@pytest.mark.parametrize("kern", F32_KERNELS)
def test_f32_gaussian_floats_N256_sampled_channels(kern):
    """Config 3's shape class (N = 256, T = 1000) with genuinely non-integer Gaussian floats: sampled channels (first,
    last, two seeded) against the fp64-accumulating oracle at north_star's tolerance 1e-5 * sqrt(V_ii V_jj)."""
    N, F, T = 256, 24, 1000
    rng = np.random.default_rng(2563)
    x = (rng.standard_normal((T, F, N, 2, 2)) * 4.0 + rng.standard_normal((T, F, 1, 1, 2))).astype(np.float32)
    p = xcb.Plan(N, F, T)
    p.set_option(xcb.OPT_F32_KERNEL, kern)
    vis = torch.full(p.vis_shape(), float("nan"), dtype=torch.float32, device="cuda")
    p.correlate_f32(torch.from_numpy(x).cuda(), vis)
    torch.cuda.synchronize()
    fsel = sorted({0, F - 1, *rng.integers(0, F, size=2).tolist()})
    got = vis[torch.tensor(fsel, device="cuda")].cpu().numpy().astype(np.float64)
    assert torch.isfinite(vis).all()
    worst = f32_tolerance_check(got, xo.channels_f64(x, fsel), N)
    assert worst > 1e-9                                       # the comparison is not vacuous: fp32 rounding is visible


@pytest.mark.parametrize("kern", F32_KERNELS)
def test_f32_random_shapes_exact_on_integer_input_and_accumulate(kern):
    """The fp32 kernels at ragged sizes (CUDA cores: 16 x 16-station warp blocks and diagonal skipping; tensor cores: pair
    tiles, zero-filled edges, lo parts all zero): integer-valued input keeps every fp32 sum exact, so the result must equal
    the integer oracle bit for bit; accumulate adds exactly."""
    rng = np.random.default_rng(99)
    shapes = [(int(rng.integers(1, 200)), int(rng.integers(1, 4)), int(rng.integers(1, 300))) for _ in range(16)]
    shapes += [(15, 1, 16), (16, 1, 17), (17, 2, 15), (47, 1, 33), (48, 1, 48), (49, 1, 31), (96, 2, 50), (97, 1, 64)]
    for N, F, T in shapes:
        x = wl.full_range(N, F, T, seed=13 * N + T)
        ref = xo.correlate_i8(x).astype(np.float32)
        p = xcb.Plan(N, F, T)
        p.set_option(xcb.OPT_F32_KERNEL, kern)
        xd = torch.from_numpy(x).cuda().to(torch.float32)
        vis = torch.full(p.vis_shape(), float("nan"), dtype=torch.float32, device="cuda")
        p.correlate_f32(xd, vis)
        assert np.array_equal(vis.cpu().numpy(), ref), (N, F, T)
        p.correlate_f32(xd, vis, accumulate=True)
        assert np.array_equal(vis.cpu().numpy(), 2 * ref), (N, F, T, "acc")
        p.close()


@pytest.mark.parametrize("kern", F32_KERNELS)
def test_f32_equals_int8_for_integer_input(kern):
    """Config 3's values as float: all products and sums are exact in fp32 -> identical results."""
    w = wl.Workload("cfg3small", 256, 4, 1000, "gauss_tone", 4.0, 1003)
    x = wl.make_input(w)
    p = xcb.Plan(w.N, w.F, w.T)
    p.set_option(xcb.OPT_F32_KERNEL, kern)
    xd = torch.from_numpy(x).cuda()
    vi = p.correlate(xd)
    vf = p.correlate_f32(xd.to(torch.float32))
    torch.cuda.synchronize()
    ref = xo.correlate_i8(x)
    assert np.array_equal(vi.cpu().numpy(), ref)
    assert np.array_equal(vf.cpu().numpy(), ref.astype(np.float32))
    # accumulate flag
    p.correlate_f32(xd.to(torch.float32), vf, accumulate=True)
    torch.cuda.synchronize()
    assert np.array_equal(vf.cpu().numpy(), 2 * ref.astype(np.float32))


# ---------------------------------------------------------------------------------------------
# BASELINE.json's full sizes, in the launch configuration bench.py times
# ---------------------------------------------------------------------------------------------

FULL = ["cfg2", "cfg3", "cfg4", "cfg5_N32", "cfg5_N64", "cfg5_N100", "cfg5_N500", "cfg5_N1024"]


@pytest.mark.parametrize("name", FULL)
def test_full_size_configs(name):
    w = wl.CONFIGS[name]
    x = wl.make_input(w)
    p = xcb.Plan(w.N, w.F, w.T)
    xd = torch.from_numpy(x).cuda()
    vis = torch.full(p.vis_shape(), 0x5A5A5A5A, dtype=torch.int32, device="cuda")
    # the other tile shapes must give the very same bits (tile-schedule independence)
    first = None
    for tile, ts in MODES:
        p.set_option(xcb.OPT_TILE, tile)
        p.set_option(xcb.OPT_TSPLIT, ts)
        v2 = p.correlate(xd)
        if first is None:
            first = v2
        else:
            assert torch.equal(first, v2), (name, tile, ts)
    del first, v2
    p.set_option(xcb.OPT_TILE, xcb.TILE_AUTO)           # the launch configuration bench.py times
    p.set_option(xcb.OPT_TSPLIT, 0)
    p.correlate(xd, vis)
    torch.cuda.synchronize()
    # (a) oracle on sampled channels, all baselines
    nsel = 2 if w.N >= 1000 else (3 if w.N >= 500 else 4)
    rng = np.random.default_rng(w.seed)
    fsel = sorted({0, w.F - 1, *rng.integers(0, w.F, size=nsel - 2).tolist()})
    ref = xo.channels_i8(x, fsel)
    got = vis[torch.tensor(fsel, device="cuda")].cpu().numpy()
    assert np.array_equal(got, ref), name
    # (b) every output against an exact fp64 matmul (independent of the kernels)
    gram_check_fp64(xd, vis, f_chunk=max(1, 2048 // w.N))
    # (c) invariants that hold at any size: autocorrelations real, same-station cross-pols conjugate
    diag = torch.tensor([j * (j + 1) // 2 + j for j in range(w.N)], device="cuda")
    a = vis[:, diag]
    assert (a[:, :, 0, 0, 1] == 0).all() and (a[:, :, 1, 1, 1] == 0).all()
    assert torch.equal(a[:, :, 0, 1, 0], a[:, :, 1, 0, 0]) and torch.equal(a[:, :, 0, 1, 1], -a[:, :, 1, 0, 1])
    if name == "cfg3":
        # the same values through the fp32 path (BASELINE.json configs[2]): exact for these magnitudes
        vf = p.correlate_f32(xd.to(torch.float32))
        torch.cuda.synchronize()
        assert torch.equal(vf, vis.to(torch.float32))


def test_cfg5_two_stream_eight_blocks():
    """Config 5's pipelined run: 8 host blocks accumulated (total integration 16384 samples)."""
    w = wl.CONFIGS["cfg5_N100"]
    blocks = wl.make_blocks(w, 8)
    p = xcb.Plan(w.N, w.F, w.T)
    host = torch.from_numpy(np.stack(blocks)).pin_memory()
    dev2 = p.new_scratch(2)
    vis = p.new_vis()
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    torch.cuda.synchronize()
    p.correlate_pipelined(host, dev2, vis, s1, s2)
    s1.synchronize()
    fsel = [0, 31, 63]
    ref = xo.channels_i8(np.concatenate(blocks, axis=0), fsel)
    assert np.array_equal(vis[torch.tensor(fsel, device="cuda")].cpu().numpy(), ref)
