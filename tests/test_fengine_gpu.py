"""GPU parity tests of the F-engine + corner turn (xc_fengine / xc_fengine_f32 / xc_fx) against the CPU
oracle oracle/fo_oracle.c (a plain fp64 O(F^2) DFT), through the C ABI.

Floating point decides an integer here (the int8 cube), so parity has two parts (reading 21):
  * the fp32 spectrum (xc_fengine_f32) agrees with the fp64 oracle within TOL(F) = 4 * 2^-24 * (log2 F + 1) * sqrt(F) * 181
    (a bound on the rounding error of a log2 F-stage fp32 FFT on int8 complex samples, |x| <= 181);
  * the quantised cube equals the oracle's wherever the oracle's margin (distance of X * scale from the nearest k + 1/2)
    exceeds scale * TOL(F); elsewhere it may differ by one step, and such near-ties must be rare.  The bins 0, F/4, F/2,
    3F/4 of integer input are exact on both sides, ties included.
The FX chain is compared bit for bit on cases where the oracle reports no near-tie at all.
"""
import numpy as np
import pytest
import torch

import paper_1107_4264_b200 as xcb
import xc_workloads as wl
from oracle import fo, xo
from paper_1107_4264_b200 import build as xc_build

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _built():
    xc_build.build()
    xcb.load_library()
    assert torch.cuda.is_available()


def tol(F):
    return 4.0 * 2.0 ** -24 * (np.log2(F) + 1.0) * np.sqrt(F) * 181.0


def gpu_cube(p, volt, scale, pitch=None):
    N, F, T = p.N, p.F, p.T
    pitch = p.scratch_pitch if pitch is None else pitch
    cube = torch.full((T, F, pitch), 0x55, dtype=torch.int8, device="cuda")
    p.fengine(torch.from_numpy(volt).cuda(), scale, cube)
    torch.cuda.synchronize()
    c = cube.cpu().numpy()
    assert (c[:, :, 4 * N:] == 0x55).all()                     # nothing is written beyond the 4N valid bytes of a row
    return c[:, :, :4 * N].reshape(T, F, N, 2, 2)


def check_cube(got, ref, margin, F, scale):
    """Equal wherever the oracle's margin is clear of the fp32 error bound; +-1 at near-ties; near-ties rare."""
    eps = scale * tol(F)
    diff = got.astype(np.int32) - ref.astype(np.int32)
    clear = margin > eps
    assert (diff[clear] == 0).all(), f"{(diff[clear] != 0).sum()} mismatches away from rounding boundaries"
    assert np.abs(diff).max() <= 1
    q = np.zeros(F, bool)
    q[::max(F // 4, 1)] = True                                  # exact bins: both sides are exact, ties included
    assert (diff[:, q] == 0).all()
    return int((diff != 0).sum()), int((~clear[:, ~q]).sum())   # (mismatches, near-ties outside the exact bins)


@pytest.mark.parametrize("LOGF", list(range(0, 13)))
def test_spectrum_and_cube_every_power_of_two(LOGF):
    F = 1 << LOGF
    N, T = (5, 3) if F >= 1024 else ((9, 5) if F >= 64 else (33, 7))      # ragged in stations and time blocks
    volt = wl.voltages(N, F, T, seed=100 + LOGF, full_range_mix=True)
    scale = wl.fengine_scale(F)
    ref_cube, margin, ref_spec = fo.fengine(volt, F, scale, want_spec=True)
    p = xcb.Plan(N, F, T)
    spec = torch.full(p.in_shape(), float("nan"), dtype=torch.float32, device="cuda")
    p.fengine_f32(torch.from_numpy(volt).cuda(), spec)
    torch.cuda.synchronize()
    got = spec.cpu().numpy().astype(np.float64)
    assert np.isfinite(got).all()
    err = np.abs(got - ref_spec).max()
    assert err <= tol(F), (F, err, tol(F))
    nbad, nnear = check_cube(gpu_cube(p, volt, scale), ref_cube, margin, F, scale)
    assert nnear <= max(4, 0.01 * ref_cube.size), (nnear, ref_cube.size)      # near-ties are rare away from the exact bins
    p.close()


def test_exact_ties_and_clipping_on_gpu():
    """The golden tie cases of the oracle's quantiser, through the kernel: F = 4 impulse at k = 0 gives X[f] = A in every
    bin, scale 1/2 makes odd A an exact tie (round half to even); saturation is symmetric (never -128)."""
    p = xcb.Plan(1, 4, 1)
    for A, q in [(1, 0), (3, 2), (5, 2), (-1, 0), (-3, -2), (127, 64), (-128, -64)]:
        v = np.zeros((1, 2, 4, 2), np.int8)
        v[0, 0, 0, 0] = A
        c = gpu_cube(p, v, 0.5)
        assert (c[0, :, 0, 0, 0] == q).all() and (c[0, :, 0, 0, 1] == 0).all() and (c[0, :, 0, 1] == 0).all(), (A, c[0, :, 0, 0])
        assert np.array_equal(c, fo.fengine(v, 4, 0.5)[0])
    p = xcb.Plan(2, 16, 2)
    for fill in (127, -128):
        v = np.full((2, 2, 32, 2), fill, np.int8)
        c = gpu_cube(p, v, 1.0)
        assert np.array_equal(c, fo.fengine(v, 16, 1.0)[0])
        assert c[0, 0, 0, 0].tolist() == ([127, 127] if fill > 0 else [-127, -127])


def test_quarter_turn_tone_and_sign_on_gpu():
    """x[k] = A i^k on every signal: all energy in bin +F/4, exactly A F; bins 0, F/2, 3F/4 exactly 0 (PAPER.md:55 sign)."""
    N, F, T, A = 3, 256, 2, 3
    x = A * np.array([1, 1j, -1, -1j] * (F // 4))
    v = np.zeros((N, 2, T * F, 2), np.int8)
    v[..., 0] = np.tile(x.real, T)
    v[..., 1] = np.tile(x.imag, T)
    p = xcb.Plan(N, F, T)
    spec = p.fengine_f32(torch.from_numpy(v).cuda()).cpu().numpy()
    assert (spec[:, F // 4, :, :, 0] == A * F).all() and (spec[:, F // 4, :, :, 1] == 0).all()
    for f in (0, F // 2, 3 * F // 4):
        assert (spec[:, f] == 0).all()
    rest = np.delete(spec, F // 4, axis=1)
    assert np.abs(rest).max() < 1e-2


@pytest.mark.parametrize("N,F,T,pitch", [(33, 64, 5, 132), (33, 64, 5, 256), (100, 128, 3, 400), (100, 128, 3, 512),
                                         (8, 32, 9, 32), (500, 16, 4, 2048), (40, 1024, 2, 160)])
def test_cube_pitch_and_layout(N, F, T, pitch):
    """Dense (4N) and 128-byte-multiple row pitches give the same samples; every CTA tile shape (8 / 16 / 32 stations,
    several time blocks per CTA) and ragged N, T are covered; padding bytes stay untouched."""
    volt = wl.voltages(N, F, T, seed=7 * N + F)
    scale = wl.fengine_scale(F)
    ref_cube, margin = fo.fengine(volt, F, scale)
    p = xcb.Plan(N, F, T)
    check_cube(gpu_cube(p, volt, scale, pitch), ref_cube, margin, F, scale)
    p.close()


def test_error_paths():
    p = xcb.Plan(4, 12, 2)                                      # F not a power of two
    volt = torch.zeros(p.volt_shape(), dtype=torch.int8, device="cuda")
    with pytest.raises(xcb.XcError) as e:
        p.fengine(volt, 1.0)
    assert e.value.code == -2
    p = xcb.Plan(4, 8, 2)
    volt = torch.zeros(p.volt_shape(), dtype=torch.int8, device="cuda")
    with pytest.raises(xcb.XcError):
        p.fengine(volt, 1.0, torch.zeros((2, 8, 12), dtype=torch.int8, device="cuda"))      # pitch < 4N
    with pytest.raises(xcb.XcError):
        p.fengine(volt, 1.0, torch.zeros((2, 8, 18), dtype=torch.int8, device="cuda"))      # pitch % 4 != 0
    p.fengine(volt, 1.0)                                        # and the plan stays usable


@pytest.mark.parametrize("N,F,T,seed", [(6, 16, 12, 1), (9, 8, 20, 10)])
def test_fx_chain_bit_exact_when_no_near_tie(N, F, T, seed):
    """F-engine oracle -> X-engine oracle against xc_fx on seeded cases in which the ORACLE reports no sample within 3x the
    fp32 error bound of a rounding boundary (outside the exact bins): the cubes must then be identical, and the visibilities
    bit-exact; accumulate adds."""
    volt = wl.voltages(N, F, T, seed)
    scale = wl.fengine_scale(F)
    ref_cube, margin = fo.fengine(volt, F, scale)
    q = np.ones(F, bool)
    q[::max(F // 4, 1)] = False
    assert margin[:, q].min() > 3 * scale * tol(F)              # precondition, from the oracle alone
    ref_vis = xo.correlate_i8(ref_cube)
    p = xcb.Plan(N, F, T)
    assert np.array_equal(gpu_cube(p, volt, scale), ref_cube)
    vd = torch.from_numpy(volt).cuda()
    scratch = p.new_cube()
    vis = torch.full(p.vis_shape(), 0x5A5A5A5A, dtype=torch.int32, device="cuda")
    p.fx(vd, scale, scratch, vis)
    assert p.last_launches == 2
    torch.cuda.synchronize()
    assert np.array_equal(vis.cpu().numpy(), ref_vis)
    p.fx(vd, scale, scratch, vis, accumulate=True)
    torch.cuda.synchronize()
    assert np.array_equal(vis.cpu().numpy(), 2 * ref_vis)


def test_fx_chain_midsize_clean_baselines_bit_exact():
    """xc_fx against the two oracles chained at a size (N = 64, F = 64, T = 24: 3.9e5 quantised samples) where no seed is free
    of near-ties.  From the oracle's margins ALONE: station s is 'clean' in channel f when none of its samples there lies
    within scale * TOL(F) of a rounding boundary; the cube must equal the oracle's on every clean (f, s), and the visibility
    of every baseline whose two stations are clean must equal X-engine-oracle(F-engine-oracle(volt)) bit for bit (a sample
    that may round either way touches only baselines of its own station and channel)."""
    N, F, T = 64, 64, 24
    volt = wl.voltages(N, F, T, seed=64)
    scale = wl.fengine_scale(F)
    ref_cube, margin = fo.fengine(volt, F, scale)
    ref_vis = xo.correlate_i8(ref_cube)
    q = np.zeros(F, bool)
    q[::F // 4] = True                                           # exact bins: ties included
    clean = (margin > scale * tol(F)).all(axis=(0, 3, 4))        # [F][N]
    clean[q] = True
    assert 0.5 < clean.mean() < 1.0                              # the case has near-ties, and most stations have none
    p = xcb.Plan(N, F, T)
    vd = torch.from_numpy(volt).cuda()
    cube = p.new_cube()
    vis = torch.full(p.vis_shape(), 0x5A5A5A5A, dtype=torch.int32, device="cuda")
    p.fx(vd, scale, cube, vis)
    torch.cuda.synchronize()
    got_cube = cube.cpu().numpy()[:, :, :4 * N].reshape(T, F, N, 2, 2)
    check_cube(got_cube, ref_cube, margin, F, scale)
    same = (got_cube == ref_cube).all(axis=(0, 3, 4))
    assert same[clean].all()
    jj, ii = np.tril_indices(N)                                  # i <= j, baseline b = j (j + 1) / 2 + i
    b = jj * (jj + 1) // 2 + ii
    ok = np.zeros((F, N * (N + 1) // 2), bool)
    ok[:, b] = clean[:, ii] & clean[:, jj]
    assert ok.mean() > 0.3
    got_vis = vis.cpu().numpy()
    assert np.array_equal(got_vis[ok], ref_vis[ok])
    assert (got_vis != 0x5A5A5A5A).any(axis=(2, 3, 4)).all()     # every baseline was written
    p.close()


@pytest.mark.parametrize("N,F,T", [(9, 16, 20), (40, 64, 12), (130, 256, 5), (33, 1, 7)])
def test_fengine_and_fx_on_channel_ranges(N, F, T):
    """xc_fengine_channels / xc_fx_channels (one channel range per GPU): the pruned cube of a range equals
    those channels of the full cube bit for bit (same transforms, only the stores are pruned; poisoned padding untouched),
    and the ranges' visibilities, written into the full cube on two streams, equal xc_fx's; accumulate adds to the range only."""
    volt = wl.voltages(N, F, T, seed=70 + N)
    scale = wl.fengine_scale(F)
    p = xcb.Plan(N, F, T)
    vd = torch.from_numpy(volt).cuda()
    full_cube = p.fengine(vd, scale)
    full_vis = p.fx(vd, scale, p.new_cube())
    torch.cuda.synchronize()
    cuts = sorted({0, F // 3, (2 * F) // 3 + (1 if F > 2 else 0), F})
    ranges = [(a, b - a) for a, b in zip(cuts[:-1], cuts[1:]) if b > a]
    poison = 0x5A5A5A5A
    vis = torch.full(p.vis_shape(), poison, dtype=torch.int32, device="cuda")
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    torch.cuda.synchronize()
    scratch = []
    for k, (f0, nf) in enumerate(ranges):
        cube = torch.full((T, nf, p.scratch_pitch), 0x55, dtype=torch.int8, device="cuda")
        p.fengine_channels(vd, scale, f0, nf, cube)
        torch.cuda.synchronize()
        assert torch.equal(cube[:, :, :4 * N], full_cube[:, f0:f0 + nf, :4 * N])
        assert bool((cube[:, :, 4 * N:] == 0x55).all())
        scratch.append(p.new_cube_range(nf))
        p.fx_channels(vd, scale, scratch[-1], vis, f0, nf, stream=streams[k % 2])
        assert p.last_launches == 2
    torch.cuda.synchronize()
    assert torch.equal(vis, full_vis)
    f0, nf = ranges[-1]
    p.fx_channels(vd, scale, scratch[-1], vis, f0, nf, accumulate=True)
    torch.cuda.synchronize()
    want = full_vis.clone()
    want[f0:f0 + nf] *= 2
    assert torch.equal(vis, want)
    for f0, nf in [(-1, 1), (0, 0), (F, 1), (0, F + 1)]:
        with pytest.raises(xcb.XcError):
            p.fengine_channels(vd, scale, f0, nf, torch.empty((T, nf, p.scratch_pitch), dtype=torch.int8, device="cuda"))
    p.close()


def test_fx_chain_config3_shape_sampled():
    """The FX chain at BASELINE.json's config 3 shape class (N = 256, F = 512, T = 64 time blocks): sampled spectra of the
    cube against the oracle (near-tie rule), and xc_fx's visibilities equal to the X-engine run on the very cube the
    F-engine wrote (the X-engine itself is parity-tested against its oracle on any cube)."""
    N, F, T = 256, 512, 64
    volt = wl.voltages(N, F, T, seed=33)
    scale = wl.fengine_scale(F)
    p = xcb.Plan(N, F, T)
    vd = torch.from_numpy(volt).cuda()
    cube = p.new_cube()
    vis = p.new_vis()
    p.fx(vd, scale, cube, vis)
    torch.cuda.synchronize()
    got = cube.cpu().numpy()[:, :, :4 * N].reshape(T, F, N, 2, 2)
    rng = np.random.default_rng(5)
    sel = [(0, 0, 0), (N - 1, 1, T - 1)] + [(int(rng.integers(N)), int(rng.integers(2)), int(rng.integers(T))) for _ in range(30)]
    X = fo.spectra(volt, F, sel)                                 # [nsel][F] complex128
    nbad = 0
    for (s, pol, t), Xs in zip(sel, X):
        for c, part in enumerate((Xs.real, Xs.imag)):
            y = part * np.float64(np.float32(scale))
            ref = fo.quantise(part, scale)
            m = np.abs(y - np.floor(y) - 0.5)
            d = got[t, :, s, pol, c].astype(int) - ref.astype(int)
            assert (d[m > scale * tol(F)] == 0).all() and np.abs(d).max() <= 1, (s, pol, t, c)
            nbad += int((d != 0).sum())
    assert nbad <= 3
    p.set_in_pitch(p.scratch_pitch)
    assert torch.equal(p.correlate(cube), vis)


@pytest.mark.parametrize("N,F,T", [(128, 1024, 24), (1024, 64, 40), (500, 64, 33)])
def test_cube_other_config_shapes_sampled(N, F, T):
    """The other BASELINE shape classes (config 2: 1024-point transforms, radix 32 x 32; config 5: N = 1024 and the ragged
    N = 500 with 64-point transforms), a few time blocks each: sampled spectra of the cube against the oracle (near-tie rule)."""
    volt = wl.voltages(N, F, T, seed=N + F, tones=1)
    scale = wl.fengine_scale(F)
    p = xcb.Plan(N, F, T)
    got = gpu_cube(p, volt, scale)
    rng = np.random.default_rng(N)
    sel = [(0, 0, 0), (N - 1, 1, T - 1)] + [(int(rng.integers(N)), int(rng.integers(2)), int(rng.integers(T))) for _ in range(22)]
    X = fo.spectra(volt, F, sel)
    nbad = 0
    for (s, pol, t), Xs in zip(sel, X):
        for c, part in enumerate((Xs.real, Xs.imag)):
            y = part * np.float64(np.float32(scale))
            ref = fo.quantise(part, scale)
            m = np.abs(y - np.floor(y) - 0.5)
            d = got[t, :, s, pol, c].astype(int) - ref.astype(int)
            assert (d[m > scale * tol(F)] == 0).all() and np.abs(d).max() <= 1, (s, pol, t, c)
            nbad += int((d != 0).sum())
    assert nbad <= 3
    # the chain: xc_fx's cube is the one xc_fengine writes, and its visibilities are the X-engine's on that very cube
    cube = p.new_cube()
    vis = p.fx(torch.from_numpy(volt).cuda(), scale, cube)
    torch.cuda.synchronize()
    assert np.array_equal(cube.cpu().numpy()[:, :, :4 * N].reshape(T, F, N, 2, 2), got)
    p.set_in_pitch(p.scratch_pitch)
    assert torch.equal(p.correlate(cube), vis)
    p.close()


def test_random_shapes_fengine_and_fx():
    """Seeded sweep of ragged shapes (N, power-of-two F, T, cube pitch): the cube against the oracle (near-tie rule), and the
    X-engine run on that cube equal to xc_fx's visibilities."""
    rng = np.random.default_rng(20261105)
    for _ in range(14):
        N = int(rng.integers(1, 140))
        F = 1 << int(rng.integers(0, 10))
        T = int(rng.integers(1, max(2, 3000 // F)))
        volt = wl.voltages(N, F, T, seed=int(rng.integers(1 << 30)), tones=int(rng.integers(0, 3)), full_range_mix=True)
        scale = wl.fengine_scale(F) * float(rng.choice([0.5, 1.0, 4.0]))
        ref_cube, margin = fo.fengine(volt, F, scale)
        p = xcb.Plan(N, F, T)
        pitch = p.scratch_pitch if rng.integers(2) else ((4 * N + 15) // 16) * 16
        check_cube(gpu_cube(p, volt, scale, pitch), ref_cube, margin, F, scale)
        cube = p.new_cube()
        vis = p.fx(torch.from_numpy(volt).cuda(), scale, cube)
        p.set_in_pitch(p.scratch_pitch)
        assert torch.equal(p.correlate(cube), vis), (N, F, T)
        got = cube.cpu().numpy()[:, :, :4 * N].reshape(T, F, N, 2, 2)
        if np.array_equal(got, ref_cube):                     # no near-tie flipped: then the chain must match the oracles bit for bit
            assert np.array_equal(vis.cpu().numpy(), xo.correlate_i8(ref_cube)), (N, F, T)
        p.close()
