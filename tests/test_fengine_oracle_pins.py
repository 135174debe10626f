"""Pins of the F-engine oracle (oracle/fo_oracle.c) against what the paper and the mathematics fix -- none of these
retypes the oracle's own O(F^2) sum: hand-worked values (tests/golden/fengine_hand_examples.txt), closed forms (impulse,
quarter-turn tone), a library FFT (numpy.fft), Parseval, linearity, the circular shift theorem, the cube layout by probing
and the quantiser's tie / clip rules.  CPU only."""
import cmath
import os

import numpy as np
import pytest

import xc_workloads as wl
from oracle import fo, xo

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "fengine_hand_examples.txt")


def _volt_one(x, N=1, s=0, p=0):
    """volt [N][2][F][2] holding the complex sequence x in signal (s, p), zeros elsewhere (T = 1)."""
    F = len(x)
    v = np.zeros((N, 2, F, 2), np.int8)
    v[s, p, :, 0] = np.real(x)
    v[s, p, :, 1] = np.imag(x)
    return v


def _golden(kind):
    for line in open(GOLDEN):
        if line.startswith(kind + " "):
            yield [part.split() for part in line[len(kind):].split("|")]


def test_hand_examples_dft():
    n = 0
    for head, xs, Xs in _golden("dft"):
        F = int(head[0])
        x = np.array(xs, float).reshape(F, 2)
        want = np.array(Xs, float).reshape(F, 2)
        got = fo.spectrum(_volt_one(x[:, 0] + 1j * x[:, 1]), F, 0, 0, 0)
        assert np.array_equal(np.stack([got.real, got.imag], -1), want), (F, got)     # small integers: exact
        n += 1
    assert n == 3


def test_hand_example_exact_bins_of_an_impulse():
    for head, rest in _golden("bin"):
        F, k0, A = map(int, head)
        x = np.zeros(F, complex)
        x[k0] = A
        got = fo.spectrum(_volt_one(x), F, 0, 0, 0)
        vals = np.array(rest, float).reshape(-1, 3)
        for f, re, im in vals:
            assert got[int(f)] == complex(re, im), (f, got[int(f)])


@pytest.mark.parametrize("F", [1, 2, 4, 8, 16, 64, 256, 1024, 12, 100])
def test_twiddles_exact_at_eighth_turns_and_accurate_elsewhere(F):
    for m in range(F):
        w = fo.twiddle(F, m)
        ref = cmath.exp(-2j * cmath.pi * m / F)
        assert abs(w - ref) < 1e-15                             # cmath's own argument 2 pi m / F is rounded too
        assert abs(abs(w) - 1.0) < 3e-16
        if (4 * m) % F == 0:                                   # quarter turns: exactly 1, -i, -1, i
            assert w == [1, -1j, -1, 1j][(4 * m) // F]
        elif (8 * m) % F == 0:                                 # odd eighth turns: +-sqrt(1/2) in both parts
            assert abs(w.real) == abs(w.imag) == np.sqrt(0.5)


@pytest.mark.parametrize("F,k0", [(8, 0), (8, 3), (64, 17), (1024, 1000)])
def test_impulse_flat_spectrum_linear_phase(F, k0):
    """x[k] = A delta(k - k0)  ->  X[f] = A exp(-2 pi i f k0 / F): |X| flat, phase linear in f (closed form)."""
    A = 7 - 3j
    x = np.zeros(F, complex)
    x[k0] = A
    got = fo.spectrum(_volt_one(x), F, 0, 0, 0)
    want = np.array([A * cmath.exp(-2j * cmath.pi * ((f * k0) % F) / F) for f in range(F)])
    assert np.abs(got - want).max() < 1e-13
    assert np.abs(np.abs(got) - abs(A)).max() < 1e-13
    if k0 == 0:
        assert (got == A).all()


@pytest.mark.parametrize("F", [4, 16, 256, 1024])
def test_quarter_turn_tone_single_exact_bin_and_sign_of_exponent(F):
    """x[k] = A i^k = A exp(+2 pi i (F/4) k / F), exact in int8: the whole energy lands in bin +F/4 (X = A F exactly), not in
    3F/4 -- which fixes the sign of the exponent (e^{-i 2 pi nu tau}); the bins 0, F/2, 3F/4 see only
    quarter-turn twiddles and are exactly 0."""
    A = 5
    x = A * np.array([1, 1j, -1, -1j] * (F // 4))
    got = fo.spectrum(_volt_one(x), F, 0, 0, 0)
    assert got[F // 4] == A * F
    assert got[0] == 0 and got[F // 2] == 0 and got[3 * F // 4] == 0
    rest = np.delete(got, F // 4)
    assert np.abs(rest).max() < 1e-9


@pytest.mark.parametrize("N,F,T,seed", [(3, 8, 2, 1), (2, 64, 3, 2), (1, 256, 2, 3), (1, 1024, 1, 4), (2, 2, 5, 5), (2, 1, 4, 6)])
def test_equals_numpy_fft(N, F, T, seed):
    """A library FFT (pocketfft) on the same samples; error budget a few ulps of sqrt(F) * 181 * log2(F)."""
    v = wl.voltages(N, F, T, seed, full_range_mix=True)
    cube, margin, spec = fo.fengine(v, F, 1.0, want_spec=True)
    z = v[..., 0].astype(np.float64) + 1j * v[..., 1]                   # [N][2][T*F]
    ref = np.fft.fft(z.reshape(N, 2, T, F), axis=-1)                      # [N][2][T][F]
    ref = ref.transpose(2, 3, 0, 1)                                       # corner turn -> [T][F][N][2]
    got = spec[..., 0] + 1j * spec[..., 1]
    assert np.abs(got - ref).max() < 1e-12 * F * 181
    # the single-spectrum entry point is the same numbers
    assert np.array_equal(fo.spectrum(v, F, N - 1, 1, T - 1), got[T - 1, :, N - 1, 1])
    sel = [(0, 0, 0), (N - 1, 1, T - 1)]
    assert np.array_equal(fo.spectra(v, F, sel), np.stack([got[0, :, 0, 0], got[T - 1, :, N - 1, 1]]))


def test_parseval_linearity_shift():
    F, rng = 128, np.random.default_rng(7)
    a = rng.integers(-40, 41, size=(F, 2))
    b = rng.integers(-40, 41, size=(F, 2))                   # 2 a - b stays inside int8
    xa, xb = a[:, 0] + 1j * a[:, 1], b[:, 0] + 1j * b[:, 1]
    Xa, Xb = (fo.spectrum(_volt_one(x), F, 0, 0, 0) for x in (xa, xb))
    # Parseval: sum |X|^2 = F sum |x|^2
    assert abs((np.abs(Xa) ** 2).sum() - F * (np.abs(xa) ** 2).sum()) < 1e-9 * F * (np.abs(xa) ** 2).sum()
    # linearity (2 xa - xb still fits int8)
    Xc = fo.spectrum(_volt_one(2 * xa - xb), F, 0, 0, 0)
    assert np.abs(Xc - (2 * Xa - Xb)).max() < 1e-10
    # circular shift by m samples <-> phase ramp exp(-2 pi i f m / F)
    m = 5
    Xs = fo.spectrum(_volt_one(np.roll(xa, m)), F, 0, 0, 0)
    ramp = np.exp(-2j * np.pi * np.arange(F) * m / F)
    assert np.abs(Xs - Xa * ramp).max() < 1e-10
    # real input -> conjugate-symmetric spectrum
    Xr = fo.spectrum(_volt_one(a[:, 0].astype(complex)), F, 0, 0, 0)
    assert np.abs(Xr[1:] - np.conj(Xr[1:][::-1])).max() < 1e-10


def test_cube_layout_and_time_blocks_by_probing():
    """Corner turn: signal (s, p), time block t -> cube[t, :, s, p]; block t uses samples [tF, (t+1)F)."""
    N, F, T = 3, 8, 4
    for (s, p, t, k0) in [(0, 0, 0, 0), (2, 1, 3, 5), (1, 0, 2, 7)]:
        v = np.zeros((N, 2, T * F, 2), np.int8)
        v[s, p, t * F + k0, 0] = 10
        cube, margin, spec = fo.fengine(v, F, 1.0, want_spec=True)
        nz = np.argwhere(np.abs(spec).sum(axis=(1, 4)) > 0)               # (t, s, p) triples holding anything
        assert nz.tolist() == [[t, s, p]]
        want = 10 * np.exp(-2j * np.pi * np.arange(F) * k0 / F)
        got = spec[t, :, s, p, 0] + 1j * spec[t, :, s, p, 1]
        assert np.abs(got - want).max() < 1e-13
        assert np.array_equal(cube[t, :, s, p], np.rint(np.stack([want.real, want.imag], -1)).astype(np.int8))


def test_quantiser_ties_to_even_and_symmetric_clip():
    n = 0
    for head, Xs, qs in _golden("quant"):
        scale = float(head[0])
        got = fo.quantise(np.array(Xs, float), scale)
        assert got.tolist() == [int(q) for q in qs], (scale, got.tolist())
        n += 1
    assert n == 3
    # through the whole F-engine: F = 4 impulse of A at k = 0 gives X[f] = A in every bin; scale 1/2 -> ties
    for A, q in [(1, 0), (3, 2), (5, 2), (-1, 0), (-3, -2), (127, 64), (-128, -64)]:
        v = np.zeros((1, 2, 4, 2), np.int8)
        v[0, 0, 0, 0] = A
        cube, margin = fo.fengine(v, 4, 0.5)
        assert (cube[0, :, 0, 0, 0] == q).all() and (cube[0, :, 0, 0, 1] == 0).all(), (A, cube[0, :, 0, 0])
        if A % 2:
            assert (margin[0, :, 0, 0, 0] == 0).all()                    # exact ties are reported as margin 0
    # saturation: all 127 -> X[0] = 127 F
    v = np.full((1, 2, 16, 2), 127, np.int8)
    cube, margin = fo.fengine(v, 16, 1.0)
    assert cube[0, 0, 0, 0].tolist() == [127, 127]
    v = np.full((1, 2, 16, 2), -128, np.int8)
    cube, margin = fo.fengine(v, 16, 1.0)
    assert cube[0, 0, 0, 0].tolist() == [-127, -127]                       # symmetric clip: never -128


def test_margin_hand_examples():
    """fo_margin against values worked by hand (tests/golden/fengine_hand_examples.txt), not against its own formula; the
    2^24 + 1 entry fails if the margin were taken from the fp32 product the quantiser uses."""
    n = 0
    for head, Xs, ms in _golden("margin"):
        scale = float(head[0])
        got = fo.margin(np.array(Xs, float), scale)
        assert np.allclose(got, np.array(ms, float), rtol=0, atol=1e-7), (scale, got.tolist())
        n += 1
    assert n == 2
    # the same through the whole F-engine: F = 1 is the identity, so X = the sample itself (scale 1/8: 3/8 -> 0.125, 4/8 -> 0)
    v = np.zeros((1, 2, 1, 2), np.int8)
    v[0, 0, 0] = (3, 4)
    v[0, 1, 0] = (-1, 21)
    cube, margin = fo.fengine(v, 1, 0.125)
    assert margin[0, 0, 0].tolist() == [[0.125, 0.0], [0.375, 0.125]]
    assert cube[0, 0, 0].tolist() == [[0, 0], [0, 3]]                       # 0.375 -> 0, 0.5 -> 0 (tie to even), -0.125 -> 0, 2.625 -> 3


def test_margin_is_distance_to_rounding_boundary():
    v = wl.voltages(2, 64, 2, seed=11)
    scale = wl.fengine_scale(64)
    cube, margin, spec = fo.fengine(v, 64, scale, want_spec=True)
    y = spec * np.float64(np.float32(scale))
    d = np.abs(y - np.floor(y) - 0.5)
    assert np.allclose(margin, d, atol=1e-6)
    far = margin > 1e-3
    assert np.array_equal(cube[far], np.clip(np.rint(y[far]), -127, 127).astype(np.int8))
    assert 2.0 < cube.astype(float).std() < 40.0                            # the recipe's scale gives a few bits of signal


def test_fx_chain_of_the_two_oracles_sees_the_common_tone():
    """F-engine oracle -> X-engine oracle (both pinned separately): a tone common to all stations shows up as a rank-1
    visibility matrix in its own channel with phase phi_i - phi_j, and not in the others."""
    N, F, T = 6, 16, 64
    v = wl.voltages(N, F, T, seed=5, sigma=2.0, tones=1, amp=40.0)
    cube, margin = fo.fengine(v, F, wl.fengine_scale(F, sigma=2.0, target=2.0))
    vis = xo.correlate_i8(cube)
    power = np.abs(vis[:, :, 0, 0, 0].astype(float) + 1j * vis[:, :, 0, 0, 1]).sum(axis=1)
    f_tone = int(np.argmax(power))
    assert power[f_tone] > 5 * np.median(power)
    # rank 1 in the tone channel: V_01 V_12 ~ V_02 V_11 (closure), to the noise level
    def V(i, j):
        b = j * (j + 1) // 2 + i
        return complex(vis[f_tone, b, 0, 0, 0], vis[f_tone, b, 0, 0, 1])
    lhs, rhs = V(0, 1) * V(1, 2), V(0, 2) * V(1, 1)
    assert abs(lhs - rhs) < 0.2 * abs(rhs)
