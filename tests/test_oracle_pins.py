"""Pins for the CPU oracle (oracle/xo_oracle.c) against what the paper and mathematics fix.

None of these retypes the oracle's loop: each pin is a different route to the same numbers
(Python `complex` brute force, numpy's matmul X @ X^H, hand-worked values, closed forms,
invariants), chosen so that a dropped term, a wrong sign, a swapped index or a transposed
operand fails at least one.  CPU only (-m "not gpu").
"""
import os

import numpy as np
import pytest

from oracle import xo
import xc_workloads as wl

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def tri(i, j):
    return j * (j + 1) // 2 + i


def to_complex(x):
    """int8 [T][F][N][2][2] -> complex128 [T][F][2N] with row index a = 2*s + p."""
    T, F, N = x.shape[:3]
    z = x[..., 0].astype(np.float64) + 1j * x[..., 1].astype(np.float64)
    return z.reshape(T, F, 2 * N)


def vis_to_complex(vis):
    return vis[..., 0].astype(np.float64) + 1j * vis[..., 1].astype(np.float64)


# --- counts and index order -------------------------------------------

def test_baseline_count_config1():
    assert xo.n_baselines(16) == 136          # BASELINE.json configs[0]: "136 baselines"
    x = wl.uniform_small(16, 4, 8, 1)
    assert xo.correlate_i8(x).shape == (4, 136, 2, 2, 2)


@pytest.mark.parametrize("N", [1, 2, 3, 5, 8])
def test_triangle_order_by_probing(N):
    """Light up one station pair at a time; exactly slot j(j+1)/2+i (and the two autos) respond."""
    for j in range(N):
        for i in range(j + 1):
            x = np.zeros((1, 1, N, 2, 2), np.int8)
            x[0, 0, i, 0, 0] = 1
            x[0, 0, j, 0, 0] = 1
            v = xo.correlate_i8(x)[0]
            nz = set(np.nonzero(np.abs(v).sum(axis=(1, 2, 3)))[0].tolist())
            assert nz == {tri(i, i), tri(i, j), tri(j, j)}
    assert tri(0, 0) == 0 and tri(0, 1) == 1 and tri(1, 1) == 2 and tri(N - 1, N - 1) == xo.n_baselines(N) - 1


def test_pol_and_reim_slot_order():
    """Only (station 0, pol 0) = 1 and (station 1, pol 1) = i are non-zero: the cross term must sit in
    [pi=0][pj=1] with value 1 * conj(i) = -i, nowhere else."""
    x = np.zeros((1, 1, 2, 2, 2), np.int8)
    x[0, 0, 0, 0, 0] = 1
    x[0, 0, 1, 1, 1] = 1
    v = xo.correlate_i8(x)[0, tri(0, 1)]
    exp = np.zeros((2, 2, 2), np.int32)
    exp[0, 1, 1] = -1
    assert np.array_equal(v, exp)


# --- hand-worked values -----------------------------------------------------------------------

def test_hand_examples():
    xs, vs = [], []
    with open(os.path.join(GOLDEN, "hand_examples.txt")) as fh:
        for line in fh:
            tok = line.split()
            if not tok or tok[0].startswith("#"):
                continue
            (xs if tok[0] == "x" else vs).append([int(t) for t in tok[1:]])
    x = np.zeros((1, 1, 2, 2, 2), np.int8)
    for s, p, re, im in xs:
        x[0, 0, s, p] = (re, im)
    vis = xo.correlate_i8(x)[0]
    assert len(vs) == 12
    for i, pi, j, pj, re, im in vs:
        assert tuple(vis[tri(i, j), pi, pj]) == (re, im), (i, pi, j, pj)


# --- brute force with Python complex arithmetic -----------------------------------------------

@pytest.mark.parametrize("N,F,T,seed", [(1, 1, 1, 0), (2, 2, 3, 1), (3, 1, 8, 2), (4, 3, 5, 3)])
def test_brute_force_python_complex(N, F, T, seed):
    x = wl.full_range(N, F, T, seed)
    vis = xo.correlate_i8(x)
    for f in range(F):
        for j in range(N):
            for i in range(j + 1):
                for pi in range(2):
                    for pj in range(2):
                        s = 0j
                        for t in range(T):
                            a = complex(int(x[t, f, i, pi, 0]), int(x[t, f, i, pi, 1]))
                            b = complex(int(x[t, f, j, pj, 0]), int(x[t, f, j, pj, 1]))
                            s += a * b.conjugate()
                        got = vis[f, tri(i, j), pi, pj]
                        assert (int(got[0]), int(got[1])) == (round(s.real), round(s.imag))


# --- textbook routine: Hermitian rank-T update X X^H (numpy matmul) ---------------------------

@pytest.mark.parametrize("N,F,T,seed", [(5, 2, 33, 10), (16, 4, 256, 1001), (33, 2, 100, 11)])
def test_equals_numpy_herk(N, F, T, seed):
    x = wl.full_range(N, F, T, seed) if seed != 1001 else wl.uniform_small(N, F, T, seed)
    z = to_complex(x)                                   # [T][F][2N]
    vis = vis_to_complex(xo.correlate_i8(x))            # [F][NB][2][2]
    for f in range(F):
        X = z[:, f, :].T                                # [2N][T]
        S = X @ X.conj().T                              # exact: |entries| < 2^53
        for j in range(N):
            for i in range(j + 1):
                blk = S[2 * i:2 * i + 2, 2 * j:2 * j + 2]
                assert np.array_equal(vis[f, tri(i, j)], blk)


# --- Hermitian symmetry of the full matrix and triangle = full ------------------

def test_full_matrix_hermitian_and_triangle_consistent():
    N, F, T = 7, 3, 40
    x = wl.full_range(N, F, T, 21)
    vis = xo.correlate_i8(x)
    for f in range(F):
        full = xo.full_i8(x, f)                         # [2N][2N][2]
        assert np.array_equal(full[..., 0], full[..., 0].T)          # Re symmetric
        assert np.array_equal(full[..., 1], -full[..., 1].T)         # Im antisymmetric
        for j in range(N):
            for i in range(j + 1):
                assert np.array_equal(vis[f, tri(i, j)].astype(np.int64),
                                      full[2 * i:2 * i + 2, 2 * j:2 * j + 2])


def test_single_baseline_entry_point_matches():
    N, F, T = 6, 2, 17
    x = wl.full_range(N, F, T, 22)
    vis = xo.correlate_i8(x)
    for f in range(F):
        for j in range(N):
            for i in range(N):
                b = xo.baseline_i8(x, f, i, j)
                if i <= j:
                    assert np.array_equal(b, vis[f, tri(i, j)])
                else:   # upper triangle = conjugate transpose of the stored lower entry
                    low = vis[f, tri(j, i)].astype(np.int64)
                    assert np.array_equal(b[..., 0], low[..., 0].T)
                    assert np.array_equal(b[..., 1], -low[..., 1].T)


# --- autocorrelations ("auto-correlation of self pairs along the diagonal") -------

def test_autocorrelations_real_and_sum_abs2():
    N, F, T = 9, 2, 64
    x = wl.full_range(N, F, T, 31)
    vis = xo.correlate_i8(x)
    p2 = (x.astype(np.int64) ** 2).sum(axis=-1).sum(axis=0)        # [F][N][2]  sum_t |x|^2
    for f in range(F):
        for i in range(N):
            v = vis[f, tri(i, i)]
            for p in range(2):
                assert v[p, p, 1] == 0
                assert v[p, p, 0] == p2[f, i, p]
            assert v[0, 1, 0] == v[1, 0, 0] and v[0, 1, 1] == -v[1, 0, 1]


# --- common tone: rank 1, known magnitude and phase (fixes the conjugation side, R1) ----------

def test_common_tone_rank1_phase():
    N, F, T, A = 6, 3, 50, 3
    x, wq = wl.common_tone(N, F, T, 41, A)
    vis = vis_to_complex(xo.correlate_i8(x))
    w = np.array([1, 1j, -1, -1j])[wq]                             # [F][N][2]
    for f in range(F):
        for j in range(N):
            for i in range(j + 1):
                for pi in range(2):
                    for pj in range(2):
                        exp = T * A * A * w[f, i, pi] * np.conj(w[f, j, pj])   # arg = phi_i - phi_j
                        assert vis[f, tri(i, j), pi, pj] == exp


# --- linearity in time / accumulate mode -----------------------------------

def test_time_split_accumulate():
    N, F, T = 8, 3, 90
    x = wl.full_range(N, F, T, 51)
    whole = xo.correlate_i8(x)
    part = xo.correlate_i8(x[:31])
    part = xo.correlate_i8(x[31:64], vis_prev=part)
    part = xo.correlate_i8(x[64:], vis_prev=part)
    assert np.array_equal(whole, part)
    assert np.array_equal(xo.correlate_i8(x[:0]), np.zeros_like(whole))     # T = 0: empty sum


# --- channel independence -------------------------------------------------------

def test_channel_independence():
    N, F, T = 5, 6, 20
    x = wl.full_range(N, F, T, 61)
    vis = xo.correlate_i8(x)
    perm = np.array([3, 0, 5, 1, 4, 2])
    assert np.array_equal(xo.correlate_i8(x[:, perm]), vis[perm])
    assert np.array_equal(xo.channels_i8(x, [5, 0, 2]), vis[[5, 0, 2]])
    assert np.array_equal(xo.correlate_i8(x[:, 2:3]), vis[2:3])


# --- int32 range (reading R7) -----------------------------------------------------------------

def test_overflow_is_detected_and_edge_fits():
    # 2 * 128^2 * T: T = 65535 fits int32, T = 65536 does not.
    x = np.full((65536, 1, 1, 2, 2), -128, np.int8)
    v = xo.correlate_i8(x[:65535])
    assert v[0, 0, 0, 0, 0] == 2 * 128 * 128 * 65535
    with pytest.raises(xo.OracleError) as e:
        xo.correlate_i8(x)
    assert e.value.code == xo.XO_ERR_OVERFLOW


# --- float oracle -----------------------------------------------------------------------------

def test_float_oracle_equals_int_oracle_on_integer_valued_input():
    N, F, T = 6, 2, 77
    x = wl.full_range(N, F, T, 71)
    vi = xo.correlate_i8(x)
    vf = xo.channels_f64(x.astype(np.float32))
    assert np.array_equal(vf, vi.astype(np.float64))


def test_float_oracle_equals_numpy_complex128():
    N, F, T = 5, 2, 40
    rng = np.random.default_rng(72)
    x = rng.standard_normal((T, F, N, 2, 2)).astype(np.float32)
    vf = xo.channels_f64(x)
    z = (x[..., 0].astype(np.float64) + 1j * x[..., 1].astype(np.float64)).reshape(T, F, 2 * N)
    for f in range(F):
        S = np.einsum("ta,tb->ab", z[:, f], z[:, f].conj())
        for j in range(N):
            for i in range(j + 1):
                got = vf[f, tri(i, j), ..., 0] + 1j * vf[f, tri(i, j), ..., 1]
                np.testing.assert_allclose(got, S[2 * i:2 * i + 2, 2 * j:2 * j + 2], rtol=1e-12, atol=1e-12)


# --- statistics (sanity, not parity) ----------------------------------------------------------

def test_gaussian_statistics():
    N, F, T, sigma = 8, 4, 4000, 4.0
    x = wl.gaussian(N, F, T, 81, sigma)
    vis = xo.correlate_i8(x).astype(np.float64)
    auto = np.array([vis[f, tri(i, i), p, p, 0] for f in range(F) for i in range(N) for p in range(2)])
    exp = 2 * T * (sigma ** 2 + 1.0 / 12.0)
    assert abs(auto.mean() / exp - 1) < 0.02
    cross = np.array([vis[f, tri(i, j), :, :, :].ravel() for f in range(F) for j in range(N) for i in range(j)])
    assert abs(cross.mean()) < 0.1 * sigma ** 2 * np.sqrt(2 * T)
    assert abs(cross.std() / (sigma ** 2 * np.sqrt(2 * T)) - 1) < 0.1


def test_config3_tone_structure():
    """Config 3's recipe: off-diagonal V ~ amp^2 * T * exp(i(phi_i - phi_j)) above the noise."""
    N, F, T = 32, 2, 1000
    x = wl.gaussian_tone(N, F, T, 1003)
    vis = vis_to_complex(xo.correlate_i8(x))
    phi = 2 * np.pi * 5 * np.arange(N) / N
    num = den = 0.0
    for j in range(N):
        for i in range(j):
            num += (vis[:, tri(i, j), 0, 0] * np.exp(-1j * (phi[i] - phi[j]))).sum()
            den += F
    mean = num / den
    assert abs(mean.real / (4 * T) - 1) < 0.1 and abs(mean.imag) < 0.1 * 4 * T


def test_wide_oracle_long_integration():
    """Long integrations: the int64 entry point equals the int32 one where that fits, equals
    numpy's complex x x^H beyond it, and reaches the closed form 2 * 128^2 * T for all -128 input where int32 overflows."""
    x = wl.full_range(6, 3, 50, seed=21)
    assert np.array_equal(xo.channels_i8_wide(x), xo.correlate_i8(x).astype(np.int64))
    assert np.array_equal(xo.channels_i8_wide(x, [2, 0]), xo.correlate_i8(x).astype(np.int64)[[2, 0]])
    T = 70000                                                  # > XC_MAX_T: 2 * 128^2 * T = 2 293 760 000 > 2^31
    big = np.full((T, 1, 2, 2, 2), -128, np.int8)
    w = xo.channels_i8_wide(big)
    assert w[0, :, :, :, 0].min() == w[0, :, :, :, 0].max() == 2 * 128 * 128 * T > 2 ** 31
    assert (w[..., 1] == 0).all()
    with pytest.raises(xo.OracleError):
        xo.correlate_i8(big)
    # random long block against numpy (complex128 is exact here: |sums| < 2^53)
    y = wl.full_range(3, 2, 66000, seed=22)
    z = y.astype(np.float64)
    zc = (z[..., 0] + 1j * z[..., 1]).reshape(66000, 2, 6)      # [t][f][(s,p)]
    ref = np.einsum("tfa,tfb->fab", zc, zc.conj())
    w = xo.channels_i8_wide(y)
    for j in range(3):
        for i in range(j + 1):
            for pi in range(2):
                for pj in range(2):
                    v = ref[:, 2 * i + pi, 2 * j + pj]
                    b = j * (j + 1) // 2 + i
                    assert np.array_equal(w[:, b, pi, pj, 0], np.rint(v.real).astype(np.int64))
                    assert np.array_equal(w[:, b, pi, pj, 1], np.rint(v.imag).astype(np.int64))


def test_unpack_i4_all_codes_and_hand_example():
    """4-bit format (reading 17): low nibble real, high nibble imaginary, two's complement.  All 256 byte
    codes against Python integer arithmetic; one product by hand: byte 0x2F = (-1 + 2i), byte 0x9A = (-6 - 7i):
    (-1 + 2i) conj(-6 - 7i) = (-1 + 2i)(-6 + 7i) = 6 - 7i - 12i - 14 = -8 - 19i."""
    codes = np.arange(256, dtype=np.uint8).reshape(256, 1, 1, 1).repeat(2, axis=3)
    got = xo.unpack_i4(codes)
    for b in range(256):
        re = (b & 15) - 16 if (b & 15) >= 8 else (b & 15)
        im = (b >> 4) - 16 if (b >> 4) >= 8 else (b >> 4)
        assert tuple(got[b, 0, 0, 0]) == (re, im) and tuple(got[b, 0, 0, 1]) == (re, im)
    assert got.min() == -8 and got.max() == 7
    x4 = np.zeros((1, 1, 2, 2), np.uint8)
    x4[0, 0, 0, 0] = 0x2F
    x4[0, 0, 1, 0] = 0x9A
    v = xo.correlate_i4(x4)
    assert tuple(v[0, 1, 0, 0]) == (-8, -19)                  # baseline (i=0, j=1), pols (0, 0)
    assert tuple(v[0, 0, 0, 0]) == (5, 0) and tuple(v[0, 2, 0, 0]) == (85, 0)   # |-1+2i|^2, |-6-7i|^2
    x = wl.packed_i4(5, 2, 40, seed=4)
    assert np.array_equal(xo.correlate_i4(x), xo.correlate_i8(xo.unpack_i4(x)))
    assert xo.unpack_i4(x)[0, 0, 0].tolist() == [[-8, -8], [7, 7]]
