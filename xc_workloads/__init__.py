"""Seeded synthetic voltage data for the X-engine (shared by tests, bench and the oracle legs).

This module holds NONE of the method's arithmetic: it only draws samples.  It is the one
module both the CUDA path's callers and the oracle's callers may import (neither of those
two imports the other).  All generators are host-side numpy (`numpy.random.default_rng(seed)`,
PCG64) so the oracle and the GPU receive the very same bytes.

Layout of every array: int8 [T][F][N][2 pol][2 re,im]  (station fastest, then frequency, then
time: Sec. 4.1 "the corner turn has been applied").

The paper measures on no public dataset and does not say what its input buffers held
(SURVEY.md 8(d)); these inputs take the SHAPES of its workloads (N up to 512-2048 dual-pol
stations, 8-bit samples, I ~ 1024-2048, fixed F*I: PAPER.md:190, 263, 283, 341) and the value
distributions BASELINE.json's `configs` name.  Rounding is round-half-to-even (rint), then clip.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

__all__ = ["Workload", "CONFIGS", "SWEEP_N", "make_input", "make_blocks", "uniform_small",
           "gaussian", "gaussian_tone", "common_tone", "full_range", "packed_i4", "voltages", "fengine_scale"]


@dataclass(frozen=True)
class Workload:
    name: str
    N: int
    F: int
    T: int
    kind: str          # "uniform" | "gauss" | "gauss_tone"
    sigma: float
    seed: int

    @property
    def NB(self) -> int:
        return self.N * (self.N + 1) // 2

    @property
    def in_bytes(self) -> int:
        return 4 * self.N * self.F * self.T

    @property
    def vis_bytes(self) -> int:
        return 32 * self.NB * self.F

    @property
    def cmacs(self) -> int:
        """Complex MACs counted by Eq. 5: 1/2 * 2N(2N+1) per sample per channel."""
        return self.F * self.T * self.N * (2 * self.N + 1)

    @property
    def ops(self) -> int:
        return 8 * self.cmacs


SWEEP_N = (32, 64, 100, 500, 1024)

CONFIGS: dict[str, Workload] = {
    "cfg1": Workload("cfg1", 16, 4, 256, "uniform", 0.0, 1001),
    "cfg2": Workload("cfg2", 128, 1024, 1000, "gauss", 4.0, 1002),
    "cfg3": Workload("cfg3", 256, 512, 1000, "gauss_tone", 4.0, 1003),
    "cfg4": Workload("cfg4", 512, 256, 1000, "gauss", 16.0, 1004),
}
for _k, _n in enumerate(SWEEP_N):
    CONFIGS[f"cfg5_N{_n}"] = Workload(f"cfg5_N{_n}", _n, 64, 2048, "gauss", 4.0, 1050 + _k)


def _quantise(x: np.ndarray, lo: int, hi: int) -> np.ndarray:
    return np.clip(np.rint(x), lo, hi).astype(np.int8)


def uniform_small(N: int, F: int, T: int, seed: int, lo: int = -8, hi: int = 7) -> np.ndarray:
    """re, im i.i.d. uniform integers in [lo, hi] (config 1)."""
    rng = np.random.default_rng(seed)
    return rng.integers(lo, hi + 1, size=(T, F, N, 2, 2), dtype=np.int8)


def gaussian(N: int, F: int, T: int, seed: int, sigma: float, t_chunk: int = 64) -> np.ndarray:
    """clip(rint(N(0, sigma^2)), -127, 127) per real component (configs 2, 4, 5)."""
    rng = np.random.default_rng(seed)
    out = np.empty((T, F, N, 2, 2), np.int8)
    for t0 in range(0, T, t_chunk):
        t1 = min(T, t0 + t_chunk)
        g = rng.standard_normal(size=(t1 - t0, F, N, 2, 2), dtype=np.float32)
        out[t0:t1] = _quantise(g * np.float32(sigma), -127, 127)
    return out


def gaussian_tone(N: int, F: int, T: int, seed: int, sigma: float = 4.0, amp: float = 2.0,
                  turns: float = 5.0, t_chunk: int = 64) -> np.ndarray:
    """Noise + a common sky tone (config 3): n + amp * exp(i(theta_{t,f} + phi_s)); theta i.i.d.
    uniform per (t,f), common to all stations and both pols; phi_s = 2 pi * turns * s / N."""
    rng = np.random.default_rng(seed)
    out = np.empty((T, F, N, 2, 2), np.int8)
    phi = (2.0 * np.pi * turns * np.arange(N) / N).astype(np.float32)
    for t0 in range(0, T, t_chunk):
        t1 = min(T, t0 + t_chunk)
        g = rng.standard_normal(size=(t1 - t0, F, N, 2, 2), dtype=np.float32) * np.float32(sigma)
        theta = rng.random(size=(t1 - t0, F), dtype=np.float32) * np.float32(2.0 * np.pi)
        ph = theta[:, :, None] + phi[None, None, :]
        g[..., 0] += np.float32(amp) * np.cos(ph)[..., None]
        g[..., 1] += np.float32(amp) * np.sin(ph)[..., None]
        out[t0:t1] = _quantise(g, -127, 127)
    return out


def common_tone(N: int, F: int, T: int, seed: int, A: int = 3):
    """Every station/pol carries A * u_t * w_{s,p} with u, w in {1, i, -1, -i} (exact in int8).
    Returns (x, wq) with wq[f][s][p] in {0,1,2,3} the quarter-turn phase of w."""
    rng = np.random.default_rng(seed)
    uq = rng.integers(0, 4, size=(T, F))
    wq = rng.integers(0, 4, size=(F, N, 2))
    q = (uq[:, :, None, None] + wq[None]) % 4
    re = np.array([1, 0, -1, 0])[q]
    im = np.array([0, 1, 0, -1])[q]
    x = np.stack([re, im], axis=-1) * A
    return x.astype(np.int8), wq


def full_range(N: int, F: int, T: int, seed: int) -> np.ndarray:
    """Uniform over the whole int8 range including -128, with -128 forced into every position
    class (re/im x pol) somewhere (SURVEY.md 8(c) reading 6)."""
    rng = np.random.default_rng(seed)
    x = rng.integers(-128, 128, size=(T, F, N, 2, 2), dtype=np.int8)
    if T > 0:
        x[0, :, :, :, :] = -128
        x[T - 1, :, 0, :, :] = -128
    return x


def make_input(w: Workload, T: int | None = None, seed: int | None = None) -> np.ndarray:
    T = w.T if T is None else T
    seed = w.seed if seed is None else seed
    if w.kind == "uniform":
        return uniform_small(w.N, w.F, T, seed)
    if w.kind == "gauss":
        return gaussian(w.N, w.F, T, seed, w.sigma)
    if w.kind == "gauss_tone":
        return gaussian_tone(w.N, w.F, T, seed, w.sigma)
    raise ValueError(w.kind)


def make_blocks(w: Workload, n_blocks: int, seed0: int = 1060) -> list[np.ndarray]:
    """Config 5's two-stream run: n_blocks input blocks of w's shape, seeds seed0 + k."""
    return [make_input(w, seed=seed0 + k) for k in range(n_blocks)]


def packed_i4(N: int, F: int, T: int, seed: int) -> np.ndarray:
    """4-bit complex samples, one byte per (t, f, station, pol): uniform random bytes, i.e. both nibbles uniform over
    all 16 codes, with the codes 0x8 (-8) and 0x7 (+7) forced into every nibble position class of the first row.
    uint8 [T][F][N][2].  No arithmetic of the method here: the two sides each decode the nibbles themselves."""
    rng = np.random.default_rng(seed)
    x = rng.integers(0, 256, size=(T, F, N, 2), dtype=np.uint8)
    x[0, 0, 0, 0] = 0x88
    x[0, 0, 0, 1] = 0x77
    if T > 1:
        x[1, 0, 0, 0] = 0x78
        x[1, 0, 0, 1] = 0x87
    return x


def voltages(N: int, F: int, T: int, seed: int, sigma: float = 16.0, tones: int = 2, amp: float = 12.0,
             full_range_mix: bool = False) -> np.ndarray:
    """Time-domain station voltages for the F-engine in front of the X-engine: complex int8, station-major,
    int8 [N][2 pol][T*F samples][2 re,im] ("the voltage time-series from each antenna ... digitized").
    Gaussian noise of `sigma` per real component plus `tones` sky tones common to all stations (bin-centred on seeded
    channels of an F-point transform, station-dependent fixed phase, fresh random phase per time block so that the tone is
    coherent between stations but not in time), rounded half to even and clipped to [-127, 127].  full_range_mix
    replaces one signal in eight by uniform samples over the whole int8 range (-128 included).  Only draws samples: the
    transform itself is the oracle's and the library's business."""
    rng = np.random.default_rng(seed)
    out = np.empty((N, 2, T * F, 2), np.int8)
    f_tone = rng.integers(0, F, size=max(tones, 0))
    phi = rng.random(size=(max(tones, 0), N)).astype(np.float32) * np.float32(2 * np.pi)
    k = np.arange(F, dtype=np.float32)
    for s in range(N):
        g = rng.standard_normal(size=(2, T, F, 2), dtype=np.float32) * np.float32(sigma)
        for j in range(len(f_tone)):
            theta = np.random.default_rng(seed * 1000003 + j).random(size=T).astype(np.float32) * np.float32(2 * np.pi)
            ph = (np.float32(2 * np.pi) * np.float32(f_tone[j]) * k / np.float32(F))[None, :] + theta[:, None] + phi[j, s]
            g[:, :, :, 0] += np.float32(amp) * np.cos(ph)[None]
            g[:, :, :, 1] += np.float32(amp) * np.sin(ph)[None]
        out[s] = _quantise(g, -127, 127).reshape(2, T * F, 2)
        if full_range_mix and s % 8 == 3:
            out[s, s % 2] = rng.integers(-128, 128, size=(T * F, 2), dtype=np.int8)
    return out


def fengine_scale(F: int, sigma: float = 16.0, target: float = 8.0) -> float:
    """A power-of-two output scale for the F-engine's quantiser such that Gaussian input of `sigma` per component gives
    channel samples of about `target` per component (the spectrum grows like sigma * sqrt(F))."""
    return float(2.0 ** np.round(np.log2(target / (sigma * np.sqrt(F)))))
