"""ctypes loader for the CPU oracle (oracle/xo_oracle.c).  TEST INFRASTRUCTURE, NOT PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It imports nothing from the product package and the product package
imports nothing from here.  Arguments are numpy arrays (host memory); every function returns
a fresh numpy array.  Definitions and citations are in xo_oracle.c's header.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "xo_oracle.c")
_LIB = os.path.join(_HERE, "libxo_oracle.so")

XO_OK, XO_ERR_ARG, XO_ERR_OVERFLOW, XO_ERR_NOMEM = 0, -1, -3, -7


class OracleError(RuntimeError):
    def __init__(self, code: int, where: str):
        super().__init__(f"{where}: oracle returned {code}")
        self.code = code


def build(force: bool = False) -> str:
    """Compile xo_oracle.c -> libxo_oracle.so with gcc -O2 -fopenmp (plain C, no intrinsics)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fopenmp", "-shared", "-fPIC", "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        i, p = ctypes.c_int, ctypes.c_void_p
        L.xo_num_threads.restype = i
        L.xo_set_num_threads.argtypes = [i]
        L.xo_channel_i8.argtypes = [p, i, i, i, i, p, i]
        L.xo_correlate_i8.argtypes = [p, i, i, i, p, i]
        L.xo_channels_i8.argtypes = [p, i, i, i, p, i, p]
        L.xo_channels_i8_wide.argtypes = [p, i, i, i, p, i, p]
        L.xo_baseline_i8.argtypes = [p, i, i, i, i, i, i, p]
        L.xo_full_i8.argtypes = [p, i, i, i, i, p]
        L.xo_channel_f64.argtypes = [p, i, i, i, i, p]
        L.xo_channels_f64.argtypes = [p, i, i, i, p, i, p]
        for name in ("xo_channel_i8", "xo_correlate_i8", "xo_channels_i8", "xo_channels_i8_wide", "xo_baseline_i8",
                     "xo_full_i8", "xo_channel_f64", "xo_channels_f64"):
            getattr(L, name).restype = i
        _lib = L
    return _lib


def num_threads() -> int:
    return int(lib().xo_num_threads())


def set_num_threads(n: int) -> None:
    lib().xo_set_num_threads(int(n))


def n_baselines(N: int) -> int:
    """1/2 N (N+1) station pairs including autocorrelations."""
    return N * (N + 1) // 2


def _check_in(x: np.ndarray, dtype) -> tuple[np.ndarray, int, int, int]:
    if x.dtype != dtype or x.ndim != 5 or x.shape[3:] != (2, 2):
        raise ValueError(f"input must be {dtype} [T][F][N][2][2], got {x.dtype} {x.shape}")
    x = np.ascontiguousarray(x)
    T, F, N = x.shape[:3]
    return x, N, F, T


def _ptr(a: np.ndarray) -> ctypes.c_void_p:
    return ctypes.c_void_p(a.ctypes.data)


def correlate_i8(x: np.ndarray, vis_prev: np.ndarray | None = None) -> np.ndarray:
    """All channels. x: int8 [T][F][N][2][2] -> int32 [F][NB][2][2][2]; adds to vis_prev if given."""
    x, N, F, T = _check_in(x, np.int8)
    NB = n_baselines(N)
    if vis_prev is None:
        vis = np.empty((F, NB, 2, 2, 2), np.int32)
        acc = 0
    else:
        vis = np.array(vis_prev, dtype=np.int32, copy=True).reshape(F, NB, 2, 2, 2)
        acc = 1
    rc = lib().xo_correlate_i8(_ptr(x), N, F, T, _ptr(vis), acc)
    if rc != XO_OK:
        raise OracleError(rc, "xo_correlate_i8")
    return vis


def channels_i8(x: np.ndarray, fsel) -> np.ndarray:
    """Chosen channels only -> int32 [len(fsel)][NB][2][2][2]."""
    x, N, F, T = _check_in(x, np.int8)
    fs = np.ascontiguousarray(np.asarray(fsel, dtype=np.int32))
    vis = np.empty((len(fs), n_baselines(N), 2, 2, 2), np.int32)
    rc = lib().xo_channels_i8(_ptr(x), N, F, T, _ptr(fs), len(fs), _ptr(vis))
    if rc != XO_OK:
        raise OracleError(rc, "xo_channels_i8")
    return vis


def channels_i8_wide(x: np.ndarray, fsel=None) -> np.ndarray:
    """Long integrations: chosen channels (default all) with int64 sums and no int32 check
    -> int64 [len(fsel)][NB][2][2][2]; x holds the whole integration (blocks concatenated along t)."""
    x, N, F, T = _check_in(x, np.int8)
    fs = np.ascontiguousarray(np.asarray(range(F) if fsel is None else fsel, dtype=np.int32))
    vis = np.empty((len(fs), n_baselines(N), 2, 2, 2), np.int64)
    rc = lib().xo_channels_i8_wide(_ptr(x), N, F, T, _ptr(fs), len(fs), _ptr(vis))
    if rc != XO_OK:
        raise OracleError(rc, "xo_channels_i8_wide")
    return vis


def unpack_i4(x4: np.ndarray) -> np.ndarray:
    """4-bit complex samples ("typically four to eight bits of precision is sufficient"; two's complement,
    PAPER.md:45).  The paper fixes no packing; reading 17: one byte per complex sample, LOW nibble = real part,
    HIGH nibble = imaginary part, each a two's-complement 4-bit integer in [-8, 7].
    x4: uint8 [T][F][N][2 pol] -> int8 [T][F][N][2][2 re,im].  Written out per nibble: value = n if n < 8 else n - 16."""
    x4 = np.ascontiguousarray(x4)
    if x4.dtype != np.uint8 or x4.ndim != 4 or x4.shape[3] != 2:
        raise ValueError("packed input must be uint8 [T][F][N][2]")
    lo = (x4 & np.uint8(0x0F)).astype(np.int16)
    hi = (x4 >> np.uint8(4)).astype(np.int16)
    re = np.where(lo < 8, lo, lo - 16)
    im = np.where(hi < 8, hi, hi - 16)
    return np.stack([re, im], axis=-1).astype(np.int8)


def correlate_i4(x4: np.ndarray) -> np.ndarray:
    """Eq. 4 on 4-bit samples: unpack, then the int8 definition.  -> int32 [F][NB][2][2][2]."""
    return correlate_i8(unpack_i4(x4))


def baseline_i8(x: np.ndarray, f: int, i: int, j: int) -> np.ndarray:
    """One station pair (any i, j) of one channel -> int64 [2][2][2]."""
    x, N, F, T = _check_in(x, np.int8)
    out = np.empty((2, 2, 2), np.int64)
    rc = lib().xo_baseline_i8(_ptr(x), N, F, T, int(f), int(i), int(j), _ptr(out))
    if rc != XO_OK:
        raise OracleError(rc, "xo_baseline_i8")
    return out


def full_i8(x: np.ndarray, f: int) -> np.ndarray:
    """Full 2N x 2N matrix of one channel as complex int64 pairs -> int64 [2N][2N][2]."""
    x, N, F, T = _check_in(x, np.int8)
    out = np.empty((2 * N, 2 * N, 2), np.int64)
    rc = lib().xo_full_i8(_ptr(x), N, F, T, int(f), _ptr(out))
    if rc != XO_OK:
        raise OracleError(rc, "xo_full_i8")
    return out


def channels_f64(x: np.ndarray, fsel=None) -> np.ndarray:
    """Float-input oracle with fp64 products and sums -> float64 [len(fsel)][NB][2][2][2]."""
    x, N, F, T = _check_in(x, np.float32)
    fs = np.ascontiguousarray(np.arange(F, dtype=np.int32) if fsel is None else np.asarray(fsel, dtype=np.int32))
    vis = np.empty((len(fs), n_baselines(N), 2, 2, 2), np.float64)
    rc = lib().xo_channels_f64(_ptr(x), N, F, T, _ptr(fs), len(fs), _ptr(vis))
    if rc != XO_OK:
        raise OracleError(rc, "xo_channels_f64")
    return vis
