"""ctypes loader for the F-engine CPU oracle (oracle/fo_oracle.c).  TEST INFRASTRUCTURE, NOT PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline legs may import this module.  It imports nothing from
the product package and the product package imports nothing from here.  Definitions, readings and citations are in
fo_oracle.c's header.  Arguments are numpy arrays (host memory); every function returns fresh numpy arrays.

Layouts: volt int8 [N][2 pol][T*F samples][2 re,im] (station-major time series);
         cube / spec / margin [T][F][N][2][2] (the X-engine's input order).
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "fo_oracle.c")
_LIB = os.path.join(_HERE, "libfo_oracle.so")


class OracleError(RuntimeError):
    def __init__(self, code: int, where: str):
        super().__init__(f"{where}: oracle returned {code}")
        self.code = code


def build(force: bool = False) -> str:
    """gcc -O2 -ffp-contract=off: plain C; no FMA contraction, so that the arithmetic is the one written down."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-o", tmp, _SRC,
                               "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        i, p, f32, sz = ctypes.c_int, ctypes.c_void_p, ctypes.c_float, ctypes.c_size_t
        L.fo_num_threads.restype = i
        L.fo_twiddle_f64.argtypes = [i, i, p]
        L.fo_spectrum_i8.argtypes = [p, i, i, i, i, i, i, p]
        L.fo_spectra_i8.argtypes = [p, i, i, i, p, i, p]
        L.fo_fengine_i8.argtypes = [p, i, i, i, f32, p, p, p]
        L.fo_quantise_f64.argtypes = [p, sz, f32, p]
        L.fo_margin_f64.argtypes = [p, sz, f32, p]
        for n in ("fo_twiddle_f64", "fo_spectrum_i8", "fo_spectra_i8", "fo_fengine_i8", "fo_quantise_f64", "fo_margin_f64"):
            getattr(L, n).restype = i
        _lib = L
    return _lib


def num_threads() -> int:
    return int(lib().fo_num_threads())


def _ptr(a):
    return ctypes.c_void_p(a.ctypes.data) if a is not None else None


def _check_volt(volt, F):
    v = np.ascontiguousarray(volt)
    if v.dtype != np.int8 or v.ndim != 4 or v.shape[1] != 2 or v.shape[3] != 2 or v.shape[2] % F:
        raise ValueError("volt must be int8 [N][2][T*F][2]")
    return v, v.shape[0], v.shape[2] // F


def twiddle(F: int, m: int) -> complex:
    out = np.empty(2, np.float64)
    rc = lib().fo_twiddle_f64(F, m, _ptr(out))
    if rc:
        raise OracleError(rc, "fo_twiddle_f64")
    return complex(out[0], out[1])


def spectrum(volt: np.ndarray, F: int, s: int, p: int, t: int) -> np.ndarray:
    """complex128 [F]: the spectrum of station s, pol p, time block t."""
    v, N, T = _check_volt(volt, F)
    X = np.empty((F, 2), np.float64)
    rc = lib().fo_spectrum_i8(_ptr(v), N, F, T, s, p, t, _ptr(X))
    if rc:
        raise OracleError(rc, "fo_spectrum_i8")
    return X[:, 0] + 1j * X[:, 1]


def spectra(volt: np.ndarray, F: int, sel) -> np.ndarray:
    """complex128 [len(sel)][F] for sel = [(s, p, t), ...]."""
    v, N, T = _check_volt(volt, F)
    sel = np.ascontiguousarray(np.asarray(sel, dtype=np.int32).reshape(-1, 3))
    X = np.empty((len(sel), F, 2), np.float64)
    rc = lib().fo_spectra_i8(_ptr(v), N, F, T, _ptr(sel), len(sel), _ptr(X))
    if rc:
        raise OracleError(rc, "fo_spectra_i8")
    return X[..., 0] + 1j * X[..., 1]


def fengine(volt: np.ndarray, F: int, scale: float, want_spec: bool = False):
    """(cube int8 [T][F][N][2][2], margin float32 same shape[, spec float64 same shape])."""
    v, N, T = _check_volt(volt, F)
    cube = np.empty((T, F, N, 2, 2), np.int8)
    margin = np.empty((T, F, N, 2, 2), np.float32)
    spec = np.empty((T, F, N, 2, 2), np.float64) if want_spec else None
    rc = lib().fo_fengine_i8(_ptr(v), N, F, T, np.float32(scale), _ptr(spec), _ptr(cube), _ptr(margin))
    if rc:
        raise OracleError(rc, "fo_fengine_i8")
    return (cube, margin, spec) if want_spec else (cube, margin)


def quantise(X: np.ndarray, scale: float) -> np.ndarray:
    X = np.ascontiguousarray(X, dtype=np.float64)
    q = np.empty(X.shape, np.int8)
    rc = lib().fo_quantise_f64(_ptr(X), X.size, np.float32(scale), _ptr(q))
    if rc:
        raise OracleError(rc, "fo_quantise_f64")
    return q


def margin(X: np.ndarray, scale: float) -> np.ndarray:
    """float32 margins (reading 21) of the given fp64 values, for the pins."""
    X = np.ascontiguousarray(X, dtype=np.float64)
    m = np.empty(X.shape, np.float32)
    rc = lib().fo_margin_f64(_ptr(X), X.size, np.float32(scale), _ptr(m))
    if rc:
        raise OracleError(rc, "fo_margin_f64")
    return m
