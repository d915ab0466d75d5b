"""ctypes loader for oracle/hs_oracle_ext.c — TEST INFRASTRUCTURE, NOT THE PRODUCT.

The three "next" rows of SURVEY.md section 8(f): every integer H up to 64 and eq. 2's window as printed,
the normalised power spectrum of a complex Fourier series, and the two-dimensional harmonic sum over the
f - fdot plane.  All arithmetic lives in hs_oracle_ext.c; this file builds it (gcc -O2 -ffp-contract=off)
and marshals NumPy arrays.  Only tests/, __graft_entry__.smoke() and bench.py's CPU legs may import it; it never
imports paper_1812_02647_b200.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "hs_oracle_ext.c")
_LIB = os.path.join(_HERE, "libhs_oracle_ext.so")

STANDARD, MAX, FREQBIN, GREEDY = 0, 1, 2, 3
VARIANTS = {"standard": STANDARD, "max": MAX, "freqbin": FREQBIN, "greedy": GREEDY}
WINDOWS = {"c2": 0, "printed": 1, "interp": 2}      # "interp": eq. 1 with linearly interpolated terms (C15)

_lib = None


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-std=c99", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-Wall", "-Wextra",
                               "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        i64, p, i, f = ctypes.c_int64, ctypes.c_void_p, ctypes.c_int, ctypes.c_float
        lib.hsx_partial_sum.argtypes = [p, i64, i64, i, i, i, p]
        lib.hsx_partial_sum.restype = ctypes.c_double
        lib.hsx_harmonic_sum_all.argtypes = [p, i64, i64, i, i, i, p, p, p, p, p, p]
        lib.hsx_harmonic_sum_all.restype = i
        lib.hsx_points_all.argtypes = [p, i64, i64, i, i, i, i64, p, p, p, p]
        lib.hsx_points_all.restype = i
        lib.hsx_power_spectrum.argtypes = [p, i64, f, p]
        lib.hsx_power_spectrum.restype = i
        lib.hsx_partial_sum_2d.argtypes = [p, i64, i64, i64, i64, i, i]
        lib.hsx_partial_sum_2d.restype = ctypes.c_double
        lib.hsx_harmonic_sum_2d.argtypes = [p, i64, i64, i64, i, i, p, p, p, p, p]
        lib.hsx_harmonic_sum_2d.restype = i
        _lib = lib
    return _lib


def _v(v):
    return VARIANTS[v] if isinstance(v, str) else int(v)


def _w(w):
    return WINDOWS[w] if isinstance(w, str) else int(w)


def _batch(x):
    x = np.ascontiguousarray(x, dtype=np.float32)
    if x.ndim == 1:
        x = x[None, :]
    assert x.ndim == 2
    return x


def partial_sum(x, n: int, H: int, variant, window="c2"):
    x = np.ascontiguousarray(x, dtype=np.float32)
    j = ctypes.c_int(0)
    S = _load().hsx_partial_sum(x.ctypes.data, x.shape[0], int(n), int(H), _v(variant), _w(window), ctypes.byref(j))
    return S, j.value


def harmonic_sum_all(x, Hmax: int, variant, window="c2", want_sums=True, want_reduced=True, want_jpath=False) -> dict:
    """Every integer H = 1..Hmax (level index H - 1): sums[B][Hmax][N], max, argmax, gap, second, jpath."""
    x = _batch(x)
    B, N = x.shape
    out = {}
    if want_sums:
        out["sums"] = np.empty((B, Hmax, N), np.float64)
    if want_reduced:
        out["max"] = np.empty((B, N), np.float64)
        out["argmax"] = np.empty((B, N), np.uint8)
        out["gap"] = np.empty((B, N), np.float64)
        out["second"] = np.empty((B, N), np.uint8)
    if want_jpath:
        out["jpath"] = np.empty((B, Hmax, N), np.uint8)
    g = lambda k: out[k].ctypes.data if k in out else None
    rc = _load().hsx_harmonic_sum_all(x.ctypes.data, N, B, int(Hmax), _v(variant), _w(window), g("sums"), g("max"),
                                      g("argmax"), g("gap"), g("second"), g("jpath"))
    if rc:
        raise ValueError("hsx_harmonic_sum_all: invalid arguments")
    return out


def points_all(x, Hmax: int, variant, bidx, nidx, window="c2"):
    x = _batch(x)
    B, N = x.shape
    bidx = np.ascontiguousarray(bidx, dtype=np.int64)
    nidx = np.ascontiguousarray(nidx, dtype=np.int64)
    P = bidx.shape[0]
    h = np.empty((P, Hmax), np.float64)
    j = np.empty((P, Hmax), np.uint8)
    rc = _load().hsx_points_all(x.ctypes.data, N, B, int(Hmax), _v(variant), _w(window), P, bidx.ctypes.data,
                                nidx.ctypes.data, h.ctypes.data, j.ctypes.data)
    if rc:
        raise ValueError("hsx_points_all: invalid arguments")
    return h, j


def power_spectrum(F, scale: float) -> np.ndarray:
    """x = (re^2 + im^2) * scale - 1 in fp32, each operation rounded separately.  F: complex64 array or float32 [..., 2]."""
    F = np.ascontiguousarray(F)
    if np.iscomplexobj(F):
        F = np.ascontiguousarray(F.astype(np.complex64)).view(np.float32).reshape(F.shape + (2,))
    F = np.ascontiguousarray(F, dtype=np.float32)
    assert F.shape[-1] == 2
    x = np.empty(F.shape[:-1], np.float32)
    rc = _load().hsx_power_spectrum(F.ctypes.data, x.size, ctypes.c_float(scale), x.ctypes.data)
    if rc:
        raise ValueError("hsx_power_spectrum: invalid arguments")
    return x


def partial_sum_2d(plane, n: int, zi: int, H: int, variant) -> float:
    plane = np.ascontiguousarray(plane, dtype=np.float32)
    Z, N = plane.shape
    return _load().hsx_partial_sum_2d(plane.ctypes.data, N, Z, int(n), int(zi), int(H), _v(variant))


def harmonic_sum_2d(x, Hmax: int, variant, want_sums=True) -> dict:
    """Planes x[B][Z][N] (Z odd).  sums[B][L][Z][N], max/gap [B][Z][N], argmax/second u8."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    if x.ndim == 2:
        x = x[None]
    B, Z, N = x.shape
    L = int(Hmax).bit_length()
    out = {"max": np.empty((B, Z, N), np.float64), "argmax": np.empty((B, Z, N), np.uint8),
           "gap": np.empty((B, Z, N), np.float64), "second": np.empty((B, Z, N), np.uint8)}
    if want_sums:
        out["sums"] = np.empty((B, L, Z, N), np.float64)
    rc = _load().hsx_harmonic_sum_2d(x.ctypes.data, N, Z, B, int(Hmax), _v(variant),
                                     out["sums"].ctypes.data if want_sums else None, out["max"].ctypes.data,
                                     out["argmax"].ctypes.data, out["gap"].ctypes.data, out["second"].ctypes.data)
    if rc:
        raise ValueError("hsx_harmonic_sum_2d: invalid arguments")
    return out
