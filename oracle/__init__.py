"""ctypes loader for oracle/hs_oracle.c — TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this.  It never imports paper_1812_02647_b200 and shares nothing with it.
All arithmetic of eqs. 1-4 lives in hs_oracle.c; this file only builds it (gcc -O2, no -ffast-math),
marshals NumPy arrays and names the variants as the paper does.  The one
definition written here is candidates(): the threshold selection that follows the harmonic sum
in the pipeline, stated on the reduced output the C code returns.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "hs_oracle.c")
_LIB = os.path.join(_HERE, "libhs_oracle.so")

STANDARD, MAX, FREQBIN, GREEDY = 0, 1, 2, 3
VARIANTS = {"standard": STANDARD, "max": MAX, "freqbin": FREQBIN, "greedy": GREEDY}

_lib = None


def build(force: bool = False) -> str:
    """Compile hs_oracle.c into oracle/libhs_oracle.so (plain C, -O2, IEEE arithmetic)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-std=c99", "-O2", "-fPIC", "-shared", "-Wall", "-Wextra",
                               "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        i64, p = ctypes.c_int64, ctypes.c_void_p
        lib.hso_levels.argtypes = [ctypes.c_int]
        lib.hso_levels.restype = ctypes.c_int
        lib.hso_partial_sum.argtypes = [p, i64, i64, ctypes.c_int, ctypes.c_int, p]
        lib.hso_partial_sum.restype = ctypes.c_double
        lib.hso_harmonic_sum.argtypes = [p, i64, i64, ctypes.c_int, ctypes.c_int, p, p, p, p, p, p]
        lib.hso_harmonic_sum.restype = ctypes.c_int
        lib.hso_points.argtypes = [p, i64, i64, ctypes.c_int, ctypes.c_int, i64, p, p, p, p]
        lib.hso_points.restype = ctypes.c_int
        _lib = lib
    return _lib


def levels(Hmax: int) -> int:
    L = _load().hso_levels(int(Hmax))
    if L < 0:
        raise ValueError(f"Hmax must be one of 1,2,4,8,16,32, got {Hmax}")
    return L


def _as_batch(x) -> np.ndarray:
    x = np.ascontiguousarray(x, dtype=np.float32)
    if x.ndim == 1:
        x = x[None, :]
    if x.ndim != 2 or x.shape[1] < 1 or x.shape[0] < 1:
        raise ValueError("x must be [batch][nbins] with at least one bin")
    return x


def _variant(v) -> int:
    return VARIANTS[v] if isinstance(v, str) else int(v)


def harmonic_sum(x, Hmax: int, variant, want_sums: bool = True, want_reduced: bool = True,
                 want_jpath: bool = False) -> dict:
    """Whole batch.  Returns a dict with any of
    sums[B][L][N] f64, max[B][N] f64, argmax[B][N] u8, gap[B][N] f64, second[B][N] u8, jpath[B][L][N] u8."""
    x = _as_batch(x)
    B, N = x.shape
    L = levels(Hmax)
    out = {}
    if want_sums:
        out["sums"] = np.empty((B, L, N), np.float64)
    if want_reduced:
        out["max"] = np.empty((B, N), np.float64)
        out["argmax"] = np.empty((B, N), np.uint8)
        out["gap"] = np.empty((B, N), np.float64)
        out["second"] = np.empty((B, N), np.uint8)
    if want_jpath:
        out["jpath"] = np.empty((B, L, N), np.uint8)

    def ptr(k):
        return out[k].ctypes.data if k in out else None

    rc = _load().hso_harmonic_sum(x.ctypes.data, N, B, int(Hmax), _variant(variant),
                                  ptr("sums"), ptr("max"), ptr("argmax"), ptr("gap"), ptr("second"),
                                  ptr("jpath"))
    if rc != 0:
        raise ValueError("hso_harmonic_sum: invalid arguments")
    return out


def points(x, Hmax: int, variant, bidx, nidx):
    """Sampled outputs: h[P][L] f64 and Greedy j[P][L] u8 at (spectrum bidx[p], bin nidx[p])."""
    x = _as_batch(x)
    B, N = x.shape
    L = levels(Hmax)
    bidx = np.ascontiguousarray(bidx, dtype=np.int64)
    nidx = np.ascontiguousarray(nidx, dtype=np.int64)
    if bidx.shape != nidx.shape or bidx.ndim != 1:
        raise ValueError("bidx and nidx must be 1-D and of equal length")
    P = bidx.shape[0]
    h = np.empty((P, L), np.float64)
    j = np.empty((P, L), np.uint8)
    rc = _load().hso_points(x.ctypes.data, N, B, int(Hmax), _variant(variant), P,
                            bidx.ctypes.data, nidx.ctypes.data, h.ctypes.data, j.ctypes.data)
    if rc != 0:
        raise ValueError("hso_points: invalid arguments")
    return h, j


def partial_sum(x, n: int, H: int, variant):
    """One un-normalised S_H(n) of a single spectrum and Greedy's j after harmonic H."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    if x.ndim != 1 or not (0 <= n < x.shape[0]):
        raise ValueError("x must be 1-D and n in range")
    j = ctypes.c_int(0)
    S = _load().hso_partial_sum(x.ctypes.data, x.shape[0], int(n), int(H), _variant(variant),
                                ctypes.byref(j))
    return S, j.value


def candidates(x, Hmax: int, variant, threshold: float) -> dict:
    """The step after the harmonic sum ("SNR detection", "SNR recovered"): every (spectrum b,
    bin n) whose maximum over the levels m(b, n) = max_l h_{2^l}(b, n) exceeds `threshold` strictly, with that maximum
    and its level (smallest on ties, CONVENTIONS.md C8).  Plain definition: the reduced output of harmonic_sum, then a
    comparison.  Returns spectrum[], bin[] (int64, sorted by (spectrum, bin)), value[] f64, level[] u8, and `margin[]`
    = |m - threshold| for every bin of the batch as [B][N] f64 (so that a comparison can set aside the bins that sit
    within rounding of the threshold)."""
    ref = harmonic_sum(x, Hmax, variant, want_sums=False, want_reduced=True)
    m = ref["max"]
    b, n = np.nonzero(m > float(threshold))
    return {"spectrum": b.astype(np.int64), "bin": n.astype(np.int64), "value": m[b, n], "level": ref["argmax"][b, n],
            "margin": np.abs(m - float(threshold)), "gap": ref["gap"], "second": ref["second"], "max": m,
            "argmax_all": ref["argmax"]}
