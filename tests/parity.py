"""Comparison rules of CONVENTIONS.md C10 (BASELINE.json north_star): used by the -m gpu parity tests, smoke() and
bench.py.  NumPy only; imports neither the oracle nor the CUDA binding."""
from __future__ import annotations

import numpy as np

TOL = 1e-5


def check_sums(got, ref, what=""):
    """|gpu - ref| <= 1e-5 (1 + |ref|) element by element; returns the worst ratio err / (1 + |ref|)."""
    got = np.asarray(got, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    assert got.shape == ref.shape, (what, got.shape, ref.shape)
    assert np.isfinite(got).all(), f"{what}: non-finite output"
    err = np.abs(got - ref) / (1.0 + np.abs(ref))
    worst = float(err.max()) if err.size else 0.0
    if worst > TOL:
        idx = np.unravel_index(int(err.argmax()), err.shape)
        raise AssertionError(f"{what}: |err|/(1+|ref|) = {worst:.3e} > {TOL} at {idx}: got {got[idx]!r} ref {ref[idx]!r}")
    return worst


def check_argmax(got, ref_best, ref_second, ref_gap, ref_max, what=""):
    """Best level exact, except where the oracle's top two levels differ by < 1e-5 (1 + |best|): then either is
    accepted.  Returns the number of bins where the exemption was used."""
    got = np.asarray(got).astype(np.int64)
    ref_best = np.asarray(ref_best).astype(np.int64)
    ref_second = np.asarray(ref_second).astype(np.int64)
    near = np.asarray(ref_gap) < TOL * (1.0 + np.abs(np.asarray(ref_max)))
    ok = (got == ref_best) | (near & (got == ref_second))
    if not ok.all():
        idx = np.unravel_index(int((~ok).argmax()), ok.shape)
        raise AssertionError(f"{what}: best level {got[idx]} != oracle {ref_best[idx]} at {idx} "
                             f"(gap {np.asarray(ref_gap)[idx]:.3e}, {int((~ok).sum())} bins differ)")
    return int((got != ref_best).sum())


def argmax_from_levels(h):
    """Best/second level, gap and max from oracle level values h[..., L] (smallest level on ties, C8)."""
    h = np.asarray(h, dtype=np.float64)
    L = h.shape[-1]
    best = h.argmax(axis=-1)
    vmax = np.take_along_axis(h, best[..., None], -1)[..., 0]
    if L == 1:
        return best, best.copy(), np.full(vmax.shape, np.inf), vmax
    masked = h.copy()
    np.put_along_axis(masked, best[..., None], -np.inf, -1)
    second = masked.argmax(axis=-1)
    gap = vmax - np.take_along_axis(masked, second[..., None], -1)[..., 0]
    return best, second, gap, vmax


def check_candidates(count, got, ref, shape, what=""):
    """Candidate lists (hs_execute_candidates vs oracle.candidates): the order is unspecified, so both are compared as
    sets keyed by (spectrum, bin).  Every oracle candidate must be present and every record must be an oracle candidate,
    except bins whose oracle maximum lies within the tolerance of the threshold (either side may have them); values
    within the tolerance, levels by the rule of check_argmax.  `got` = dict of NumPy arrays (spectrum, bin, value, level)
    holding ALL `count` records.  Returns the number of threshold-borderline bins that were set aside."""
    B, N = shape
    gs, gb = np.asarray(got["spectrum"]).astype(np.int64), np.asarray(got["bin"]).astype(np.int64)
    assert count == gs.shape[0], f"{what}: count {count} != {gs.shape[0]} records"
    assert ((gs >= 0) & (gs < B) & (gb >= 0) & (gb < N)).all(), f"{what}: record outside the batch"
    gkey = gs * N + gb
    assert np.unique(gkey).shape[0] == gkey.shape[0], f"{what}: a bin was appended twice"
    rkey = np.asarray(ref["spectrum"]).astype(np.int64) * N + np.asarray(ref["bin"]).astype(np.int64)
    border = (ref["margin"] <= TOL * (1.0 + np.abs(ref["max"]))).reshape(-1)
    missing = np.setdiff1d(rkey, gkey)
    extra = np.setdiff1d(gkey, rkey)
    assert border[missing].all(), f"{what}: {int((~border[missing]).sum())} oracle candidates missing, e.g. {missing[:3]}"
    assert border[extra].all(), f"{what}: {int((~border[extra]).sum())} records are no oracle candidates, e.g. {extra[:3]}"
    m = ref["max"].reshape(-1)[gkey]
    check_sums(np.asarray(got["value"]), m, what + " value")
    check_argmax(np.asarray(got["level"]), (ref["argmax_all"]).reshape(-1)[gkey], ref["second"].reshape(-1)[gkey],
                 ref["gap"].reshape(-1)[gkey], m, what + " level")
    return int(missing.shape[0] + extra.shape[0])
