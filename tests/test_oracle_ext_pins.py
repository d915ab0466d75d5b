"""Pins of oracle/hs_oracle_ext.c against things other than itself: exact-rational
brute force, NumPy library routines, closed forms, and the already pinned hs_oracle.c where the two must agree."""
import math
from fractions import Fraction

import numpy as np
import pytest

import oracle
from oracle import ext

VARIANTS = ["standard", "max", "freqbin", "greedy"]


def xz(x, k):
    return float(x[k]) if 0 <= k < len(x) else 0.0


def brute(x, n, H, variant, window="c2"):
    """S_H(n) straight from the printed equations with exact rational index arithmetic."""
    N = len(x)
    if variant == "standard":
        S = 0.0
        for i in range(1, H + 1):
            q = Fraction(n * i, H) + Fraction(1, 2)          # nearest bin, half up
            S += float(x[math.floor(q)])
        return S, 0
    if variant == "freqbin":
        return sum(xz(x, i * n) for i in range(1, H + 1)), 0
    if variant == "max":
        js = (lambda i: range(1, i + 1)) if window == "printed" else (lambda i: range(0, i))
        return sum(max(xz(x, i * n + j) for j in js(i)) for i in range(1, H + 1)), 0
    S, j = float(x[n]), 0
    for i in range(2, H + 1):
        l, r = xz(x, i * n + j), xz(x, i * n + j + 1)
        if r > l:
            S, j = S + r, j + 1
        else:
            S = S + l
    return S, j


# ---------------------------------------------------------------------------------------------- (f)-3
@pytest.mark.parametrize("variant", VARIANTS)
def test_every_integer_H_against_exact_rational_brute_force(variant):
    rng = np.random.default_rng(11)
    for N in (1, 2, 7, 33, 64):
        x = rng.standard_normal(N).astype(np.float32)
        x[rng.integers(0, N)] = 0.0
        for window in (("c2", "printed") if variant == "max" else ("c2",)):
            ref = ext.harmonic_sum_all(x, 64, variant, window, want_jpath=True)
            for n in range(N):
                for H in range(1, 65):
                    S, j = brute(x, n, H, variant, window)
                    assert ref["sums"][0, H - 1, n] == pytest.approx(S / math.sqrt(H), rel=1e-12, abs=1e-12)
                    assert ref["jpath"][0, H - 1, n] == j
                    assert ext.partial_sum(x, n, H, variant, window)[0] == pytest.approx(S, rel=1e-12, abs=1e-12)


@pytest.mark.parametrize("variant", VARIANTS)
def test_dyadic_levels_agree_with_the_pinned_dyadic_oracle(variant):
    """At H = 1, 2, 4, .., 32 the all-H functions must reproduce hs_oracle.c bit for bit (for even H the nearest-bin
    index floor((2 n i + H)/(2 H)) is C1's floor((n i + H/2)/H))."""
    rng = np.random.default_rng(12)
    x = (rng.standard_exponential((3, 3000)) - 1).astype(np.float32)
    a = ext.harmonic_sum_all(x, 32, variant, want_jpath=True)
    d = oracle.harmonic_sum(x, 32, variant, want_jpath=True)
    for l, H in enumerate((1, 2, 4, 8, 16, 32)):
        np.testing.assert_array_equal(a["sums"][:, H - 1], d["sums"][:, l])
        np.testing.assert_array_equal(a["jpath"][:, H - 1], d["jpath"][:, l])


def test_eq1_any_H_is_the_repeat_identity_and_closed_forms():
    """x(nearest(n i / H)) = np.repeat(x, 2 H)[2 n i + H]: NumPy's repeat fixes the rounding (m // (2 H) is the bin that
    sample m of the 2H-fold oversampled spectrum came from).  Constant spectrum -> c sqrt(H); ramp with H | n -> n (H + 1) / 2."""
    N = 2000
    x = np.arange(N, dtype=np.float32)
    rng = np.random.default_rng(16)
    y = rng.standard_normal(N).astype(np.float32)
    n = np.arange(N)
    for arr in (x, y):
        ref = ext.harmonic_sum_all(arr, 64, "standard")["sums"][0]
        for H in (1, 3, 5, 6, 7, 12, 31, 33, 63, 64):
            over = np.repeat(arr.astype(np.float64), 2 * H)
            terms = np.stack([over[np.minimum(2 * n * i + H, over.size - 1)] for i in range(1, H + 1)])
            np.testing.assert_allclose(ref[H - 1], terms.sum(0) / math.sqrt(H), rtol=1e-12, atol=1e-12)
    ref = ext.harmonic_sum_all(x, 64, "standard")["sums"][0]
    for H in (1, 3, 5, 6, 7, 12, 31, 33, 63, 64):
        m = np.arange(0, N, H)
        np.testing.assert_allclose(ref[H - 1][m] * math.sqrt(H), m * (H + 1) / 2, rtol=1e-12)
    c = ext.harmonic_sum_all(np.full(500, 2.5, np.float32), 64, "standard")["sums"][0]
    for H in range(1, 65):
        np.testing.assert_allclose(c[H - 1], 2.5 * math.sqrt(H), rtol=1e-12)


def test_printed_window_is_the_c2_window_of_the_spectrum_shifted_by_one_bin():
    """max_{1<=j<=i} x(i n + j) = max_{0<=j<=i-1} x'(i n + j) with x'(k) = x(k + 1): NumPy fixes the shift."""
    rng = np.random.default_rng(13)
    x = (rng.standard_exponential((2, 5000)) - 1).astype(np.float32)
    shifted = np.concatenate([x[:, 1:], np.zeros((2, 1), np.float32)], axis=1)
    a = ext.harmonic_sum_all(x, 40, "max", "printed")
    b = ext.harmonic_sum_all(shifted, 40, "max", "c2")
    np.testing.assert_array_equal(a["sums"], b["sums"])
    assert a["sums"][0, 0, 7] == x[0, 8]                       # h_1(n) = x(n + 1): what the printed window implies


# ---- eq. 1 with interpolated terms (reading R-INTERP, CONVENTIONS.md C15)
def brute_interp(x, n, H):
    """sum_i of the straight line through the two bins around n i / H, in exact rational arithmetic on the fp32 values."""
    S = Fraction(0)
    for i in range(1, H + 1):
        p = Fraction(n * i, H)
        q = math.floor(p)
        w = p - q
        right = Fraction(float(x[q + 1])) if q + 1 < len(x) else Fraction(0)
        S += (1 - w) * Fraction(float(x[q])) + w * right
    return S


def test_interpolated_eq1_against_exact_rational_brute_force():
    rng = np.random.default_rng(18)
    x = rng.standard_normal(61).astype(np.float32)
    ref = ext.harmonic_sum_all(x, 64, "standard", "interp")["sums"][0]
    for H in range(1, 65):
        for n in range(61):
            assert ref[H - 1, n] * math.sqrt(H) == pytest.approx(float(brute_interp(x, n, H)), rel=1e-12, abs=1e-12)
            assert ext.partial_sum(x, n, H, "standard", "interp")[0] == pytest.approx(float(brute_interp(x, n, H)), rel=1e-12, abs=1e-12)


def test_interpolated_eq1_is_numpy_interp_and_is_exact_on_straight_lines():
    """np.interp is the library's piecewise-linear interpolation: S_H(n) = sum_i interp(n i / H).  On a ramp x(k) = a k + b
    the line between two bins IS the ramp, so S_H(n) = a n (H + 1)/2 + b H exactly (the nearest-bin sum is not: it rounds
    every n i / H to a bin); h_1 = x; and at bins n that are multiples of H every harmonic sits on a bin, so the
    interpolated and the nearest-bin sums agree there."""
    rng = np.random.default_rng(19)
    N = 700
    x = rng.standard_normal(N).astype(np.float32)
    r = ext.harmonic_sum_all(x, 64, "standard", "interp")["sums"][0]
    nearest = ext.harmonic_sum_all(x, 64, "standard")["sums"][0]
    n = np.arange(N, dtype=np.float64)
    k = np.arange(N, dtype=np.float64)
    np.testing.assert_array_equal(r[0], x)
    for H in (2, 3, 5, 7, 16, 33, 64):
        want = sum(np.interp(n * i / H, k, x.astype(np.float64)) for i in range(1, H + 1)) / math.sqrt(H)
        np.testing.assert_allclose(r[H - 1], want, rtol=1e-12, atol=1e-12)
        np.testing.assert_allclose(r[H - 1, ::H], nearest[H - 1, ::H], rtol=1e-13, atol=1e-13)
        assert np.abs(r[H - 1] - nearest[H - 1]).max() > 0.1                       # elsewhere the two readings differ
    ramp = (0.25 * np.arange(N) - 3.0).astype(np.float32)                          # exactly representable
    rr = ext.harmonic_sum_all(ramp, 64, "standard", "interp")["sums"][0]
    for H in range(1, 65):
        np.testing.assert_allclose(rr[H - 1], (0.25 * n * (H + 1) / 2 - 3.0 * H) / math.sqrt(H), rtol=1e-13, atol=1e-12)
    red = ext.harmonic_sum_all(x, 48, "standard", "interp")                         # reduced output: NumPy reductions
    np.testing.assert_array_equal(red["argmax"], red["sums"].argmax(axis=1))
    np.testing.assert_array_equal(red["max"], red["sums"].max(axis=1))
    for bad in ("max", "freqbin", "greedy"):                                        # only eq. 1 has an argument between bins
        with pytest.raises(ValueError):
            ext.harmonic_sum_all(x, 8, bad, "interp")


@pytest.mark.parametrize("variant", ["max", "freqbin", "greedy"])
def test_partial_sums_are_cumulative_in_every_integer_H(variant):
    rng = np.random.default_rng(14)
    x = rng.standard_normal(700).astype(np.float32)
    S = ext.harmonic_sum_all(x, 64, variant)["sums"][0] * np.sqrt(np.arange(1, 65))[:, None]
    n = np.arange(700)
    for H in range(2, 65):
        if variant == "freqbin":
            term = np.array([xz(x, H * k) for k in n])
        elif variant == "max":
            term = np.array([max(xz(x, H * k + j) for j in range(H)) for k in n])
        else:
            continue
        np.testing.assert_allclose(S[H - 1] - S[H - 2], term, atol=1e-9)
    if variant == "greedy":
        jp = ext.harmonic_sum_all(x, 64, variant, want_jpath=True)["jpath"][0].astype(int)
        assert (np.diff(jp, axis=0) >= 0).all() and (jp <= np.arange(64)[:, None]).all()


def test_reduced_output_over_all_levels_is_numpy_argmax():
    rng = np.random.default_rng(15)
    x = rng.standard_normal((2, 400)).astype(np.float32)
    for variant in VARIANTS:
        r = ext.harmonic_sum_all(x, 48, variant)
        np.testing.assert_array_equal(r["argmax"], r["sums"].argmax(axis=1))          # first maximum: smallest level
        np.testing.assert_array_equal(r["max"], r["sums"].max(axis=1))
        srt = np.sort(r["sums"], axis=1)
        np.testing.assert_allclose(r["gap"], srt[:, -1] - srt[:, -2])
    z = ext.harmonic_sum_all(np.zeros(64, np.float32), 64, "max")
    assert (z["argmax"] == 0).all()


def numpy_second(levels_first):
    """Runner-up level from level values h[..., L, ...] with the level axis at position 1: the largest value once the best
    level is masked out, smallest level on ties (NumPy's argmax returns the first maximum)."""
    h = np.moveaxis(np.asarray(levels_first, dtype=np.float64), 1, -1).copy()
    best = h.argmax(axis=-1)
    np.put_along_axis(h, best[..., None], -np.inf, -1)
    return h.argmax(axis=-1), h.max(axis=-1)


def test_second_best_level_over_all_levels_is_numpy_argmax_of_the_rest():
    """`second` (what the near-tie rule of the parity tests accepts instead of `argmax`) and `gap`, on random data and on
    small-integer data where several levels tie exactly."""
    rng = np.random.default_rng(16)
    cases = [rng.standard_normal((2, 300)).astype(np.float32), rng.integers(-1, 2, (2, 300)).astype(np.float32),
             np.zeros((1, 64), np.float32)]
    for x in cases:
        for variant in VARIANTS:
            r = ext.harmonic_sum_all(x, 48, variant)
            second, runner = numpy_second(r["sums"])
            np.testing.assert_array_equal(r["second"], second)
            np.testing.assert_array_equal(r["gap"], r["max"] - runner)
            assert (r["second"] != r["argmax"]).all()
    one = ext.harmonic_sum_all(cases[0], 1, "max")                # a single level has no runner-up
    assert np.isinf(one["gap"]).all() and (one["second"] == 0).all()


@pytest.mark.parametrize("variant", VARIANTS)
def test_points_entry_matches_whole_batch_for_every_integer_H(variant):
    """hsx_points_all (what the GPU tests sample full-size runs with) against hsx_harmonic_sum_all, which the brute-force
    pins above fix: every level of every sampled point, Greedy's j included, both eq. 2 windows."""
    rng = np.random.default_rng(17)
    B, N, Hmax = 3, 500, 37
    x = rng.standard_normal((B, N)).astype(np.float32)
    bidx = np.concatenate([rng.integers(0, B, 200), [0, B - 1, B - 1]])
    nidx = np.concatenate([rng.integers(0, N, 200), [0, 0, N - 1]])
    for window in (("c2", "printed") if variant == "max" else ("c2", "interp") if variant == "standard" else ("c2",)):
        whole = ext.harmonic_sum_all(x, Hmax, variant, window, want_jpath=True)
        h, j = ext.points_all(x, Hmax, variant, bidx, nidx, window)
        assert h.shape == (len(bidx), Hmax) and j.shape == (len(bidx), Hmax)
        np.testing.assert_array_equal(h, whole["sums"][bidx, :, nidx])
        np.testing.assert_array_equal(j, whole["jpath"][bidx, :, nidx])
    with pytest.raises(ValueError):
        ext.points_all(x, Hmax, variant, [B], [0])
    with pytest.raises(ValueError):
        ext.points_all(x, Hmax, variant, [0], [N])


# ---------------------------------------------------------------------------------------------- (f)-1
def test_power_spectrum_matches_numpy_and_is_formed_in_fp32_step_by_step():
    rng = np.random.default_rng(21)
    F = (rng.standard_normal(4096) + 1j * rng.standard_normal(4096)).astype(np.complex64) * 300
    scale = np.float32(1.0 / 312500.0)
    x = ext.power_spectrum(F, float(scale))
    ref64 = (F.real.astype(np.float64) ** 2 + F.imag.astype(np.float64) ** 2) * float(scale) - 1
    np.testing.assert_allclose(x, ref64, rtol=0, atol=4e-7 * (1 + np.abs(ref64)).max())
    # the exact fp32 recipe, operation by operation, with NumPy's correctly rounded fp32 arithmetic
    re, im = F.real.astype(np.float32), F.imag.astype(np.float32)
    step = ((re * re) + (im * im)) * scale - np.float32(1)
    np.testing.assert_array_equal(x, step.astype(np.float32))


def test_power_spectrum_parseval_and_a_unit_sinusoid():
    """White noise: sum_k |F_k|^2 = n sum_t s_t^2 (Parseval), so with scale = 1/n the mean of x + 1 over all n bins is
    the series' mean square.  A sinusoid of amplitude A on bin m puts |F_m|^2 = (A n / 2)^2 into bins m and n - m."""
    rng = np.random.default_rng(22)
    n = 4096
    s = rng.standard_normal(n)
    F = np.fft.fft(s).astype(np.complex64)
    x = ext.power_spectrum(F, 1.0 / n).astype(np.float64)
    assert (x + 1).sum() / n == pytest.approx((s ** 2).mean(), rel=1e-5)
    A, m = 3.0, 137
    F = np.fft.fft(A * np.cos(2 * np.pi * m * np.arange(n) / n)).astype(np.complex64)
    x = ext.power_spectrum(F, 1.0 / n).astype(np.float64)
    assert x[m] + 1 == pytest.approx((A * n / 2) ** 2 / n, rel=1e-5) and x[n - m] + 1 == pytest.approx((A * n / 2) ** 2 / n, rel=1e-5)
    rest = np.delete(x, [m, n - m])
    assert np.abs(rest + 1).max() < 1e-3


# ---------------------------------------------------------------------------------------------- (f)-4
def brute_2d(plane, n, zi, H, variant):
    Z, N = plane.shape
    Zc = (Z - 1) // 2
    z = zi - Zc
    S = 0.0
    for i in range(1, H + 1):
        if variant == "standard":
            k = math.floor(Fraction(n * i, H) + Fraction(1, 2))
            zz = math.floor(Fraction(z * i, H) + Fraction(1, 2))
            S += float(plane[zz + Zc, k])
        else:
            k, row = i * n, i * z + Zc
            if k < N and 0 <= row < Z:
                S += float(plane[row, k])
    return S


@pytest.mark.parametrize("variant", ["standard", "freqbin"])
def test_2d_against_exact_rational_brute_force(variant):
    rng = np.random.default_rng(31)
    for Z, N in ((1, 9), (3, 17), (7, 40), (9, 64)):
        plane = rng.standard_normal((Z, N)).astype(np.float32)
        ref = ext.harmonic_sum_2d(plane, 32, variant)["sums"][0]
        for l, H in enumerate((1, 2, 4, 8, 16, 32)):
            for zi in range(Z):
                for n in range(N):
                    assert ref[l, zi, n] == pytest.approx(brute_2d(plane, n, zi, H, variant) / math.sqrt(H), rel=1e-12, abs=1e-12)


@pytest.mark.parametrize("variant", ["standard", "freqbin"])
def test_2d_reduces_to_the_1d_sum_on_the_zero_drift_row_and_for_a_single_row(variant):
    rng = np.random.default_rng(32)
    plane = (rng.standard_exponential((11, 900)) - 1).astype(np.float32)
    r2 = ext.harmonic_sum_2d(plane, 32, variant)
    r1 = oracle.harmonic_sum(plane[5], 32, variant)
    np.testing.assert_array_equal(r2["sums"][0, :, 5, :], r1["sums"][0])          # z = 0: every harmonic stays on the row
    np.testing.assert_array_equal(r2["argmax"][0, 5], r1["argmax"][0])
    one = ext.harmonic_sum_2d(plane[3:4], 32, variant)
    np.testing.assert_array_equal(one["sums"][0, :, 0, :], oracle.harmonic_sum(plane[3], 32, variant)["sums"][0])


def test_2d_standard_on_an_additive_plane_splits_into_two_1d_standard_sums():
    """x(z, k) = a(z) + b(k): S_H(n, z) = sum_i a(z_i) + sum_i b(k_i), and for z >= 0 the drift part is eq. 1 applied to
    the array a[Zc:], so the pinned 1-D oracle fixes both parts."""
    rng = np.random.default_rng(33)
    Z, N = 21, 300
    Zc = 10
    a = rng.standard_normal(Z).astype(np.float32)
    b = rng.standard_normal(N).astype(np.float32)
    plane = (a[:, None].astype(np.float64) + b[None, :].astype(np.float64))
    plane32 = plane.astype(np.float32)
    r = ext.harmonic_sum_2d(plane32, 32, "standard")["sums"][0]
    sa = oracle.harmonic_sum(a[Zc:], 32, "standard")["sums"][0]            # [L][Z - Zc]
    sb = oracle.harmonic_sum(b, 32, "standard")["sums"][0]                 # [L][N]
    for l in range(6):
        expect = sa[l][:, None] + sb[l][None, :]
        np.testing.assert_allclose(r[l, Zc:, :], expect, atol=2e-5)        # (plane32 rounds a + b to fp32)


def test_2d_integer_harmonic_track_is_fully_recovered():
    """A signal at fundamental (r0, z0) has harmonic k at (k r0, k z0) (the sum puts the power "back into a
    single Fourier bin"): on a zero plane both 2-D variants return sum_{k<=H} a_k / sqrt(H), the standard one at
    (H r0, H z0), the freq-bin one at (r0, z0)."""
    Z, N, r0, z0 = 129, 4096, 100, -2
    Zc = 64
    amp = (5.0 * 0.9 ** np.arange(32) + 0.25).astype(np.float32)
    plane = np.zeros((Z, N), np.float32)
    for k in range(1, 33):
        plane[k * z0 + Zc, k * r0] = amp[k - 1]
    for l, H in enumerate((1, 2, 4, 8, 16, 32)):
        want = float(np.cumsum(amp.astype(np.float64))[H - 1]) / math.sqrt(H)
        assert ext.partial_sum_2d(plane, H * r0, H * z0 + Zc, H, "standard") / math.sqrt(H) == pytest.approx(want, rel=1e-12)
        assert ext.partial_sum_2d(plane, r0, z0 + Zc, H, "freqbin") / math.sqrt(H) == pytest.approx(want, rel=1e-12)
    red = ext.harmonic_sum_2d(plane, 32, "freqbin", want_sums=False)
    assert red["argmax"][0, z0 + Zc, r0] == int(np.argmax(np.cumsum(amp.astype(np.float64))[[0, 1, 3, 7, 15, 31]] / np.sqrt([1, 2, 4, 8, 16, 32])))


@pytest.mark.parametrize("variant", ["standard", "freqbin"])
def test_2d_reduced_outputs_are_numpy_reductions_of_the_level_planes(variant):
    """max / argmax / gap / second of hsx_harmonic_sum_2d on every row of the plane (not only the zero-drift one),
    against NumPy reductions of its own level planes, which the brute-force pin above fixes; integer data for exact ties."""
    rng = np.random.default_rng(34)
    for plane in ((rng.standard_exponential((2, 7, 120)) - 1).astype(np.float32),
                  rng.integers(-1, 2, (1, 5, 90)).astype(np.float32), np.zeros((1, 3, 40), np.float32)):
        for Hmax in (32, 4):
            r = ext.harmonic_sum_2d(plane, Hmax, variant)
            np.testing.assert_array_equal(r["argmax"], r["sums"].argmax(axis=1))      # first maximum: smallest level (C8)
            np.testing.assert_array_equal(r["max"], r["sums"].max(axis=1))
            second, runner = numpy_second(r["sums"])
            np.testing.assert_array_equal(r["second"], second)
            np.testing.assert_array_equal(r["gap"], r["max"] - runner)
            red = ext.harmonic_sum_2d(plane, Hmax, variant, want_sums=False)          # the reduced-only call: same values
            for k in ("max", "argmax", "gap", "second"):
                np.testing.assert_array_equal(red[k], r[k])


def test_2d_constant_plane_closed_form():
    r = ext.harmonic_sum_2d(np.full((5, 50), 1.5, np.float32), 32, "standard")["sums"][0]
    for l, H in enumerate((1, 2, 4, 8, 16, 32)):
        np.testing.assert_allclose(r[l], 1.5 * math.sqrt(H), rtol=1e-12)
