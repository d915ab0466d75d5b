"""Pins for oracle/hs_oracle.c: things the paper and the mathematics fix, none of which call the CUDA path.

P2  exact-rational brute force on tiny spectra (different language, different formula path)
P3  per-term NumPy library routines at 2^18 bins (strided slice, block reshape-max, repeat)
P4  closed forms of eq. 1 (constant, ramp)
P5  eq. 1 is cumulative over dyadic levels          P6  eqs. 2-4 are cumulative in H
P7  an integer-bin comb makes all four variants agree (BASELINE.json north_star)
P8  Max >= freq-bin, Max >= Greedy, Greedy <= best monotone path <= Max
P9/P10 Exp(1) moment closed forms for eq. 2 / eq. 4  P11 monotone spectra: Greedy == freq-bin / Max
P12 Greedy j bounds                                  P13 reduced-output invariants
Citations: eq. 1, eq. 2, eq. 3, eq. 4; CONVENTIONS.md C1-C11.
"""
import itertools
import math
from fractions import Fraction

import numpy as np
import pytest

LEVELS = [1, 2, 4, 8, 16, 32]
VARIANTS = ["standard", "max", "freqbin", "greedy"]


# ----------------------------------------------------------------------------- P2 brute force
def _pad(x, k):
    return x[k] if 0 <= k < len(x) else Fraction(0)


def brute_standard(x, n, H):
    # nearest bin to the rational n*i/H, an exact half goes up (C1)
    tot = Fraction(0)
    for i in range(1, H + 1):
        q = Fraction(n * i, H)
        k = math.floor(q)
        if q - k >= Fraction(1, 2):
            k += 1
        tot += x[k]
    return tot


def brute_max(x, n, H):
    padded = list(x) + [Fraction(0)] * (32 * len(x) + 32)
    return sum(max(padded[i * n:i * n + i]) for i in range(1, H + 1))


def brute_freqbin(x, n, H):
    return sum(_pad(x, i * n) for i in range(1, H + 1))


def brute_greedy_chain(x, n, H):
    S, j = x[n], 0
    for i in range(2, H + 1):
        l, r = _pad(x, i * n + j), _pad(x, i * n + j + 1)
        if r > l:
            S, j = S + r, j + 1
        else:
            S = S + l
    return S, j


def _tiny_spectra():
    rng = np.random.default_rng(20181202)
    out = []
    for N in (1, 2, 3, 5, 7, 16, 31, 33, 50, 64):
        out.append(rng.standard_normal(N).astype(np.float32))
        out.append((rng.standard_exponential(N) - 1).astype(np.float32))
        out.append(rng.integers(-3, 4, N).astype(np.float32))          # many exact ties, zeros, negatives
    out.append(np.zeros(40, np.float32))
    out.append(-np.ones(40, np.float32))                                   # zero padding beats in-range values
    out.append(np.arange(48, dtype=np.float32))
    out.append(np.arange(48, dtype=np.float32)[::-1].copy())
    return out


@pytest.mark.parametrize("variant", VARIANTS)
def test_p2_brute_force_tiny(oracle, variant):
    for x in _tiny_spectra():
        xf = [Fraction(float(v)) for v in x]
        N = len(xf)
        o = oracle.harmonic_sum(x, 32, variant, want_jpath=True)
        for l, H in enumerate(LEVELS):
            for n in range(N):
                if variant == "standard":
                    S, j = brute_standard(xf, n, H), 0
                elif variant == "max":
                    S, j = brute_max(xf, n, H), 0
                elif variant == "freqbin":
                    S, j = brute_freqbin(xf, n, H), 0
                else:
                    S, j = brute_greedy_chain(xf, n, H)
                ref = float(S) / math.sqrt(H)
                got = o["sums"][0, l, n]
                assert abs(got - ref) <= 1e-12 * (1 + abs(ref)), (variant, N, H, n)
                assert o["jpath"][0, l, n] == j, (variant, N, H, n)


def test_p2_hmax_subsets_and_batch(oracle):
    rng = np.random.default_rng(5)
    x = rng.standard_normal((3, 37)).astype(np.float32)
    for v in VARIANTS:
        full = oracle.harmonic_sum(x, 32, v)["sums"]
        for Hmax in (1, 2, 4, 8, 16):
            L = oracle.levels(Hmax)
            part = oracle.harmonic_sum(x, Hmax, v)["sums"]
            assert part.shape == (3, L, 37)
            np.testing.assert_array_equal(part, full[:, :L, :])
        for b in range(3):
            np.testing.assert_array_equal(oracle.harmonic_sum(x[b], 32, v)["sums"][0], full[b])
    with pytest.raises(ValueError):
        oracle.levels(3)
    with pytest.raises(ValueError):
        oracle.levels(64)


# ----------------------------------------------------------------------------- P1, P3 library routines
@pytest.fixture(scope="module")
def noise18():
    return (np.random.default_rng(18).standard_exponential(1 << 18).astype(np.float32) - np.float32(1))


@pytest.fixture(scope="module")
def outs18(oracle, noise18):
    return {v: oracle.harmonic_sum(noise18, 32, v, want_jpath=True) for v in VARIANTS}


def test_p1_h1_is_x(outs18, noise18):
    for v in VARIANTS:
        np.testing.assert_array_equal(outs18[v]["sums"][0, 0], noise18.astype(np.float64))


def _term_freqbin(x, i):
    t = np.zeros(x.shape[0])
    d = x[::i].astype(np.float64)
    t[:d.shape[0]] = d
    return t


def _term_max(x, i):
    N = x.shape[0]
    nblk = -(-N // i)
    p = np.zeros(nblk * i)
    p[:N] = x
    t = np.zeros(N)
    t[:nblk] = p.reshape(nblk, i).max(axis=1)
    return t


def test_p3_freqbin_and_max_terms_are_slices_and_block_maxima(outs18, noise18):
    for v, term in (("freqbin", _term_freqbin), ("max", _term_max)):
        S = np.zeros(noise18.shape[0])
        for i in range(1, 33):
            S = S + term(noise18, i)
            if i in LEVELS:
                ref = S / math.sqrt(i)
                got = outs18[v]["sums"][0, LEVELS.index(i)]
                np.testing.assert_allclose(got, ref, rtol=0, atol=1e-12 * (1 + np.abs(ref).max()))


def test_p3_standard_is_freqbin_of_the_repeated_spectrum(oracle):
    # x(floor((n i + H/2)/H)) = y(n i) with y = repeat(x, H) advanced by H/2: eq. 1 at level H is eq. 3 at level H
    # of the H-fold nearest-neighbour up-sampled spectrum (np.repeat fixes the rounding, not the oracle).
    x = np.random.default_rng(3).standard_normal(5000).astype(np.float32)
    std = oracle.harmonic_sum(x, 32, "standard")["sums"][0]
    for l, H in enumerate(LEVELS):
        y = np.concatenate([np.repeat(x, H)[H // 2:], np.zeros(H // 2, np.float32)])
        fb = oracle.harmonic_sum(y, H, "freqbin")["sums"][0, l, :x.shape[0]]
        np.testing.assert_allclose(std[l], fb, rtol=0, atol=1e-12)


# ----------------------------------------------------------------------------- P4 closed forms of eq. 1
def test_p4_constant_and_ramp(oracle):
    c = np.full(777, 1.25, np.float32)
    s = oracle.harmonic_sum(c, 32, "standard")["sums"][0]
    for l, H in enumerate(LEVELS):
        np.testing.assert_allclose(s[l], 1.25 * math.sqrt(H), rtol=1e-14)
    ramp = np.arange(4096, dtype=np.float32)
    s = oracle.harmonic_sum(ramp, 32, "standard")["sums"][0]
    for l, H in enumerate(LEVELS):
        n = np.arange(0, 4096, H)                     # H divides n: sum_i n i/H = n (H+1)/2
        np.testing.assert_allclose(s[l, n], n * (H + 1) / 2 / math.sqrt(H), rtol=1e-14)
        # any n: the sum of the nearest integers to n i/H
        for nn in (1, 5, 33, 1001, 4095):
            ref = sum(math.floor(Fraction(nn * i, H) + Fraction(1, 2)) for i in range(1, H + 1))
            assert s[l, nn] == pytest.approx(ref / math.sqrt(H), rel=1e-14)


# ----------------------------------------------------------------------------- P5, P6 cumulative structure
def test_p5_standard_dyadic_cumulative_and_index_range(outs18, noise18):
    N = noise18.shape[0]
    n = np.arange(N)
    S = outs18["standard"]["sums"][0] * np.sqrt(np.array(LEVELS, dtype=np.float64))[:, None]
    for l in range(5):
        H = LEVELS[l]
        odd = np.zeros(N)
        for i in range(1, 2 * H, 2):
            k = (n * i + H) // (2 * H)
            assert k.max() <= N - 1 and (k <= n).all()
            odd += noise18[k].astype(np.float64)
        np.testing.assert_allclose(S[l + 1] - S[l], odd, rtol=0, atol=1e-11)


def test_p6_eqs234_cumulative_in_H(oracle):
    x = np.random.default_rng(6).standard_normal(3000).astype(np.float32)
    N = x.shape[0]
    for v in ("max", "freqbin", "greedy"):
        for H in range(1, 32):
            for n in (0, 1, 2, 7, 45, 93, 94, 500, 1499, 1500, 2999):
                a, ja = oracle.partial_sum(x, n, H, v)
                b, jb = oracle.partial_sum(x, n, H + 1, v)
                i = H + 1
                blk = [float(x[k]) if k < N else 0.0 for k in range(i * n, i * n + i)]
                if v == "max":
                    term = max(blk)
                elif v == "freqbin":
                    term = blk[0]
                else:
                    l_, r_ = blk[ja], (blk[ja + 1] if ja + 1 < i else (float(x[i * n + i]) if i * n + i < N else 0.0))
                    term = max(l_, r_)
                    assert jb == ja + (1 if r_ > l_ else 0)
                assert b - a == pytest.approx(term, abs=1e-12)


# ----------------------------------------------------------------------------- P7 comb: all variants agree
def test_p7_integer_bin_comb_all_variants_agree(oracle):
    N, m = 1 << 16, 1251
    a = (10.0 * 0.9 ** np.arange(32) + 0.5).astype(np.float32)
    x = np.zeros(N, np.float32)
    x[m * np.arange(1, 33)] = a
    cum = np.cumsum(a.astype(np.float64))
    outs = {v: oracle.harmonic_sum(x, 32, v, want_jpath=True) for v in VARIANTS}
    for l, H in enumerate(LEVELS):
        ref = cum[H - 1] / math.sqrt(H)
        assert outs["standard"]["sums"][0, l, H * m] == pytest.approx(ref, rel=1e-14)
        for v in ("max", "freqbin", "greedy"):
            assert outs[v]["sums"][0, l, m] == pytest.approx(ref, rel=1e-14)
        assert outs["greedy"]["jpath"][0, l, m] == 0
    # all levels are positive and growing slower than sqrt(H) from some point: best level is unique and shared
    best = {v: int(outs[v]["argmax"][0, m]) for v in ("max", "freqbin", "greedy")}
    assert len(set(best.values())) == 1
    lvl = best["max"]
    assert int(outs["standard"]["argmax"][0, LEVELS[lvl] * m]) >= 0


# ----------------------------------------------------------------------------- P8 inequalities and path enumeration
def test_p8_max_dominates(outs18):
    for l in range(6):
        assert (outs18["max"]["sums"][0, l] >= outs18["freqbin"]["sums"][0, l] - 1e-12).all()
        assert (outs18["max"]["sums"][0, l] >= outs18["greedy"]["sums"][0, l] - 1e-12).all()
    # Greedy >= freq-bin is NOT a theorem; make sure the data actually exercises both orders
    d = outs18["greedy"]["sums"][0, 5] - outs18["freqbin"]["sums"][0, 5]
    assert (d > 0).any() and (d < 0).any()


def test_p8_greedy_is_one_monotone_path_bounded_by_the_best_path_and_max(oracle):
    rng = np.random.default_rng(8)
    for N in (40, 64):
        x = rng.standard_normal(N).astype(np.float32)
        xz = lambda k: float(x[k]) if 0 <= k < N else 0.0
        for H in (2, 4, 8):
            for n in range(N):
                # a monotone path: j_1 = 0, j_i in {j_{i-1}, j_{i-1}+1}; its sum takes x(i n + j_i)
                best = -math.inf
                for steps in itertools.product((0, 1), repeat=H - 1):
                    j, S = 0, xz(n)
                    for i, s in zip(range(2, H + 1), steps):
                        j += s
                        S += xz(i * n + j)
                    best = max(best, S)
                g, _ = oracle.partial_sum(x, n, H, "greedy")
                m, _ = oracle.partial_sum(x, n, H, "max")
                assert g <= best + 1e-12 <= m + 2e-12


# ----------------------------------------------------------------------------- P9, P10 moments under Exp(1)-1 noise
def test_p9_p10_exponential_noise_moments(oracle):
    rng = np.random.default_rng(910)
    B, N = 256, 4096
    x = (rng.standard_exponential((B, N)) - 1).astype(np.float32)
    sel = slice(40, N // 32 - 1)                      # n > 32 and every window of every harmonic in range
    Hn = np.cumsum(1.0 / np.arange(1, 33))            # harmonic numbers
    H2 = np.cumsum(1.0 / np.arange(1, 33) ** 2)
    got = {v: oracle.harmonic_sum(x, 32, v, want_reduced=False)["sums"][:, :, sel] for v in VARIANTS}
    nsamp = got["max"][:, 0].size
    for l, H in enumerate(LEVELS):
        # eq. 2: max of i iid Exp(1) has mean H_i and variance sum_{m<=i} 1/m^2; blocks of different i overlap,
        # so only the mean is pinned tightly
        mean_ref = (Hn[:H] - 1).sum() / math.sqrt(H)
        assert got["max"][:, l].mean() == pytest.approx(mean_ref, abs=6 * math.sqrt(H2[:H].sum() / H * 32 / nsamp) + 1e-9)
        # eq. 4: each step takes the max of two fresh bins: mean 1/2, variance 5/4; first term mean 0 variance 1
        mean_ref = (H - 1) / (2 * math.sqrt(H))
        var_ref = (1 + 1.25 * (H - 1)) / H
        assert got["greedy"][:, l].mean() == pytest.approx(mean_ref, abs=6 * math.sqrt(var_ref * 32 / nsamp) + 1e-9)
        assert got["greedy"][:, l].var() == pytest.approx(var_ref, rel=0.05)
        # eqs. 1 and 3: sums of H unit-variance zero-mean bins, normalised by sqrt(H)
        for v in ("standard", "freqbin"):
            assert got[v][:, l].mean() == pytest.approx(0.0, abs=6 * math.sqrt(32 / nsamp))
            assert got[v][:, l].var() == pytest.approx(1.0, rel=0.05)
    assert (Hn[:32] - 1).sum() / math.sqrt(32) == pytest.approx(12.362, abs=1e-3)   # SURVEY P9 figure


# ----------------------------------------------------------------------------- P11 monotone spectra
def test_p11_monotone_spectra(oracle):
    N = 2048
    dec = np.linspace(10.0, 1.0, N).astype(np.float32)
    inc = np.arange(N, dtype=np.float32)
    g = oracle.harmonic_sum(dec, 32, "greedy", want_jpath=True)
    f = oracle.harmonic_sum(dec, 32, "freqbin")
    lim = N // 32 - 2                                   # all harmonics and their neighbours in range
    np.testing.assert_array_equal(g["sums"][0, :, :lim], f["sums"][0, :, :lim])
    assert (g["jpath"][0, :, :lim] == 0).all()
    g = oracle.harmonic_sum(inc, 32, "greedy", want_jpath=True)
    m = oracle.harmonic_sum(inc, 32, "max")
    np.testing.assert_array_equal(g["sums"][0, :, :lim], m["sums"][0, :, :lim])
    n = np.arange(lim)
    for l, H in enumerate(LEVELS):
        assert (g["jpath"][0, l, :lim] == H - 1).all()
        np.testing.assert_allclose(g["sums"][0, l, :lim], ((n + 1) * H * (H + 1) / 2 - H) / math.sqrt(H), rtol=1e-14)


# ----------------------------------------------------------------------------- P12, P13
def test_p12_greedy_j_bounds(outs18):
    j = outs18["greedy"]["jpath"][0].astype(int)
    for l, H in enumerate(LEVELS):
        assert j[l].min() >= 0 and j[l].max() <= H - 1
    assert (np.diff(j, axis=0) >= 0).all()
    assert j[5].max() > 20                              # the drift really happens on noise


def test_p13_reduced_output_invariants(oracle, outs18):
    for v in VARIANTS:
        o = outs18[v]
        s, m, a = o["sums"][0], o["max"][0], o["argmax"][0].astype(int)
        assert a.min() >= 0 and a.max() <= 5
        np.testing.assert_array_equal(m, s.max(axis=0))
        np.testing.assert_array_equal(m, np.take_along_axis(s, a[None, :], 0)[0])
        np.testing.assert_array_equal(a, s.argmax(axis=0))           # numpy argmax = first (smallest) level on ties
        srt = np.sort(s, axis=0)
        np.testing.assert_allclose(o["gap"][0], srt[-1] - srt[-2], rtol=0, atol=0)
        sec = o["second"][0].astype(int)
        np.testing.assert_array_equal(np.take_along_axis(s, sec[None, :], 0)[0], srt[-2])
    z = oracle.harmonic_sum(np.zeros(100, np.float32), 32, "max")
    assert (z["argmax"] == 0).all() and (z["max"] == 0).all() and (z["gap"] == 0).all()
    one = oracle.harmonic_sum(np.ones(10, np.float32), 1, "standard")
    assert np.isinf(one["gap"]).all() and (one["argmax"] == 0).all()


def test_points_entry_matches_whole_batch(oracle):
    rng = np.random.default_rng(77)
    x = rng.standard_normal((4, 999)).astype(np.float32)
    b = rng.integers(0, 4, 300)
    n = rng.integers(0, 999, 300)
    for v in VARIANTS:
        o = oracle.harmonic_sum(x, 16, v, want_jpath=True)
        h, j = oracle.points(x, 16, v, b, n)
        np.testing.assert_array_equal(h, o["sums"][b, :, n])
        np.testing.assert_array_equal(j, o["jpath"][b, :, n])
    with pytest.raises(ValueError):
        oracle.points(x, 16, "max", [4], [0])


def test_candidates_definition_on_a_zero_background_comb():
    """oracle.candidates (threshold detection after the harmonic sum): on a zero background with spikes
    a_k at bins k m the freq-bin maximum over levels at bin m is max_H sum_{k<=H} a_k / sqrt(H); every bin above the
    threshold is listed exactly once, sorted, with the level of the maximum; nothing else is."""
    import oracle
    N, m = 4096, 37
    x = np.zeros((2, N), np.float32)
    a = np.array([9.0, 7.0, 5.0, 3.0, 1.0, 1.0, 1.0, 1.0], np.float64)
    for k in range(1, 9):
        x[1, k * m] = a[k - 1]
    h = [a[:H].sum() / np.sqrt(H) for H in (1, 2, 4, 8)]            # 9, 11.31, 12, 9.9 -> best level 2 (H = 4)
    res = oracle.candidates(x, 8, "freqbin", 11.5)
    assert res["spectrum"].tolist() == [1] and res["bin"].tolist() == [m]
    assert abs(res["value"][0] - max(h)) < 1e-12 and res["level"][0] == int(np.argmax(h)) == 2
    res = oracle.candidates(x, 8, "freqbin", 8.9)                    # the spike of 9 at bin m itself and at ... only m: 2m holds 7
    assert res["bin"].tolist() == [m]
    res = oracle.candidates(x, 8, "freqbin", 6.9)                    # bins m (12) and 2m (x = 7, harmonics 4m: 3, 6m: 1, 8m: 1)
    assert res["spectrum"].tolist() == [1, 1] and res["bin"].tolist() == [m, 2 * m]
    assert oracle.candidates(x, 8, "freqbin", 12.0)["bin"].size == 0  # strictly greater
    full = oracle.harmonic_sum(x, 8, "freqbin")
    ref = np.argwhere(full["sums"].max(axis=1) > 2.9)
    res = oracle.candidates(x, 8, "freqbin", 2.9)
    assert np.array_equal(np.stack([res["spectrum"], res["bin"]], 1), ref)
