/*
 * hs_oracle_ext.c — TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, single-threaded CPU statement of the three "next" rows of SURVEY.md section 8(f), in the same style as
 * hs_oracle.c (fp64 sums, one level at a time, from scratch, the paper's order and notation).  Shares no code with
 * paper_1812_02647_b200/ and does not include hs_oracle.c (the tests tie the two together where they must agree).
 *
 * (f)-3  partial sums for EVERY integer H = 1..Hmax, Hmax <= 64 ("partial sums of an increasing number
 *        of harmonics"), and eq. 2 with the window exactly as printed, 1 <= j <= i:
 *          eq. 1  S_H(n) = sum_{i=1..H} x(floor((2 n i + H)/(2 H)))     nearest bin, half up; for even H this is
 *                                                                        floor((n i + H/2)/H) of CONVENTIONS.md C1
 *          eq. 2  S_H(n) = sum_{i=1..H} max_{j in W_i} xz(i n + j)       W_i = {0..i-1} (C2) or {1..i} (as printed)
 *          eq. 3, eq. 4 as in hs_oracle.c (C3, C4)
 *        and eq. 1 with the spectrum read BETWEEN bins (reading R-INTERP, CONVENTIONS.md C15; the third sub-item of the
 *        row).  The argument of eq. 1, n i / H, is not an integer; PAPER.md:52 is about the power a
 *        harmonic loses when it falls between two Fourier bins.  With n i = q H + r, 0 <= r < H:
 *          eq. 1, interpolated  S_H(n) = sum_{i=1..H} ((H - r) x(q) + r x(q + 1)) / H
 *        the straight line through the two neighbouring bins (r = 0: the bin itself; q + 1 <= n whenever r > 0).
 *        h_H = S_H/sqrt(H); reduced output over the levels l = H - 1 = 0..Hmax-1, smallest level on ties (C8).
 * (f)-1  the step before the harmonic sum ("transformed using an FFT into frequency space. Then the
 *        harmonic sum is applied"): the normalised power spectrum of a complex Fourier series,
 *          x(k) = (Re F_k ^2 + Im F_k ^2) * scale - 1
 *        evaluated in fp32 with every operation rounded separately (no fused multiply-add): the harmonic sum's
 *        integer decisions (Greedy's comparisons, the best level) are taken on x, so both sides must form the same
 *        fp32 x.
 * (f)-4  the two-dimensional harmonic sum over the f - fdot plane of a Fourier-domain acceleration search
 *        (the paper gives no equation: reading R-2D of DESIGN.md section 16).  Plane x[Z][N], row zi
 *        <-> drift z = zi - (Z-1)/2 (Z odd), harmonic i of a signal at (n, z) sits at (n i/H, z i/H):
 *          2-D standard  S_H(n, z) = sum_{i=1..H} x(floor((z i + H/2)/H), floor((n i + H/2)/H))   (floor toward -inf)
 *          2-D freq-bin  S_H(n, z) = sum_{i=1..H} xz(i z, i n)          zero outside the plane
 *        levels H = 1, 2, 4, .., Hmax <= 32 as in CONVENTIONS.md.
 *
 * Pins: tests/test_oracle_ext_pins.py (-m "not gpu").
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>

enum { HSX_STANDARD = 0, HSX_MAX = 1, HSX_FREQBIN = 2, HSX_GREEDY = 3 };
enum { HSX_WINDOW_C2 = 0, HSX_WINDOW_PRINTED = 1, HSX_TERM_INTERP = 2 };   /* 2: eq. 1 only, interpolated terms */

static double xz(const float *x, int64_t N, int64_t k)
{
    return (k >= 0 && k < N) ? (double)x[k] : 0.0;
}

/* ------------------------------------------------------------------------------------------------ (f)-3 */
/* One un-normalised S_H(n), any integer H >= 1.  *j_out (may be NULL): Greedy's drift after harmonic H. */
double hsx_partial_sum(const float *x, int64_t N, int64_t n, int H, int variant, int window, int *j_out)
{
    double S = 0.0;
    int j = 0;
    if (variant == HSX_STANDARD && window == HSX_TERM_INTERP) {   /* eq. 1: x(n i / H) on the line between bins */
        for (int i = 1; i <= H; i++) {
            const int64_t q = (n * i) / H, r = (n * i) % H;
            S += ((double)(H - r) * (double)x[q] + (double)r * xz(x, N, q + 1)) / (double)H;
        }
    } else if (variant == HSX_STANDARD) {                 /* eq. 1: x(n i / H), nearest bin, half up */
        for (int i = 1; i <= H; i++)
            S += (double)x[(2 * n * i + H) / (2 * (int64_t)H)];
    } else if (variant == HSX_FREQBIN) {                  /* eq. 3 */
        for (int i = 1; i <= H; i++)
            S += xz(x, N, (int64_t)i * n);
    } else if (variant == HSX_MAX) {                      /* eq. 2 */
        const int j0 = (window == HSX_WINDOW_PRINTED) ? 1 : 0;
        for (int i = 1; i <= H; i++) {
            double m = xz(x, N, (int64_t)i * n + j0);
            for (int jj = j0 + 1; jj <= j0 + i - 1; jj++) {
                double v = xz(x, N, (int64_t)i * n + jj);
                if (v > m) m = v;
            }
            S += m;
        }
    } else {                                              /* eq. 4 */
        S = (double)x[n];
        for (int i = 2; i <= H; i++) {
            double l = xz(x, N, (int64_t)i * n + j);
            double r = xz(x, N, (int64_t)i * n + j + 1);
            if (r > l) { S += r; j += 1; } else { S += l; }
        }
    }
    if (j_out) *j_out = j;
    return S;
}

/*
 * Whole batch, every integer H = 1..Hmax (1 <= Hmax <= 64).  Level index l = H - 1.  Any output may be NULL:
 * sums[B][Hmax][N] f64, vmax[B][N] f64, amax[B][N] u8, gap[B][N] f64, second[B][N] u8, jpath[B][Hmax][N] u8.
 */
int hsx_harmonic_sum_all(const float *x, int64_t N, int64_t B, int Hmax, int variant, int window,
                         double *sums, double *vmax, uint8_t *amax, double *gap, uint8_t *second, uint8_t *jpath)
{
    if (!x || N < 1 || B < 1 || Hmax < 1 || Hmax > 64 || variant < 0 || variant > 3 || window < 0 || window > 2) return 1;
    if (window == HSX_TERM_INTERP && variant != HSX_STANDARD) return 1;
    for (int64_t b = 0; b < B; b++) {
        const float *xb = x + b * N;
        for (int64_t n = 0; n < N; n++) {
            double best = 0.0, runner = -INFINITY;
            int abest = 0, arunner = 0;
            for (int H = 1; H <= Hmax; H++) {
                int j = 0;
                const int l = H - 1;
                double h = hsx_partial_sum(xb, N, n, H, variant, window, &j) / sqrt((double)H);
                if (sums)  sums[(b * Hmax + l) * N + n] = h;
                if (jpath) jpath[(b * Hmax + l) * N + n] = (uint8_t)j;
                if (l == 0) { best = h; abest = 0; runner = -INFINITY; arunner = 0; }
                else if (h > best) { runner = best; arunner = abest; best = h; abest = l; }
                else if (h > runner) { runner = h; arunner = l; }
            }
            if (vmax)   vmax[b * N + n] = best;
            if (amax)   amax[b * N + n] = (uint8_t)abest;
            if (gap)    gap[b * N + n] = best - runner;
            if (second) second[b * N + n] = (uint8_t)arunner;
        }
    }
    return 0;
}

/* Sampled outputs: h[p][Hmax] f64 and j[p][Hmax] u8 at (spectrum bidx[p], bin nidx[p]). */
int hsx_points_all(const float *x, int64_t N, int64_t B, int Hmax, int variant, int window,
                   int64_t npoints, const int64_t *bidx, const int64_t *nidx, double *h, uint8_t *j)
{
    if (!x || N < 1 || B < 1 || Hmax < 1 || Hmax > 64 || variant < 0 || variant > 3 || npoints < 0) return 1;
    if (window < 0 || window > 2 || (window == HSX_TERM_INTERP && variant != HSX_STANDARD)) return 1;
    for (int64_t p = 0; p < npoints; p++) {
        if (bidx[p] < 0 || bidx[p] >= B || nidx[p] < 0 || nidx[p] >= N) return 1;
        const float *xb = x + bidx[p] * N;
        for (int H = 1; H <= Hmax; H++) {
            int jj = 0;
            double S = hsx_partial_sum(xb, N, nidx[p], H, variant, window, &jj);
            if (h) h[p * Hmax + H - 1] = S / sqrt((double)H);
            if (j) j[p * Hmax + H - 1] = (uint8_t)jj;
        }
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------------ (f)-1 */
/* x[k] = (re^2 + im^2) * scale - 1 for `count` complex values F[k] = (F[2k], F[2k+1]); fp32, each operation rounded
 * on its own (the volatile temporaries keep the compiler from contracting or widening anything). */
int hsx_power_spectrum(const float *F, int64_t count, float scale, float *x)
{
    if (!F || !x || count < 0) return 1;
    for (int64_t k = 0; k < count; k++) {
        volatile float rr = F[2 * k] * F[2 * k];
        volatile float ii = F[2 * k + 1] * F[2 * k + 1];
        volatile float p = rr + ii;
        volatile float s = p * scale;
        x[k] = s - 1.0f;
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------------ (f)-4 */
static int64_t floor_div(int64_t a, int64_t b)            /* b > 0; rounds toward minus infinity */
{
    int64_t q = a / b;
    if ((a % b != 0) && (a < 0)) q -= 1;
    return q;
}

/* One un-normalised S_H(n, z) of one plane x[Z][N]; zi = row index, z = zi - (Z-1)/2. */
double hsx_partial_sum_2d(const float *x, int64_t N, int64_t Z, int64_t n, int64_t zi, int H, int variant)
{
    const int64_t Zc = (Z - 1) / 2, z = zi - Zc;
    double S = 0.0;
    if (variant == HSX_STANDARD) {
        for (int i = 1; i <= H; i++) {
            const int64_t k = (n * i + H / 2) / H;
            const int64_t zz = floor_div(z * i + H / 2, H);
            S += (double)x[(zz + Zc) * N + k];
        }
    } else {                                              /* HSX_FREQBIN */
        for (int i = 1; i <= H; i++) {
            const int64_t k = (int64_t)i * n, row = (int64_t)i * z + Zc;
            if (k < N && row >= 0 && row < Z) S += (double)x[row * N + k];
        }
    }
    return S;
}

static int levels_of(int Hmax)
{
    int L = 0, H = 1;
    if (Hmax < 1 || Hmax > 32) return -1;
    while (H < Hmax) { H *= 2; L++; }
    return (H == Hmax) ? L + 1 : -1;
}

/* Whole batch of planes x[B][Z][N]; levels H = 1,2,4,..,Hmax.  sums[B][L][Z][N], vmax/gap[B][Z][N], amax/second u8. */
int hsx_harmonic_sum_2d(const float *x, int64_t N, int64_t Z, int64_t B, int Hmax, int variant,
                        double *sums, double *vmax, uint8_t *amax, double *gap, uint8_t *second)
{
    const int L = levels_of(Hmax);
    if (!x || N < 1 || Z < 1 || (Z % 2) == 0 || B < 1 || L < 0 || (variant != HSX_STANDARD && variant != HSX_FREQBIN)) return 1;
    for (int64_t b = 0; b < B; b++) {
        const float *xb = x + b * Z * N;
        for (int64_t zi = 0; zi < Z; zi++) {
            for (int64_t n = 0; n < N; n++) {
                double best = 0.0, runner = -INFINITY;
                int abest = 0, arunner = 0;
                for (int l = 0; l < L; l++) {
                    const int H = 1 << l;
                    double h = hsx_partial_sum_2d(xb, N, Z, n, zi, H, variant) / sqrt((double)H);
                    if (sums) sums[((b * L + l) * Z + zi) * N + n] = h;
                    if (l == 0) { best = h; abest = 0; runner = -INFINITY; arunner = 0; }
                    else if (h > best) { runner = best; arunner = abest; best = h; abest = l; }
                    else if (h > runner) { runner = h; arunner = l; }
                }
                const int64_t o = (b * Z + zi) * N + n;
                if (vmax)   vmax[o] = best;
                if (amax)   amax[o] = (uint8_t)abest;
                if (gap)    gap[o] = best - runner;
                if (second) second[o] = (uint8_t)arunner;
            }
        }
    }
    return 0;
}
