/*
 * hs_oracle.c — TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, single-threaded CPU statement of the four harmonic-sum variants of
 * arXiv 1812.02647 (Adamek & Armour), in fp64, one level at a time, exactly in the paper's
 * order and notation.  It defines what the CUDA library must compute.  It shares no code,
 * header, table or helper with paper_1812_02647_b200/; only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may call it.
 *
 * Readings of the paper (CONVENTIONS.md C1..C11) followed here:
 *   eq. 1  PAPER.md:17     S_H(n) = sum_{i=1..H} x(floor((n*i + H/2)/H))            [C1]
 *   eq. 2  PAPER.md:33     S_H(n) = sum_{i=1..H} max_{0<=j<=i-1} xz(i*n + j)        [C2]
 *   eq. 3  PAPER.md:38     S_H(n) = sum_{i=1..H} xz(i*n)                            [C3]
 *   eq. 4  PAPER.md:43-46  S_1 = x(n), j = 0; i = 2..H: l = xz(i*n+j), r = xz(i*n+j+1),
 *                          S += max(l,r), j += (r > l)                              [C4]
 *   h_H(n) = S_H(n)/sqrt(H); xz(k) = 0 outside [0,N)            [C5,C7]
 *   levels H = 1,2,4,..,Hmax (BASELINE.json north_star)                             [symbols]
 *   reduced output: max over levels, smallest level on ties                         [C8]
 *
 * Every level is evaluated from scratch (no cumulative shortcut, no block-max shortcut):
 * those shortcuts are properties the tests check, not assumptions made here.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): exact-rational brute force on <=64-bin
 * spectra, per-term NumPy library routines at 2^18 bins, closed forms (constant, ramp,
 * monotone spectra), the comb special case on which all four variants must agree,
 * Max >= freq-bin / Greedy, enumeration of all monotone j paths, and the Exp(1) moment
 * closed forms.  What no pin can distinguish — the choice between the readings C2, C4, C5
 * and their alternatives — is "parity unpinned" against the paper.
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>

enum { HSO_STANDARD = 0, HSO_MAX = 1, HSO_FREQBIN = 2, HSO_GREEDY = 3 };

/* zero-padded read, C5 */
static double xz(const float *x, int64_t N, int64_t k)
{
    return (k >= 0 && k < N) ? (double)x[k] : 0.0;
}

/* number of levels for Hmax in {1,2,4,8,16,32}; -1 if Hmax is not one of them */
int hso_levels(int Hmax)
{
    int L = 0, H = 1;
    if (Hmax < 1 || Hmax > 32) return -1;
    while (H < Hmax) { H *= 2; L++; }
    return (H == Hmax) ? L + 1 : -1;
}

/*
 * One output: un-normalised S_H(n) of one variant for one spectrum x[0..N).
 * *j_out (may be NULL) receives Greedy's drift j after harmonic H (0 for other variants).
 */
double hso_partial_sum(const float *x, int64_t N, int64_t n, int H, int variant, int *j_out)
{
    double S = 0.0;
    int j = 0;
    if (variant == HSO_STANDARD) {                       /* eq. 1 */
        for (int i = 1; i <= H; i++)
            S += (double)x[(n * i + H / 2) / H];
    } else if (variant == HSO_FREQBIN) {                 /* eq. 3 */
        for (int i = 1; i <= H; i++)
            S += xz(x, N, (int64_t)i * n);
    } else if (variant == HSO_MAX) {                     /* eq. 2 */
        for (int i = 1; i <= H; i++) {
            double m = xz(x, N, (int64_t)i * n);
            for (int jj = 1; jj <= i - 1; jj++) {
                double v = xz(x, N, (int64_t)i * n + jj);
                if (v > m) m = v;
            }
            S += m;
        }
    } else {                                             /* eq. 4 */
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
 * Whole batch.  x[B][N] fp32.  Any output pointer may be NULL.
 *   sums  [B][L][N] fp64   h_H(n) = S_H(n)/sqrt(H)
 *   vmax  [B][N]    fp64   max over levels
 *   amax  [B][N]    uint8  smallest level index attaining it
 *   gap   [B][N]    fp64   vmax minus the second-largest level value (+inf if L == 1);
 *                          lets a test apply the near-tie rule C10
 *   second[B][N]    uint8  level index of that second-largest value (== amax if L == 1)
 *   jpath [B][L][N] uint8  Greedy j after harmonic H (zeros for other variants)
 * Returns 0, or 1 on invalid arguments.
 */
int hso_harmonic_sum(const float *x, int64_t N, int64_t B, int Hmax, int variant,
                     double *sums, double *vmax, uint8_t *amax, double *gap, uint8_t *second,
                     uint8_t *jpath)
{
    int L = hso_levels(Hmax);
    if (!x || N < 1 || B < 1 || L < 0 || variant < 0 || variant > 3) return 1;
    for (int64_t b = 0; b < B; b++) {
        const float *xb = x + b * N;
        for (int64_t n = 0; n < N; n++) {
            double best = 0.0, runner = 0.0;
            int abest = 0, arunner = 0;
            for (int l = 0; l < L; l++) {
                int H = 1 << l, j = 0;
                double h = hso_partial_sum(xb, N, n, H, variant, &j) / sqrt((double)H);
                if (sums)  sums[(b * L + l) * N + n] = h;
                if (jpath) jpath[(b * L + l) * N + n] = (uint8_t)j;
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

/*
 * Sampled outputs, for parity at sizes where the whole batch would take too long:
 * for point p, spectrum bidx[p] and bin nidx[p]; h[p][L] fp64, j[p][L] uint8 (either may be NULL).
 */
int hso_points(const float *x, int64_t N, int64_t B, int Hmax, int variant,
               int64_t npoints, const int64_t *bidx, const int64_t *nidx, double *h, uint8_t *j)
{
    int L = hso_levels(Hmax);
    if (!x || N < 1 || B < 1 || L < 0 || variant < 0 || variant > 3 || npoints < 0) return 1;
    for (int64_t p = 0; p < npoints; p++) {
        if (bidx[p] < 0 || bidx[p] >= B || nidx[p] < 0 || nidx[p] >= N) return 1;
        const float *xb = x + bidx[p] * N;
        for (int l = 0; l < L; l++) {
            int H = 1 << l, jj = 0;
            double S = hso_partial_sum(xb, N, nidx[p], H, variant, &jj);
            if (h) h[p * L + l] = S / sqrt((double)H);
            if (j) j[p * L + l] = (uint8_t)jj;
        }
    }
    return 0;
}
