// hs_greedy_gather.cu — eq. 4 (CONVENTIONS.md C4, C5) as a per-thread, divergence-free gather.
//
// One thread owns one fundamental bin n and runs the chain i = 2..Hmax: l = x~(i n + j), r = x~(i n + j + 1),
// S += max(l, r), j += (r > l).  The candidates of harmonic i lie in the aligned block [i n, i n + i - 1], so for a
// warp of 32 consecutive n everything is in range while i (n_hi + 1) <= N: that bound is warp-uniform, and only
// the few harmonics that straddle the end of the spectrum take the predicated (zero-padded) path; harmonics that
// are out of range for the whole warp contribute max(0, 0) = 0 and leave j unchanged, so they are skipped.
// Averaged over a spectrum a bin has 4.06 in-range harmonics of the 32 (load imbalance of PAPER.md:21), which is why
// skipping matters more than anything else here: the direct kernel issues all 31 steps for every bin.
#include "hs_internal.cuh"
#include "hs_ptx.cuh"

namespace {

constexpr int kThreads = 128;
constexpr int kSpectraPerCta = 8;  // default Q; spectra run side by side per thread (tuned on B200: 2 -> 5.6 ms, 4 -> 4.9, 8 -> 4.7, 16 -> 5.4 for eq. 3)
constexpr int kGridY = 65535; // blockIdx.y = spectrum: CTAs are dispatched x-fastest, i.e. spectrum-major, so the gathers of
                              // all harmonics of one spectrum (1 MiB) happen close in time and hit L2 (ncu: 4 B/bin of DRAM
                              // reads; striding spectra over a small gridDim.y instead thrashed L2 at 28-33 B/bin)

// eq. 2 term of harmonic I at bin n, every element in range: max x[I n .. I n + I - 1], widest aligned vector loads
template <int I>
__device__ __forceinline__ float max_window(const float *__restrict__ w)
{
    if constexpr (I % 4 == 0) {
        float m = 0.f;
#pragma unroll
        for (int q = 0; q < I / 4; q++) {
            const float4 u = __ldg(reinterpret_cast<const float4 *>(w) + q);
            const float t = fmaxf(fmaxf(u.x, u.y), fmaxf(u.z, u.w));
            m = q == 0 ? t : fmaxf(m, t);
        }
        return m;
    } else if constexpr (I % 2 == 0) {
        float m = 0.f;
#pragma unroll
        for (int q = 0; q < I / 2; q++) {
            const float2 u = __ldg(reinterpret_cast<const float2 *>(w) + q);
            const float t = fmaxf(u.x, u.y);
            m = q == 0 ? t : fmaxf(m, t);
        }
        return m;
    } else {
        float m = __ldg(w);
#pragma unroll
        for (int q = 1; q < I; q++) m = fmaxf(m, __ldg(w + q));
        return m;
    }
}
__device__ __forceinline__ float max_window_rt(const float *__restrict__ w, int i)
{
    switch (i) {
        case 2: return max_window<2>(w);
        case 3: return max_window<3>(w);
        case 4: return max_window<4>(w);
        case 5: return max_window<5>(w);
        case 6: return max_window<6>(w);
        case 7: return max_window<7>(w);
        default: return max_window<8>(w);
    }
}

// SAME = false: the Q chains of a thread are the same bin of Q consecutive spectra.  SAME = true (long spectra, where Q
// spectra in flight per CTA row would not fit L2): the Q chains are the bins n, n + 128, .., n + 128 (Q - 1) of ONE
// spectrum; the warp-uniform bounds then span the CTA's Q blocks (safe: in range for the last block; any: for the first).
// JDBG (hs_debug_greedy_paths, eq. 4 only, OUT = 0): the drift j after each level goes to jdbg[b][l][n] instead of the outputs.
// CPLX (hs_execute_complex): x holds the complex Fourier series, every read forms the normalised power on the fly.
template <int VARIANT, int L, int OUT, int Q, bool SAME, bool JDBG = false, bool CPLX = false>
__global__ void __launch_bounds__(kThreads, Q >= 8 ? 8 : 12)
hs_greedy_gather_kernel(const float *__restrict__ x, float *__restrict__ sums, float *__restrict__ vmax,
                        uint8_t *__restrict__ amax, uint8_t *__restrict__ jdbg, int N, int batch, hs_cand_sink sink, float scale)
{
    const int n = blockIdx.x * (SAME ? kThreads * Q : kThreads) + threadIdx.x;
    const int n_lo = n & ~31;                      // first bin of this warp (of its first block)
    if (n_lo >= N) return;
    constexpr int NB = SAME ? Q : 1;               // distinct bins per thread
    bool valid[NB];
    int nn[NB];
#pragma unroll
    for (int k = 0; k < NB; k++) {
        valid[k] = n + k * kThreads < N;
        nn[k] = valid[k] ? n + k * kThreads : N - 1;   // lanes past the end shadow the last bin and store nothing
    }
    const int n_hi1 = min(n_lo + (NB - 1) * kThreads + 32, N);   // one past the warp's last bin (of its last block)
    // Warp-uniform range tests (no divisions): harmonic i is in range for EVERY lane, neighbour included, iff
    // i * n_hi1 <= N; it is in range for SOME lane iff i * n_lo < N.
    // A thread runs the same bin of Q consecutive spectra side by side: the control flow depends on n only, so the Q
    // chains share every bound and give Q independent loads in flight (Greedy's chain is serial within a spectrum).
    constexpr int QS = SAME ? 1 : Q;               // spectra per thread
    for (int b0 = blockIdx.y * QS; b0 < batch; b0 += gridDim.y * QS) {
        const float *__restrict__ xb[Q];
        bool live[Q];
        hs_emit<OUT> e[Q];
        float S[Q];
        int j[Q];
#pragma unroll
        for (int q = 0; q < Q; q++) {
            live[q] = valid[SAME ? q : 0] && b0 + (SAME ? 0 : q) < batch;
            xb[q] = x + (int64_t)min(b0 + (SAME ? 0 : q), batch - 1) * N * (CPLX ? 2 : 1);   // spectra past the batch shadow the last one
            S[q] = hs_ldx<CPLX>(xb[q], nn[SAME ? q : 0], scale);
            j[q] = 0;
        }
        auto emit = [&](int l) {
#pragma unroll
            for (int q = 0; q < Q; q++) {
                const float h = S[q] * hs_norm(l);
                if ((OUT & HS_OUT_FULL) && live[q])
                    hsptx::st_cs(sums + (((int64_t)(b0 + (SAME ? 0 : q)) * L + l) * N + nn[SAME ? q : 0]), h);
                if (OUT & HS_OUT_REDUCED) e[q].reduce(l, h);
                if (JDBG && live[q])
                    jdbg[((int64_t)(b0 + (SAME ? 0 : q)) * L + l) * N + nn[SAME ? q : 0]] = (uint8_t)j[q];
            }
        };
        auto step = [&](const int (&bases)[NB], int i, bool safe) {   // harmonic i, bases[k] == i * nn[k]
#pragma unroll
            for (int q = 0; q < Q; q++) {
                const int base = bases[SAME ? q : 0];
                if (VARIANT == HS_FREQBIN) {        // eq. 3: x~(i n)
                    S[q] += (safe || base < N) ? hs_ldx<CPLX>(xb[q], base, scale) : 0.0f;
                } else if (VARIANT == HS_MAX) {     // eq. 2 (Hmax <= 8): maximum of the aligned block x~[i n .. i n + i - 1]
                    if (safe && !CPLX) {
                        S[q] += max_window_rt(xb[q] + base, i);
                    } else {
                        float m = base < N ? hs_ldx<CPLX>(xb[q], base, scale) : 0.0f;
                        for (int t = 1; t < i; t++) m = fmaxf(m, base + t < N ? hs_ldx<CPLX>(xb[q], base + t, scale) : 0.0f);
                        S[q] += m;
                    }
                } else {                            // eq. 4: max of the bin under the drift and its right neighbour
                    const int k = base + j[q];
                    const float lft = (safe || k < N) ? hs_ldx<CPLX>(xb[q], k, scale) : 0.0f;
                    const float rgt = (safe || k + 1 < N) ? hs_ldx<CPLX>(xb[q], k + 1, scale) : 0.0f;
                    const bool right = rgt > lft;   // strictly greater (C4)
                    S[q] += right ? rgt : lft;
                    j[q] += right ? 1 : 0;
                }
            }
        };
        emit(0);
        bool tail = false;
#pragma unroll
        for (int l = 1; l < L; l++) {
            const int lo = (1 << (l - 1)) + 1, hi = 1 << l;
            if (lo * n_lo < N) {                    // some harmonic of this level is in range for some lane
                int i = lo;
                int base[NB];                       // (i - 1) * n
#pragma unroll
                for (int k = 0; k < NB; k++) base[k] = (lo - 1) * nn[k];
                for (; i <= hi && i * n_hi1 <= N; i++) {
#pragma unroll
                    for (int k = 0; k < NB; k++) base[k] += nn[k];
                    step(base, i, true);
                }
                for (; i <= hi && i * n_lo < N; i++) {
#pragma unroll
                    for (int k = 0; k < NB; k++) base[k] += nn[k];
                    step(base, i, false);
                }
                emit(l);
            } else if ((OUT & 3) != HS_OUT_REDUCED || JDBG) {
                emit(l);
            } else {
                tail = true;
            }
        }
        // Levels whose harmonics are all out of range leave S unchanged, and h_l = S c_l is monotone in l: for S >= 0
        // no later level exceeds the running maximum, for S < 0 the last level is the largest.  Test level L-1 only.
        if ((OUT & 3) == HS_OUT_REDUCED && tail) emit(L - 1);
        if (OUT & HS_OUT_REDUCED) {
#pragma unroll
            for (int q = 0; q < Q; q++) {
                const int64_t bq = b0 + (SAME ? 0 : q);
                const int nq = n + (SAME ? q * kThreads : 0);
                if (live[q] && (OUT & HS_OUT_CAND)) {
                    hs_push(sink, bq, nq, e[q].m, e[q].a);
                } else if (live[q]) {
                    // (plain stores: measured 4 % faster here than the evict-first stores the other kernels use)
                    vmax[bq * N + nq] = e[q].m;
                    amax[bq * N + nq] = (uint8_t)e[q].a;
                }
            }
        }
    }
}

template <int VARIANT, int L, int OUT, int Q, bool SAME, bool JDBG, bool CPLX>
int launch_qc(const hs_plan *p, const hs_buffers &buf, int64_t batch, cudaStream_t stream)
{
    const int N = (int)p->nbins;
    const int per_cta = SAME ? kThreads * Q : kThreads;
    const int tiles = (N + per_cta - 1) / per_cta;
    const int64_t max_spectra = (int64_t)1 << 30;            // int b inside the kernel
    for (int64_t b0 = 0; b0 < batch; b0 += max_spectra) {
        const int64_t nb = (batch - b0 < max_spectra) ? batch - b0 : max_spectra;
        const int64_t off = b0 * (int64_t)N;
        const int64_t gy = SAME ? nb : (nb + Q - 1) / Q;
        const dim3 grid((unsigned)tiles, (unsigned)(gy < kGridY ? gy : kGridY), 1);
        hs_cand_sink sink = buf.sink;
        sink.b0 += (int)b0;
        hs_greedy_gather_kernel<VARIANT, L, OUT, Q, SAME, JDBG, CPLX><<<grid, kThreads, 0, stream>>>(
            buf.x + off * (CPLX ? 2 : 1), buf.sums ? buf.sums + off * L : nullptr, buf.vmax ? buf.vmax + off : nullptr,
            buf.amax ? buf.amax + off : nullptr, buf.jdbg ? buf.jdbg + off * L : nullptr, N, (int)nb, sink, buf.scale);
        HS_CUDA_OK(cudaGetLastError());
    }
    return HS_OK;
}

template <int VARIANT, int L, int OUT, int Q, bool SAME = false, bool JDBG = false>
int launch_q(const hs_plan *p, const hs_buffers &buf, int64_t batch, cudaStream_t stream)
{
    if constexpr (!JDBG) {
        if (buf.cplx) return launch_qc<VARIANT, L, OUT, Q, SAME, false, true>(p, buf, batch, stream);
    }
    return launch_qc<VARIANT, L, OUT, Q, SAME, JDBG, false>(p, buf, batch, stream);
}

// Spectra side by side per thread: 8 while 8 spectra (and what is in flight around them) stay in L2; longer spectra run
// fewer at a time so that the gathers of all harmonics of a spectrum still hit L2 (2^22 bins = 16 MiB per spectrum).
template <int VARIANT, int L, int OUT, bool JDBG = false>
int launch(const hs_plan *p, const hs_buffers &buf, int64_t batch, cudaStream_t stream)
{
    // spectra of more than 2^22 bins (32 MiB and up): 8 bin blocks of ONE spectrum per thread instead of 8 spectra
    // (B200, 2^30 bins in all, 2^23-bin spectra: eq. 3 Hmax 2 2.11 -> 1.70 ms, Hmax 32 8.16 -> 6.08 ms; eq. 4 9.21 -> 7.42 ms)
    if (p->nbins > ((int64_t)1 << 22) || (L <= 2 && VARIANT != HS_MAX && p->nbins >= 8192))   // (eqs. 3-4 with two harmonics: 5 - 8 % faster)
        return launch_q<VARIANT, L, OUT, kSpectraPerCta, true, JDBG>(p, buf, batch, stream);
    if (L >= 5) {                                                  // (with few harmonics the loads in flight matter more)
        if (p->nbins > ((int64_t)1 << 20)) return launch_q<VARIANT, L, OUT, 2, false, JDBG>(p, buf, batch, stream);
    }
    return launch_q<VARIANT, L, OUT, kSpectraPerCta, false, JDBG>(p, buf, batch, stream);
}

template <int VARIANT, int L>
int by_out(const hs_plan *p, const hs_buffers &buf, int64_t batch, cudaStream_t stream)
{
    if constexpr (VARIANT == HS_GREEDY) {                          // the same kernel and launch shape, j instead of the outputs
        if (buf.jdbg) return launch<VARIANT, L, 0, true>(p, buf, batch, stream);
    }
    switch (p->out_mode) {
        case HS_OUT_FULL: return launch<VARIANT, L, HS_OUT_FULL>(p, buf, batch, stream);
        case HS_OUT_REDUCED:
            if (buf.sink.cand) return launch<VARIANT, L, HS_OUT_REDUCED | HS_OUT_CAND>(p, buf, batch, stream);
            return launch<VARIANT, L, HS_OUT_REDUCED>(p, buf, batch, stream);
        default: return launch<VARIANT, L, HS_OUT_BOTH>(p, buf, batch, stream);
    }
}

}  // namespace

template <int VARIANT>
static int by_level(const hs_plan *p, const hs_buffers &buf, int64_t batch, cudaStream_t stream)
{
    switch (p->L) {
        case 1: return by_out<VARIANT, 1>(p, buf, batch, stream);
        case 2: return by_out<VARIANT, 2>(p, buf, batch, stream);
        case 3: return by_out<VARIANT, 3>(p, buf, batch, stream);
        case 4: return by_out<VARIANT, 4>(p, buf, batch, stream);
        case 5: return by_out<VARIANT, 5>(p, buf, batch, stream);
        default: return by_out<VARIANT, 6>(p, buf, batch, stream);
    }
}

// Greedy (eq. 4) always; freq-bin (eq. 3) as the workspace-free alternative to the two-phase kernel.
int hs_greedy_gather_launch(const hs_plan *p, const hs_buffers &buf, int64_t batch, cudaStream_t stream)
{
    if (p->variant == HS_FREQBIN) return by_level<HS_FREQBIN>(p, buf, batch, stream);
    if (p->variant == HS_MAX) {                                    // Hmax <= 8 only (hs_tiled.cu)
        switch (p->L) {
            case 1: return by_out<HS_MAX, 1>(p, buf, batch, stream);
            case 2: return by_out<HS_MAX, 2>(p, buf, batch, stream);
            case 3: return by_out<HS_MAX, 3>(p, buf, batch, stream);
            default: return by_out<HS_MAX, 4>(p, buf, batch, stream);
        }
    }
    return by_level<HS_GREEDY>(p, buf, batch, stream);
}

int hs_greedy_gather_launches(const hs_plan *p, int64_t batch)
{
    (void)p;
    const int64_t max_spectra = (int64_t)1 << 30;
    return (int)((batch + max_spectra - 1) / max_spectra);
}
