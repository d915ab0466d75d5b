// hs_direct.cu — HS_ALGO_DIRECT: one thread per output bin, loads straight from global memory (through L1/L2).
// The simple on-device statement of eqs. 1-4 (CONVENTIONS.md C1-C8).  Needs no workspace and
// accepts every plan; the tuned kernels (hs_tiled_*.cu) are checked against the oracle and against this family.
#include "hs_internal.cuh"

namespace {

constexpr int kThreads = 256;

// CPLX (hs_execute_complex): x holds the complex Fourier series, every read forms the normalised power on the fly.
template <int VARIANT, int L, int OUT, bool JDBG, bool CPLX>
__global__ void __launch_bounds__(kThreads)
hs_direct_kernel(const float *__restrict__ x, float *__restrict__ sums, float *__restrict__ vmax,
                 uint8_t *__restrict__ amax, uint8_t *__restrict__ jdbg, int N, int tiles_per_spectrum, hs_cand_sink sink,
                 float scale)
{
    const int64_t b = blockIdx.x / tiles_per_spectrum;
    const int n = (blockIdx.x % tiles_per_spectrum) * kThreads + threadIdx.x;
    if (n >= N) return;
    const float *__restrict__ xb = x + b * (int64_t)N * (CPLX ? 2 : 1);
    auto ld = [&](int k) { return hs_ldx<CPLX>(xb, k, scale); };
    auto ldz = [&](const float *, int k, int) { return k < N ? hs_ldx<CPLX>(xb, k, scale) : 0.0f; };   // zero padding, C5
    float *plane0 = (OUT & HS_OUT_FULL) ? sums + (b * L) * (int64_t)N + n : nullptr;
    uint8_t *jplane0 = JDBG ? jdbg + (b * L) * (int64_t)N + n : nullptr;
    hs_emit<OUT> e;

    float S = ld(n);
    e.level(0, S, plane0, N);
    if (JDBG) jplane0[0] = 0;

    if (VARIANT == HS_STANDARD) {
        // eq. 1, cumulative over dyadic levels: level l adds the odd i < 2^l at denominator 2^l (F1 of DESIGN.md);
        // indices never exceed n.
#pragma unroll
        for (int l = 1; l < L; l++) {
            const int H = 1 << l;
#pragma unroll
            for (int i = 1; i < H; i += 2) S += ld((n * i + (H >> 1)) >> l);
            e.level(l, S, plane0, N);
        }
    } else if (VARIANT == HS_FREQBIN) {
#pragma unroll
        for (int l = 1; l < L; l++) {
#pragma unroll
            for (int i = (1 << (l - 1)) + 1; i <= (1 << l); i++) S += ldz(xb, i * n, N);
            e.level(l, S, plane0, N);
        }
    } else if (VARIANT == HS_MAX) {
#pragma unroll 1
        for (int l = 1; l < L; l++) {
            for (int i = (1 << (l - 1)) + 1; i <= (1 << l); i++) {
                const int k0 = i * n;
                float m = ldz(xb, k0, N);
                for (int j = 1; j < i; j++) m = fmaxf(m, ldz(xb, k0 + j, N));
                S += m;
            }
            e.level(l, S, plane0, N);
        }
    } else {  // HS_GREEDY
        int j = 0;
#pragma unroll
        for (int l = 1; l < L; l++) {
#pragma unroll
            for (int i = (1 << (l - 1)) + 1; i <= (1 << l); i++) {
                const int k = i * n + j;
                const float lft = ldz(xb, k, N), rgt = ldz(xb, k + 1, N);
                const bool right = rgt > lft;  // strictly greater, C4
                S += right ? rgt : lft;
                j += right ? 1 : 0;
            }
            e.level(l, S, plane0, N);
            if (JDBG) jplane0[(int64_t)l * N] = (uint8_t)j;
        }
    }
    if (OUT & HS_OUT_REDUCED) {
        if (OUT & HS_OUT_CAND) {
            hs_push(sink, b, n, e.m, e.a);
        } else {
            vmax[b * (int64_t)N + n] = e.m;
            amax[b * (int64_t)N + n] = (uint8_t)e.a;
        }
    }
}

template <int VARIANT, int L, int OUT, bool JDBG, bool CPLX>
int launch_c(const hs_plan *p, const hs_buffers &buf, int64_t batch, cudaStream_t stream)
{
    const int N = (int)p->nbins;
    const int tiles = (N + kThreads - 1) / kThreads;
    const int64_t max_spectra = ((int64_t)1 << 30) / tiles;  // keep gridDim.x below 2^31
    for (int64_t b0 = 0; b0 < batch; b0 += max_spectra) {
        const int64_t nb = (batch - b0 < max_spectra) ? batch - b0 : max_spectra;
        const int64_t off = b0 * (int64_t)N;
        hs_cand_sink sink = buf.sink;
        sink.b0 += (int)b0;
        hs_direct_kernel<VARIANT, L, OUT, JDBG, CPLX><<<(unsigned)(nb * tiles), kThreads, 0, stream>>>(
            buf.x + off * (CPLX ? 2 : 1), buf.sums ? buf.sums + off * L : nullptr, buf.vmax ? buf.vmax + off : nullptr,
            buf.amax ? buf.amax + off : nullptr, buf.jdbg ? buf.jdbg + off * L : nullptr, N, tiles, sink, buf.scale);
        HS_CUDA_OK(cudaGetLastError());
    }
    return HS_OK;
}

template <int VARIANT, int L, int OUT, bool JDBG>
int launch(const hs_plan *p, const hs_buffers &buf, int64_t batch, cudaStream_t stream)
{
    if (buf.cplx) return launch_c<VARIANT, L, OUT, JDBG, true>(p, buf, batch, stream);
    return launch_c<VARIANT, L, OUT, JDBG, false>(p, buf, batch, stream);
}

template <int VARIANT, int L>
int by_out(const hs_plan *p, const hs_buffers &buf, int64_t batch, cudaStream_t stream)
{
    if constexpr (VARIANT == HS_GREEDY) {
        if (buf.jdbg) return launch<VARIANT, L, 0, true>(p, buf, batch, stream);
    }
    switch (p->out_mode) {
        case HS_OUT_FULL: return launch<VARIANT, L, HS_OUT_FULL, false>(p, buf, batch, stream);
        case HS_OUT_REDUCED:
            if (buf.sink.cand) return launch<VARIANT, L, HS_OUT_REDUCED | HS_OUT_CAND, false>(p, buf, batch, stream);
            return launch<VARIANT, L, HS_OUT_REDUCED, false>(p, buf, batch, stream);
        default: return launch<VARIANT, L, HS_OUT_BOTH, false>(p, buf, batch, stream);
    }
}

template <int VARIANT>
int by_level(const hs_plan *p, const hs_buffers &buf, int64_t batch, cudaStream_t stream)
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

}  // namespace

int hs_launch_direct(const hs_plan *p, const hs_buffers &buf, int64_t batch, void *, cudaStream_t stream)
{
    switch (p->variant) {
        case HS_STANDARD: return by_level<HS_STANDARD>(p, buf, batch, stream);
        case HS_MAX: return by_level<HS_MAX>(p, buf, batch, stream);
        case HS_FREQBIN: return by_level<HS_FREQBIN>(p, buf, batch, stream);
        default: return by_level<HS_GREEDY>(p, buf, batch, stream);
    }
}
