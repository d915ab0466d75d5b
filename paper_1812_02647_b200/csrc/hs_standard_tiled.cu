// hs_standard_tiled.cu — eq. 1 (CONVENTIONS.md C1) with the index windows staged in shared memory.
//
// With Hmax-scaled harmonics i = 1..Hmax, the term of harmonic i at output n is x[(n i + Hmax/2) / Hmax]; level
// H = 2^l sums the i that are multiples of Hmax/H, so all levels share the same Hmax terms and level l only adds
// the odd multiples of Hmax/2^l (eq. 1 is cumulative over dyadic levels).  A tile of T consecutive outputs reads,
// for harmonic i, the contiguous window x[idx_i(n0) .. idx_i(n0+T-1)] of about T i/Hmax words: (Hmax+1)/2 words
// per output in total.  Lane 0..Hmax-1 of warp 0 each issue one TMA bulk copy (cp.async.bulk, UBLKCP) for "their"
// window onto one mbarrier; every thread then gathers its terms from shared memory.  A warp step handles 32
// consecutive outputs, so the 32 lanes of one LDS hit at most 32 consecutive words: conflict-free (with broadcast).
#include "hs_internal.cuh"
#include "hs_ptx.cuh"

namespace {

constexpr int ilog2(int v) { return v <= 1 ? 0 : 1 + ilog2(v >> 1); }

template <int HMAX, int OUT, int WARPS, int STEPS>
__global__ void __launch_bounds__(WARPS * 32)
hs_std_tiled_kernel(const float *__restrict__ x, float *__restrict__ sums, float *__restrict__ vmax,
                    uint8_t *__restrict__ amax, int N, int tiles, hs_cand_sink sink)
{
    constexpr int LG = ilog2(HMAX), L = LG + 1, T = WARPS * STEPS * 32;
    extern __shared__ __align__(128) float win[];
    __shared__ uint64_t bar;
    __shared__ int delta[32];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t b = blockIdx.x / tiles;
    const int n0 = (blockIdx.x % tiles) * T;
    const int n_end = min(n0 + T, N);
    const float *__restrict__ xb = x + b * (int64_t)N;

    if (threadIdx.x == 0) {
        hsptx::mbar_init(&bar, HMAX);
        hsptx::mbar_fence_init();
    }
    __syncthreads();
    if (warp == 0) {
        const int i = lane + 1;
        const bool act = i <= HMAX;
        const int lo = (n0 * i + HMAX / 2) >> LG;
        const int hi = ((n_end - 1) * i + HMAX / 2) >> LG;
        const int lo_al = lo & ~3;                                    // 16-byte aligned source
        const int size = act ? ((hi - lo_al + 4) & ~3) : 0;           // words, multiple of 4, stays inside [0, N)
        int off = size;                                               // inclusive warp scan -> exclusive offset
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, off, d);
            if (lane >= d) off += t;
        }
        off -= size;
        if (act) {
            delta[lane] = off - lo_al;
            hsptx::mbar_arrive_expect_tx(&bar, (uint32_t)size * 4u);
            hsptx::bulk_g2s(win + off, xb + lo_al, (uint32_t)size * 4u, &bar);
        }
    }
    __syncthreads();

    // per-lane shared-memory address of harmonic i's word for this warp's first step
    const int nb = n0 + warp * (STEPS * 32);
    int A[HMAX];
#pragma unroll
    for (int i = 1; i <= HMAX; i++) A[i - 1] = delta[i - 1] + (nb >> LG) * i + ((lane * i + HMAX / 2) >> LG);

    hsptx::mbar_wait(&bar, 0);

#pragma unroll
    for (int t = 0; t < STEPS; t++) {
        const int n = nb + 32 * t + lane;
        if (n < N) {
            hs_emit<OUT> e;
            float *plane0 = (OUT & HS_OUT_FULL) ? sums + (b * L) * (int64_t)N + n : nullptr;
            float S = win[A[HMAX - 1] + t * 32];
            e.level(0, S, plane0, N);
#pragma unroll
            for (int l = 1; l < L; l++) {
#pragma unroll
                for (int o = 1; o < (1 << l); o += 2) {
                    const int i = o * (HMAX >> l);
                    S += win[A[i - 1] + t * (32 * i / HMAX)];
                }
                e.level(l, S, plane0, N);
            }
            if (OUT & HS_OUT_REDUCED) {
                if (OUT & HS_OUT_CAND) {
                    hs_push(sink, b, n, e.m, e.a);
                } else {
                    hsptx::st_cs(vmax + b * (int64_t)N + n, e.m);
                    hsptx::st_cs(amax + b * (int64_t)N + n, (uint8_t)e.a);
                }
            }
        }
    }
}

template <int HMAX, int OUT>
int launch(const hs_plan *p, const hs_buffers &buf, int64_t batch, cudaStream_t stream)
{
    constexpr int WARPS = 8, STEPS = 4, T = WARPS * STEPS * 32;
    const int N = (int)p->nbins;
    const int tiles = (N + T - 1) / T;
    const size_t smem = (size_t)(T * (HMAX + 1) / 2 + 8 * HMAX + 8) * sizeof(float);
    auto kern = hs_std_tiled_kernel<HMAX, OUT, WARPS, STEPS>;
    // (function attributes are per device: set on every launch rather than once per process)
    HS_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const int64_t max_spectra = ((int64_t)1 << 30) / tiles;
    for (int64_t b0 = 0; b0 < batch; b0 += max_spectra) {
        const int64_t nb = (batch - b0 < max_spectra) ? batch - b0 : max_spectra;
        const int64_t off = b0 * (int64_t)N;
        hs_cand_sink sink = buf.sink;
        sink.b0 += (int)b0;
        kern<<<(unsigned)(nb * tiles), WARPS * 32, smem, stream>>>(
            buf.x + off, buf.sums ? buf.sums + off * p->L : nullptr, buf.vmax ? buf.vmax + off : nullptr,
            buf.amax ? buf.amax + off : nullptr, N, tiles, sink);
        HS_CUDA_OK(cudaGetLastError());
    }
    return HS_OK;
}

template <int HMAX>
int by_out(const hs_plan *p, const hs_buffers &buf, int64_t batch, cudaStream_t stream)
{
    switch (p->out_mode) {
        case HS_OUT_FULL: return launch<HMAX, HS_OUT_FULL>(p, buf, batch, stream);
        case HS_OUT_REDUCED:
            if (buf.sink.cand) return launch<HMAX, HS_OUT_REDUCED | HS_OUT_CAND>(p, buf, batch, stream);
            return launch<HMAX, HS_OUT_REDUCED>(p, buf, batch, stream);
        default: return launch<HMAX, HS_OUT_BOTH>(p, buf, batch, stream);
    }
}

}  // namespace

int hs_standard_tiled_launch(const hs_plan *p, const hs_buffers &buf, int64_t batch, cudaStream_t stream)
{
    switch (p->Hmax) {
        case 1: return by_out<1>(p, buf, batch, stream);
        case 2: return by_out<2>(p, buf, batch, stream);
        case 4: return by_out<4>(p, buf, batch, stream);
        case 8: return by_out<8>(p, buf, batch, stream);
        case 16: return by_out<16>(p, buf, batch, stream);
        default: return by_out<32>(p, buf, batch, stream);
    }
}

int hs_standard_tiled_launches(const hs_plan *p, int64_t batch)
{
    const int64_t tiles = (p->nbins + 1023) / 1024;
    const int64_t max_spectra = ((int64_t)1 << 30) / tiles;
    return (int)((batch + max_spectra - 1) / max_spectra);
}
