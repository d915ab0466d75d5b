// hs_general.cu — the "next" rows of SURVEY.md section 8(f) that change WHAT is summed (DESIGN.md sections 15, 16):
//   * every integer H = 1..Hmax, Hmax <= 64, instead of the dyadic levels ("partial sums of an increasing
//     number of harmonics"), and eq. 2 with the window as printed, 1 <= j <= i, for the sensitivity study;
//   * the two-dimensional harmonic sum over the f - fdot plane of an acceleration search (reading R-2D:
//     harmonic i of a signal at bin n and drift z sits at (n i/H, z i/H)).
// One thread per output, loads straight from global memory through L1/L2, warp-uniform range skipping for the
// variants whose harmonics leave the spectrum (eqs. 2-4: a bin has H_Hmax in-range harmonics on average).
// No workspace.  These kernels are the first correct CUDA statement of the rows; they are measured in bench.py
// (--workload allh / plane) against their own algorithmic bytes, not tuned like the dyadic 1-D kernels.
#include "hs_internal.cuh"
#include "hs_ptx.cuh"

namespace {

constexpr int kThreads = 256;

// h_H = S_H / sqrt(H) for any integer H: fp32 multiply by the correctly rounded fp32 reciprocal root (C7 generalised),
// c_H = fp32(1 / sqrt(H)) evaluated in double: the nine-digit literals below round to exactly those values.  (The fp32
// expression 1.0f / sqrtf((float)H) rounds twice and is one ulp off for H = 6, 7, 17, 18, 21, 24, 28, 34, 39, 55, 58, 61.)
__constant__ float c_norm_any[64] = {
    1.0f, 0.707106769f, 0.577350259f, 0.5f, 0.44721359f, 0.408248305f, 0.377964467f, 0.353553385f,
    0.333333343f, 0.316227764f, 0.301511347f, 0.288675129f, 0.277350098f, 0.267261237f, 0.258198887f, 0.25f,
    0.242535621f, 0.235702261f, 0.22941573f, 0.223606795f, 0.218217894f, 0.213200718f, 0.208514407f, 0.204124153f,
    0.200000003f, 0.196116135f, 0.192450091f, 0.188982233f, 0.185695335f, 0.182574183f, 0.179605305f, 0.176776692f,
    0.17407766f, 0.171498582f, 0.169030845f, 0.166666672f, 0.164398983f, 0.162221417f, 0.160128146f, 0.158113882f,
    0.156173766f, 0.154303357f, 0.152498573f, 0.150755674f, 0.149071202f, 0.147441953f, 0.145864993f, 0.144337565f,
    0.142857149f, 0.141421363f, 0.140028015f, 0.138675049f, 0.137360558f, 0.136082768f, 0.134839967f, 0.133630618f,
    0.132453233f, 0.13130644f, 0.130188912f, 0.129099444f, 0.128036886f, 0.127000123f, 0.125988156f, 0.125f};
__device__ __forceinline__ float norm_any(int H) { return c_norm_any[H - 1]; }

// running reduced output over the levels l = H - 1 (C8: a level replaces the maximum only if strictly greater)
template <int OUT>
struct emit_any {
    float m;
    int a;
    __device__ __forceinline__ void level(int l, float S, float cn, float *__restrict__ plane0, int64_t stride)
    {
        const float h = l == 0 ? S : S * cn;               // h_1 = x bit-exactly
        if (OUT & HS_OUT_FULL) hsptx::st_cs(plane0 + (int64_t)l * stride, h);
        if (OUT & HS_OUT_REDUCED) {
            if (l == 0 || h > m) {
                m = h;
                a = l;
            }
        }
    }
};

// ------------------------------------------------------------------------------------------ every integer H, 1-D
// WINDOW: 0 = CONVENTIONS.md C2 (j = 0..i-1), 1 = as printed (j = 1..i): only eq. 2 looks at these;
//         2 = eq. 1 with interpolated terms (HS_TERM_INTERP, CONVENTIONS.md C15).
template <int VARIANT, int OUT, int WINDOW, bool JDBG>
__global__ void __launch_bounds__(kThreads)
hs_allh_kernel(const float *__restrict__ x, float *__restrict__ sums, float *__restrict__ vmax,
               uint8_t *__restrict__ amax, uint8_t *__restrict__ jdbg, int N, int Hmax, int L, hs_cand_sink sink)
{
    // L == Hmax: every integer H is a level (index H - 1); otherwise the dyadic levels only (index log2 H)
    const bool dyadic = L != Hmax;
    const int64_t b = blockIdx.y;
    const int n = blockIdx.x * kThreads + threadIdx.x;
    const int n_lo = n & ~31;                              // first bin of this warp
    if (n_lo >= N) return;
    const bool live = n < N;
    const int nn = live ? n : N - 1;                       // lanes past the end shadow the last bin and store nothing
    const int n_hi1 = min(n_lo + 32, N);                   // one past the warp's last bin
    const float *__restrict__ xb = x + b * (int64_t)N;
    float *plane0 = (OUT & HS_OUT_FULL) ? sums + (b * L) * (int64_t)N + nn : nullptr;
    uint8_t *jplane0 = JDBG ? jdbg + (b * L) * (int64_t)N + nn : nullptr;
    emit_any<OUT> e;
    e.m = 0.f, e.a = 0;

    constexpr int J0 = (VARIANT == HS_MAX && WINDOW == 1) ? 1 : 0;
    const float x1 = __ldg(xb + nn);
    // harmonic 1: x(n); with the window as printed h_1(n) = x~(n + 1), the right neighbour
    float S = J0 ? (nn + 1 < N ? __ldg(xb + nn + 1) : 0.0f) : x1;
    int j = 0;
    if (live) e.level(0, S, 1.0f, plane0, N);
    if (JDBG && live) jplane0[0] = 0;
    for (int H = 2; H <= Hmax; H++) {
        // eq. 1 sums every level from scratch: in the dyadic mode the H in between are not needed at all
        if (VARIANT == HS_STANDARD && dyadic && (H & (H - 1)) != 0) continue;
        // eqs. 2-4, reduced output only: once harmonic H is out of range for the whole warp so is every later one and S
        // stays what it is.  h = S c_H is then monotone in H, so of the remaining levels only the first (in the dyadic mode
        // it may be the first to see the last in-range harmonics) and the last can change the maximum.
        if (VARIANT != HS_STANDARD && (OUT & 3) == HS_OUT_REDUCED && !JDBG && (int64_t)H * n_lo + J0 >= N) {
            int Hf = H;
            if (dyadic) {
                Hf = 1;
                while (Hf < H) Hf <<= 1;                                // the first level at or after H
            }
            if (live && Hf <= Hmax) {
                e.level(dyadic ? 31 - __clz(Hf) : Hf - 1, S, norm_any(Hf), plane0, N);
                if (Hf != Hmax) e.level(L - 1, S, norm_any(Hmax), plane0, N);
            }
            break;
        }
        const float cn = norm_any(H);
        if (VARIANT == HS_STANDARD && WINDOW == 2) {
            // eq. 1, interpolated (C15): term i reads the line between bins q and q + 1 at n i / H = q + r / H.  (q, r) is
            // stepped exactly from i to i + 1 by adding n = a H + c.  q + 1 <= n for every i < H (and 1 < N for n = 0), so
            // the right neighbour is always inside the spectrum; r = 0 gives w = 0 and the term x(q) exactly.
            const int a = nn / H, c = nn - a * H;
            const float invH = __frcp_rn((float)H);
            int q = 0, r = 0;
            float T = x1;                                   // i = H: x(n)
            for (int i = 1; i < H; i++) {
                q += a;
                r += c;
                if (r >= H) {
                    r -= H;
                    q += 1;
                }
                const float x0 = __ldg(xb + q), xr = __ldg(xb + q + 1);
                T += __fmaf_rn(__fmul_rn((float)r, invH), xr - x0, x0);
            }
            S = T;
        } else if (VARIANT == HS_STANDARD) {
            // eq. 1 is not cumulative over consecutive H: every level from scratch.  Index of term i: nearest(n i / H),
            // half up = floor((2 n i + H) / (2 H)); stepped from i to i + 1 by adding 2 n = a (2 H) + c: no division per term.
            const int a = nn / H, c = 2 * (nn - a * H), d = 2 * H;
            int q = 0, r = H;
            float T = x1;                                   // i = H: x(n)
            for (int i = 1; i < H; i++) {
                q += a;
                r += c;
                if (r >= d) {
                    r -= d;
                    q += 1;
                }
                T += __ldg(xb + q);
            }
            S = T;
        } else {
            const int i = H;                                // eqs. 2-4 are cumulative: level H adds harmonic H
            if ((int64_t)i * n_lo + J0 < N) {               // in range for some lane (else the term is 0 and j stays)
                const bool safe = (int64_t)i * n_hi1 + J0 <= N;   // every candidate of every lane in range
                const int base = i * nn;
                if (VARIANT == HS_FREQBIN) {
                    S += (safe || base < N) ? __ldg(xb + base) : 0.0f;
                } else if (VARIANT == HS_MAX) {
                    float m = (safe || base + J0 < N) ? __ldg(xb + base + J0) : 0.0f;
                    for (int t = 1; t < i; t++) m = fmaxf(m, (safe || base + J0 + t < N) ? __ldg(xb + base + J0 + t) : 0.0f);
                    S += m;
                } else {
                    const int k = base + j;
                    const float lft = (safe || k < N) ? __ldg(xb + k) : 0.0f;
                    const float rgt = (safe || k + 1 < N) ? __ldg(xb + k + 1) : 0.0f;
                    const bool right = rgt > lft;           // strictly greater (C4)
                    S += right ? rgt : lft;
                    j += right ? 1 : 0;
                }
            }
        }
        if (dyadic && (H & (H - 1)) != 0) continue;        // (not a level: the chain just runs through it)
        const int l = dyadic ? 31 - __clz(H) : H - 1;
        if (live) e.level(l, S, cn, plane0, N);
        if (JDBG && live) jplane0[(int64_t)l * N] = (uint8_t)j;
    }
    if ((OUT & HS_OUT_REDUCED) && live) {
        if (OUT & HS_OUT_CAND) {
            hs_push(sink, b, n, e.m, e.a);
        } else {
            hsptx::st_cs(vmax + b * (int64_t)N + n, e.m);
            hsptx::st_cs(amax + b * (int64_t)N + n, (uint8_t)e.a);
        }
    }
}

template <int VARIANT, int OUT, int WINDOW, bool JDBG>
int launch_allh(const hs_plan *p, const hs_buffers &buf, int64_t batch, cudaStream_t stream)
{
    const int N = (int)p->nbins;
    const unsigned tiles = (unsigned)((N + kThreads - 1) / kThreads);
    for (int64_t b0 = 0; b0 < batch; b0 += 65535) {
        const unsigned nb = (unsigned)(batch - b0 < 65535 ? batch - b0 : 65535);
        const int64_t off = b0 * (int64_t)N;
        hs_cand_sink sink = buf.sink;
        sink.b0 += (int)b0;
        hs_allh_kernel<VARIANT, OUT, WINDOW, JDBG><<<dim3(tiles, nb), kThreads, 0, stream>>>(
            buf.x + off, buf.sums ? buf.sums + off * p->L : nullptr, buf.vmax ? buf.vmax + off : nullptr,
            buf.amax ? buf.amax + off : nullptr, buf.jdbg ? buf.jdbg + off * p->L : nullptr, N, p->Hmax, p->L, sink);
        HS_CUDA_OK(cudaGetLastError());
    }
    return HS_OK;
}

template <int VARIANT, int WINDOW>
int allh_by_out(const hs_plan *p, const hs_buffers &buf, int64_t batch, cudaStream_t stream)
{
    if constexpr (VARIANT == HS_GREEDY) {
        if (buf.jdbg) return launch_allh<VARIANT, 0, WINDOW, true>(p, buf, batch, stream);
    }
    switch (p->out_mode) {
        case HS_OUT_FULL: return launch_allh<VARIANT, HS_OUT_FULL, WINDOW, false>(p, buf, batch, stream);
        case HS_OUT_REDUCED:
            if (buf.sink.cand) return launch_allh<VARIANT, HS_OUT_REDUCED | HS_OUT_CAND, WINDOW, false>(p, buf, batch, stream);
            return launch_allh<VARIANT, HS_OUT_REDUCED, WINDOW, false>(p, buf, batch, stream);
        default: return launch_allh<VARIANT, HS_OUT_BOTH, WINDOW, false>(p, buf, batch, stream);
    }
}

// ------------------------------------------------------------------------------------------ two-dimensional sum
// Plane x[Z][N] per batch entry, row zi <-> drift z = zi - (Z-1)/2.  Dyadic levels.  grid = (tiles of n, Z, batch chunk).
//   2-D standard: term f = 1..Hmax at (floor((z f + Hmax/2)/Hmax), floor((n f + Hmax/2)/Hmax)); cumulative over the
//                 dyadic levels exactly like eq. 1 (the even-f terms of level 2H are the terms of level H, in both axes).
//   2-D freq-bin: term i at (i z, i n), zero outside the plane.
template <int VARIANT, int L, int OUT>
__global__ void __launch_bounds__(kThreads)
hs_2d_kernel(const float *__restrict__ x, float *__restrict__ sums, float *__restrict__ vmax, uint8_t *__restrict__ amax,
             int N, int Z, int zi0)
{
    constexpr int HMAX = 1 << (L - 1), LG = L - 1;
    const int n = blockIdx.x * kThreads + threadIdx.x;
    const int zi = zi0 + blockIdx.y, Zc = (Z - 1) >> 1, z = zi - Zc;
    const int64_t b = blockIdx.z;
    if (n >= N) return;
    const int64_t plane = (int64_t)Z * N;
    const float *__restrict__ xb = x + b * plane;
    float *plane0 = (OUT & HS_OUT_FULL) ? sums + (b * L) * plane + (int64_t)zi * N + n : nullptr;
    hs_emit<OUT> e;
    float S = __ldg(xb + (int64_t)zi * N + n);
    auto level = [&](int l) {
        const float h = S * hs_norm(l);
        if (OUT & HS_OUT_FULL) hsptx::st_cs(plane0 + (int64_t)l * plane, h);
        if (OUT & HS_OUT_REDUCED) e.reduce(l, h);
    };
    level(0);
    if (VARIANT == HS_STANDARD) {
#pragma unroll
        for (int l = 1; l < L; l++) {
            const int step = HMAX >> l;                    // level l adds the odd multiples of HMAX / 2^l
#pragma unroll
            for (int o = 1; o < (1 << l); o += 2) {
                const int f = o * step;
                const int k = (n * f + HMAX / 2) >> LG;
                const int zz = (z * f + HMAX / 2) >> LG;   // arithmetic shift: floor toward minus infinity
                S += __ldg(xb + (int64_t)(zz + Zc) * N + k);
            }
            level(l);
        }
    } else {
        // Harmonic i is inside the plane iff |i z| <= (Z-1)/2 (uniform for the CTA: z is its row) and i n < N; for the warp
        // that holds bins n_lo .. n_lo + 31 no harmonic beyond imax has any term: those harmonics, and the levels made of
        // them only, are skipped warp-uniformly (most rows of a plane have |z| > (Z-1)/4 and no harmonic but the first).
        const int n_lo = n & ~31;
        int imax = HMAX;
        if (z != 0) imax = min(imax, Zc / (z < 0 ? -z : z));
        if (n_lo > 0) imax = min(imax, (N - 1) / n_lo);
        bool tail = false;   // levels skipped because none of their harmonics is in range (reduced-only output)
#pragma unroll
        for (int l = 1; l < L; l++) {
            const int lo = (1 << (l - 1)) + 1, hi = 1 << l;
            if (lo <= imax) {
                for (int i = lo; i <= hi && i <= imax; i++) {
                    const int k = i * n;
                    if (k < N) S += __ldg(xb + (int64_t)(i * z + Zc) * N + k);
                }
                level(l);
            } else if ((OUT & 3) != HS_OUT_REDUCED) {
                level(l);
            } else {
                tail = true;
            }
        }
        // With S unchanged over the skipped levels h_l = S c_l is monotone in l: testing the last level alone is enough.
        if ((OUT & 3) == HS_OUT_REDUCED && tail) level(L - 1);
    }
    if (OUT & HS_OUT_REDUCED) {
        const int64_t o = b * plane + (int64_t)zi * N + n;
        hsptx::st_cs(vmax + o, e.m);
        hsptx::st_cs(amax + o, (uint8_t)e.a);
    }
}

// 2-D freq-bin, rows whose drift is so large that no harmonic but the first is inside the plane (|2 z| > (Z-1)/2: half of
// the rows): S_H = x for every H, a pure stream.  Four bins per thread; h_l = x c_l is monotone in l, so the first level
// wins for x >= 0 (ties included, C8) and the last one for x < 0.  Rows [0, rows_lo) and [Z - rows_lo, Z) of each plane.
template <int L, int OUT>
__global__ void __launch_bounds__(kThreads)
hs_2d_outer_rows_kernel(const float *__restrict__ x, float *__restrict__ sums, float *__restrict__ vmax,
                        uint8_t *__restrict__ amax, int N, int Z, int rows_lo)
{
    const int n = 4 * (blockIdx.x * kThreads + threadIdx.x);
    if (n >= N) return;
    const int r = blockIdx.y, zi = r < rows_lo ? r : Z - 2 * rows_lo + r;
    const int64_t plane = (int64_t)Z * N, o = (int64_t)blockIdx.z * plane + (int64_t)zi * N + n;
    const float4 v = __ldg(reinterpret_cast<const float4 *>(x + o));
    if (OUT & HS_OUT_FULL) {
        float *p0 = sums + ((int64_t)blockIdx.z * L) * plane + (int64_t)zi * N + n;
#pragma unroll
        for (int l = 0; l < L; l++) {
            const float c = hs_norm(l);
            hsptx::st_cs(reinterpret_cast<float4 *>(p0 + (int64_t)l * plane),
                         l == 0 ? v : make_float4(v.x * c, v.y * c, v.z * c, v.w * c));
        }
    }
    if (OUT & HS_OUT_REDUCED) {
        const float c = hs_norm(L - 1);
        hsptx::st_cs(reinterpret_cast<float4 *>(vmax + o), make_float4(v.x < 0.f ? v.x * c : v.x, v.y < 0.f ? v.y * c : v.y,
                                                                       v.z < 0.f ? v.z * c : v.z, v.w < 0.f ? v.w * c : v.w));
        hsptx::st_cs(reinterpret_cast<uint32_t *>(amax + o),
                     (v.x < 0.f ? (uint32_t)(L - 1) : 0u) | (v.y < 0.f ? (uint32_t)(L - 1) << 8 : 0u) |
                         (v.z < 0.f ? (uint32_t)(L - 1) << 16 : 0u) | (v.w < 0.f ? (uint32_t)(L - 1) << 24 : 0u));
    }
}

// rows at each edge of the plane that the streaming kernel takes (0: none, one launch per slab); also what
// hs_general_launches counts with
int outer_rows(int Z, int variant, int L)
{
    const int Zc = (Z - 1) / 2;
    return (variant == HS_FREQBIN && L > 1) ? Zc - Zc / 2 : 0;
}

template <int VARIANT, int L, int OUT>
int launch_2d(const hs_plan *p, const hs_buffers &buf, int64_t batch, cudaStream_t stream)
{
    const int N = (int)p->nbins, Z = (int)p->nz;
    const unsigned tiles = (unsigned)((N + kThreads - 1) / kThreads);
    const int64_t plane = (int64_t)Z * N;
    for (int64_t b0 = 0; b0 < batch; b0 += 65535) {
        const unsigned nb = (unsigned)(batch - b0 < 65535 ? batch - b0 : 65535);
        const int64_t off = b0 * plane;
        // freq-bin, L > 1: the rows with |2 z| > (Z-1)/2 have no harmonic but the first inside the plane: streamed (N % 4 == 0)
        const int rows_lo = outer_rows(Z, VARIANT, L);                            // rows zi < rows_lo <=> z < -(Zc / 2)
        hs_2d_kernel<VARIANT, L, OUT><<<dim3(tiles, (unsigned)(Z - 2 * rows_lo), nb), kThreads, 0, stream>>>(
            buf.x + off, buf.sums ? buf.sums + off * L : nullptr, buf.vmax ? buf.vmax + off : nullptr,
            buf.amax ? buf.amax + off : nullptr, N, Z, rows_lo);
        HS_CUDA_OK(cudaGetLastError());
        if (rows_lo > 0) {
            const unsigned t4 = (unsigned)((N / 4 + kThreads - 1) / kThreads);
            hs_2d_outer_rows_kernel<L, OUT><<<dim3(t4, (unsigned)(2 * rows_lo), nb), kThreads, 0, stream>>>(
                buf.x + off, buf.sums ? buf.sums + off * L : nullptr, buf.vmax ? buf.vmax + off : nullptr,
                buf.amax ? buf.amax + off : nullptr, N, Z, rows_lo);
            HS_CUDA_OK(cudaGetLastError());
        }
    }
    return HS_OK;
}

template <int VARIANT, int L>
int d2_by_out(const hs_plan *p, const hs_buffers &buf, int64_t batch, cudaStream_t stream)
{
    switch (p->out_mode) {
        case HS_OUT_FULL: return launch_2d<VARIANT, L, HS_OUT_FULL>(p, buf, batch, stream);
        case HS_OUT_REDUCED: return launch_2d<VARIANT, L, HS_OUT_REDUCED>(p, buf, batch, stream);
        default: return launch_2d<VARIANT, L, HS_OUT_BOTH>(p, buf, batch, stream);
    }
}

template <int VARIANT>
int d2_by_level(const hs_plan *p, const hs_buffers &buf, int64_t batch, cudaStream_t stream)
{
    switch (p->L) {
        case 1: return d2_by_out<VARIANT, 1>(p, buf, batch, stream);
        case 2: return d2_by_out<VARIANT, 2>(p, buf, batch, stream);
        case 3: return d2_by_out<VARIANT, 3>(p, buf, batch, stream);
        case 4: return d2_by_out<VARIANT, 4>(p, buf, batch, stream);
        case 5: return d2_by_out<VARIANT, 5>(p, buf, batch, stream);
        default: return d2_by_out<VARIANT, 6>(p, buf, batch, stream);
    }
}

}  // namespace

// The 2-D standard sum at Hmax 32 with reduced output on rows of whole 4096-bin tiles is eq. 1's register-blocked kernel
// with each harmonic's window taken from the plane row of its drift (hs_standard_rb.cu); it needs that kernel's tile counter.
size_t hs_general_workspace_bytes(const hs_plan *p)
{
    return (p->nz > 1 && hs_standard_rb_supported(p)) ? hs_standard_rb_workspace_bytes(p) : 0;
}

// kernel launches (memset nodes included) of one hs_launch_general over the plan's batch
int hs_general_launches(const hs_plan *p)
{
    if (hs_general_workspace_bytes(p)) return 2;                        // rb_kernel: memset node + kernel
    const int per_slab = (p->nz > 1 && outer_rows((int)p->nz, p->variant, p->L) > 0) ? 2 : 1;
    return per_slab * (int)((p->batch + 65534) / 65535);
}

int hs_launch_general(const hs_plan *p, const hs_buffers &buf, int64_t batch, void *ws, cudaStream_t stream)
{
    if (p->nz > 1) {
        if (hs_standard_rb_supported(p) && !buf.sink.cand) return hs_standard_rb_launch(p, buf, batch, ws, stream);
        if (p->variant == HS_STANDARD) return d2_by_level<HS_STANDARD>(p, buf, batch, stream);
        return d2_by_level<HS_FREQBIN>(p, buf, batch, stream);
    }
    switch (p->variant) {
        case HS_STANDARD:
            if (p->window == HS_TERM_INTERP) return allh_by_out<HS_STANDARD, 2>(p, buf, batch, stream);
            return allh_by_out<HS_STANDARD, 0>(p, buf, batch, stream);
        case HS_MAX:
            if (p->window == HS_WINDOW_PRINTED) return allh_by_out<HS_MAX, 1>(p, buf, batch, stream);
            return allh_by_out<HS_MAX, 0>(p, buf, batch, stream);
        case HS_FREQBIN: return allh_by_out<HS_FREQBIN, 0>(p, buf, batch, stream);
        default: return allh_by_out<HS_GREEDY, 0>(p, buf, batch, stream);
    }
}
