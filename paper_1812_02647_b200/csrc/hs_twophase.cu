// hs_twophase.cu — eqs. 2 and 3 (CONVENTIONS.md C2, C3, C5) in two phases as two plain kernels per
// group of spectra, the per-harmonic arrays going through HBM: the fallback for spectra whose arrays do not fit the
// L2-resident schemes (hs_ring_max.cu / hs_grouped.cu / hs_interleaved.cu), valid for any spectrum length.
//
// Both variants have the form S_H(n) = sum_{i<=H} A_i(n) with a per-harmonic array that depends on x only:
//     freq-bin  A_i(n) = x~(i n)                      the stride-i decimation of the spectrum
//     Max       A_i(n) = max x~[i n .. i n + i - 1]   the maximum of the aligned block of size i
// A_i has ceil(N/i) non-zero entries, sum_{i=2..32} N/i = 3.06 N words in all.  Gathering x(i n) per output touches one
// 32-byte sector per word for i >= 8 and, for Max, re-reads the spectrum once per harmonic; instead
//   phase 1 (one CTA per 4096-word input chunk) reads the chunk ONCE, coalesced, into shared memory and writes every
//           A_i segment it owns;
//   phase 2 (one CTA per 4096 outputs) reads x and the A_i with unit stride (float4), accumulates the levels,
//           normalises and emits the outputs.
// Stream order is the only synchronisation.  HBM traffic: x twice, the arrays written and read once, the outputs once.
//
// Max, phase 1: for odd j the blocks of size j are reduced by one thread each (lane stride j words: conflict-free);
// the blocks of size 2j, 4j, .. <= Hmax are unions of aligned pairs, so they come from a shuffle-xor pyramid over
// neighbouring lanes (M_2j(n) = max(M_j(2n), M_j(2n+1))).  A chunk owns the super-blocks (size j*K_j, K_j the largest
// power of two with j*K_j <= Hmax) that START inside it, and reads a 32-word halo for those that run past its end.
#include <mutex>

#include "hs_internal.cuh"
#include "hs_ptx.cuh"

namespace {

constexpr int kThreads = 256;
constexpr int kWarps = kThreads / 32;
constexpr int kChunk = 4096;   // phase-1 input words per item
constexpr int kHalo = 32;
constexpr int kTile2 = 4096;   // phase-2 outputs per item: 4 rounds of 256 threads x 4 bins
constexpr int kRounds2 = kTile2 / (4 * kThreads);
constexpr int kMinCtasPerSm = 4;

struct tp_layout {
    int off[33];  // word offset of A_i inside one spectrum's slot (multiple of 32: 128-byte rows), i = 2..Hmax
    int len[33];  // ceil(N / i): entries of A_i that can be non-zero
    int64_t slot_words;
};

tp_layout make_layout(int N, int Hmax)
{
    tp_layout lay{};
    int64_t o = 0;
    for (int i = 2; i <= Hmax; i++) {
        lay.off[i] = (int)o;
        lay.len[i] = (N + i - 1) / i;
        o += (lay.len[i] + 4 + 31) & ~31;  // padded so that a float4 at any n < len stays inside the row
    }
    lay.slot_words = (o + 63) & ~(int64_t)63;
    return lay;
}

struct tp_params {
    const float *x;
    float *A;        // ring of R slots, slot_words each
    float *sums;
    float *vmax;
    uint8_t *amax;
    hs_cand_sink sink;
    tp_layout lay;
    int N;
    int B;
    int nchunks;     // phase-1 items per spectrum (0 when Hmax == 1)
    int ntiles;      // phase-2 items per spectrum
    int R;           // workspace slots = spectra per kernel pair
};

constexpr int chain_len(int j, int hmax)  // K_j: largest power of two with j*K <= hmax
{
    int k = 1;
    while (j * k * 2 <= hmax) k *= 2;
    return k;
}

// ---------------------------------------------------------------------------------------------- phase 1
// Input of one item held in registers between the iteration that loads it and the one that uses it.
struct tp_pre {
    float4 v[kChunk / (4 * kThreads)];
    float4 halo;
};

// freq-bin: A_i[n] = x(i n) for the n with i n inside the chunk; [nlo, nhi) comes from the shared table.  Trip counts
// are compile-time, shared and global addresses are base + immediate.
template <int I>
__device__ __forceinline__ void decimate_one(const float *s_base /* sm - k0 */, float *__restrict__ Ai, int2 bd)
{
    constexpr int TMAX = (kChunk / I + 1 + kThreads - 1) / kThreads;
    const int n0 = bd.x + threadIdx.x;
    const float *__restrict__ s = s_base + I * n0;
    float *__restrict__ g = Ai + n0;
#pragma unroll
    for (int t = 0; t < TMAX; t++)
        if (n0 + t * kThreads < bd.y) g[t * kThreads] = s[I * t * kThreads];
}

template <int HMAX, int I = 2>
__device__ __forceinline__ void decimate_chunk(const tp_params &p, const float *s_base, const int2 *bounds, float *Ab)
{
    if constexpr (I <= HMAX) {
        decimate_one<I>(s_base, Ab + p.lay.off[I], bounds[I]);
        decimate_chunk<HMAX, I + 1>(p, s_base, bounds, Ab);
    }
}

// Max: A_i[n] = max x~[i n .. i n + i - 1] for the blocks that start inside the chunk, via sliding-maximum tables
// (a two-level sparse table): T4[x] = max w[x..x+3] and T16[x] = max w[x..x+15] are built IN PLACE in the chunk's
// shared-memory buffer (float4 per thread: read, barrier, write, barrier), and a block of size i is the maximum of
// ceil(i / TW) table entries: offsets 0, TW, 2 TW, .. and i - TW (overlapping reads are harmless for a maximum).
// That is 2-4 shared-memory reads per block instead of i, and the same base + immediate addressing as decimate_one.
template <int I, int TW>
__device__ __forceinline__ void blockmax_query(const float *s_base /* sm - k0 */, float *__restrict__ Ai, int2 bd)
{
    constexpr int TMAX = (kChunk / I + 1 + kThreads - 1) / kThreads;
    const int n0 = bd.x + threadIdx.x;
    const float *__restrict__ s = s_base + I * n0;
    float *__restrict__ g = Ai + n0;
#pragma unroll
    for (int t = 0; t < TMAX; t++) {
        if (n0 + t * kThreads < bd.y) {
            float v = s[I * t * kThreads];
#pragma unroll
            for (int o = TW; o + TW < I; o += TW) v = fmaxf(v, s[I * t * kThreads + o]);
            if (I > TW) v = fmaxf(v, s[I * t * kThreads + I - TW]);
            g[t * kThreads] = v;
        }
    }
}

template <int HMAX, int TW, int I, int IEND>
__device__ __forceinline__ void blockmax_range(const tp_params &p, const float *s_base, const int2 *bounds, float *Ab)
{
    if constexpr (I <= IEND && I <= HMAX) {
        blockmax_query<I, TW>(s_base, Ab + p.lay.off[I], bounds[I]);
        blockmax_range<HMAX, TW, I + 1, IEND>(p, s_base, bounds, Ab);
    }
}

constexpr int kGroups = (kChunk + kHalo) / 4;                       // float4 groups holding real data
constexpr int kBuildRounds = (kGroups + kThreads - 1) / kThreads;

// T_{4 w}[x] = max(T_w[x], T_w[x+w], T_w[x+2w], T_w[x+3w]) in place; W4 = w / 4 in float4 groups, or 0 for the first
// level (raw words -> T4, unaligned neighbours).
template <int W4>
__device__ __forceinline__ void build_table(float *sm)
{
    float4 *sm4 = reinterpret_cast<float4 *>(sm);
    float4 r[kBuildRounds];
#pragma unroll
    for (int q = 0; q < kBuildRounds; q++) {
        const int g = q * kThreads + threadIdx.x;
        if (g < kGroups) {
            if (W4 == 0) {
                const float4 a = sm4[g], b = sm4[g + 1];
                const float m12 = fmaxf(a.y, a.z), m23 = fmaxf(a.z, a.w), m30 = fmaxf(a.w, b.x);
                r[q] = make_float4(fmaxf(fmaxf(a.x, a.y), m23), fmaxf(m12, m30), fmaxf(m23, fmaxf(b.x, b.y)),
                                   fmaxf(m30, fmaxf(b.y, b.z)));
            } else {
                const float4 a = sm4[g], b = sm4[g + W4], c = sm4[g + 2 * W4], d = sm4[g + 3 * W4];
                r[q] = make_float4(fmaxf(fmaxf(a.x, b.x), fmaxf(c.x, d.x)), fmaxf(fmaxf(a.y, b.y), fmaxf(c.y, d.y)),
                                   fmaxf(fmaxf(a.z, b.z), fmaxf(c.z, d.z)), fmaxf(fmaxf(a.w, b.w), fmaxf(c.w, d.w)));
            }
        }
    }
    __syncthreads();
#pragma unroll
    for (int q = 0; q < kBuildRounds; q++) {
        const int g = q * kThreads + threadIdx.x;
        if (g < kGroups) sm4[g] = r[q];
    }
    __syncthreads();
}

template <int HMAX>
__device__ __forceinline__ void blockmax_chunk(const tp_params &p, float *sm, const int2 *bounds, float *Ab, int k0)
{
    const float *s_base = sm - k0;
    blockmax_range<HMAX, 1, 2, 3>(p, s_base, bounds, Ab);           // sizes 2, 3 from the raw words
    if (HMAX >= 4) {
        build_table<0>(sm);                                         // T4
        blockmax_range<HMAX, 4, 4, 15>(p, s_base, bounds, Ab);
        if (HMAX == 16) blockmax_range<HMAX, 4, 16, 16>(p, s_base, bounds, Ab);
    }
    if (HMAX >= 32) {
        build_table<1>(sm);                                         // T16
        blockmax_range<HMAX, 16, 16, 32>(p, s_base, bounds, Ab);
    }
}

// ---------------------------------------------------------------------------------------------- phase 2
template <int L, int OUT>
__device__ __forceinline__ void phase2_round(const tp_params &p, const float *__restrict__ Ab, int64_t row, int n, float4 S)
{
    const int N = p.N;
    const int n_first = n & ~127;                                  // first bin of this warp (warp = 128 bins)
    hs_emit<OUT> e0, e1, e2, e3;
    float *plane0 = (OUT & HS_OUT_FULL) ? p.sums + row * L + n : nullptr;
    const float *__restrict__ An = Ab + n;                         // A_i[n] = An[off_i]
    auto emit = [&](int l) {
        const float4 h = make_float4(S.x * hs_norm(l), S.y * hs_norm(l), S.z * hs_norm(l), S.w * hs_norm(l));
        if (OUT & HS_OUT_FULL) hsptx::st_cs(reinterpret_cast<float4 *>(plane0 + (int64_t)l * N), h);
        if (OUT & HS_OUT_REDUCED) {
            e0.reduce(l, h.x);
            e1.reduce(l, h.y);
            e2.reduce(l, h.z);
            e3.reduce(l, h.w);
        }
    };
    emit(0);
    bool tail = false;   // levels skipped because no harmonic of theirs is in range (reduced-only output)
#pragma unroll
    for (int l = 1; l < L; l++) {
        const int lo = (1 << (l - 1)) + 1, hi = 1 << l;
        if (lo * n_first < N) {                                    // warp-uniform: level has a harmonic in range
            if (hi * (n_first + 128) <= N) {                       // warp-uniform: every element of the level in range
#pragma unroll
                for (int i = lo; i <= hi; i++) {
                    const float4 v = hsptx::ld_cg(reinterpret_cast<const float4 *>(An + p.lay.off[i]));
                    S.x += v.x;
                    S.y += v.y;
                    S.z += v.z;
                    S.w += v.w;
                }
            } else {
#pragma unroll
                for (int i = lo; i <= hi; i++) {
                    const int len = p.lay.len[i];
                    if (n < len) {
                        const float4 v = hsptx::ld_cg(reinterpret_cast<const float4 *>(An + p.lay.off[i]));
                        S.x += v.x;                               // n < len
                        S.y += (n + 1 < len) ? v.y : 0.f;
                        S.z += (n + 2 < len) ? v.z : 0.f;
                        S.w += (n + 3 < len) ? v.w : 0.f;
                    }
                }
            }
            emit(l);
        } else if ((OUT & 3) != HS_OUT_REDUCED) {
            emit(l);
        } else {
            tail = true;
        }
    }
    // With S unchanged over the skipped levels, h_l = S c_l is monotone in l: for S >= 0 no later level can
    // exceed the running maximum, for S < 0 the last level is the largest.  Testing level L-1 alone is enough.
    if ((OUT & 3) == HS_OUT_REDUCED && tail) emit(L - 1);
    if ((OUT & HS_OUT_REDUCED) && (OUT & HS_OUT_CAND)) {
        if (fmaxf(fmaxf(e0.m, e1.m), fmaxf(e2.m, e3.m)) > p.sink.thr) {
            const int64_t b = row / p.N;
            hs_push(p.sink, b, n, e0.m, e0.a);
            hs_push(p.sink, b, n + 1, e1.m, e1.a);
            hs_push(p.sink, b, n + 2, e2.m, e2.a);
            hs_push(p.sink, b, n + 3, e3.m, e3.a);
        }
    } else if (OUT & HS_OUT_REDUCED) {
        hsptx::st_cs(reinterpret_cast<float4 *>(p.vmax + row + n), make_float4(e0.m, e1.m, e2.m, e3.m));
        hsptx::st_cs(reinterpret_cast<uint32_t *>(p.amax + row + n),
                     (uint32_t)e0.a | ((uint32_t)e1.a << 8) | ((uint32_t)e2.a << 16) | ((uint32_t)e3.a << 24));
    }
}

// ---------------------------------------------------------------------------------------------- kernels
struct tp_item {
    int kind;   // 0 = nothing to do, 1 = phase 1, 2 = phase 2
    int b;      // spectrum
    int idx;    // chunk (phase 1) or tile (phase 2)
};

// Issue the global loads of an item's input (x only: it never depends on another item) into registers.
__device__ __forceinline__ void preload(const tp_params &p, const tp_item &it, tp_pre &pre)
{
    const int N = p.N;
    const float *__restrict__ xb = p.x + (int64_t)it.b * N;
    const float4 zero = make_float4(0.f, 0.f, 0.f, 0.f);
    if (it.kind == 0) return;
    const int k0 = it.idx * kChunk;     // kChunk == kTile2: same addressing for both phases
#pragma unroll
    for (int q = 0; q < kChunk / (4 * kThreads); q++) {
        const int k = k0 + 4 * (q * kThreads + threadIdx.x);
        pre.v[q] = k < N ? __ldg(reinterpret_cast<const float4 *>(xb + k)) : zero;   // zero beyond the spectrum (C5)
    }
    if (it.kind == 1 && threadIdx.x < kHalo / 4) {
        const int k = k0 + kChunk + 4 * threadIdx.x;
        pre.halo = k < N ? __ldg(reinterpret_cast<const float4 *>(xb + k)) : zero;
    }
}

// The phase bodies as two ordinary kernels over a group of spectra (one CTA per item).
template <int VARIANT, int HMAX>
__global__ void __launch_bounds__(kThreads, 6)
tp_phase1_kernel(const __grid_constant__ tp_params p, int b0)
{
    __shared__ __align__(16) float sm[kChunk + kHalo + 16];
    __shared__ int2 s_bounds[33];
    const int b = b0 + blockIdx.y, chunk = blockIdx.x;
    const int k0 = chunk * kChunk, N = p.N;
    if (threadIdx.x < 16) sm[kChunk + kHalo + threadIdx.x] = 0.0f;
    tp_pre pre;
    preload(p, tp_item{1, b, chunk}, pre);
#pragma unroll
    for (int q = 0; q < kChunk / (4 * kThreads); q++) reinterpret_cast<float4 *>(sm)[q * kThreads + threadIdx.x] = pre.v[q];
    if (threadIdx.x < kHalo / 4) reinterpret_cast<float4 *>(sm)[kChunk / 4 + threadIdx.x] = pre.halo;
    if (threadIdx.x >= 2 && threadIdx.x <= HMAX) {
        const int i = threadIdx.x;
        s_bounds[i] = make_int2((k0 + i - 1) / i, min((k0 + kChunk + i - 1) / i, p.lay.len[i]));
    }
    __syncthreads();
    float *Ab = p.A + (int64_t)(b % p.R) * p.lay.slot_words;
    if (VARIANT == HS_FREQBIN) decimate_chunk<HMAX>(p, sm - k0, s_bounds, Ab);
    else blockmax_chunk<HMAX>(p, sm, s_bounds, Ab, k0);
    (void)N;
}

template <int L, int OUT>
__global__ void __launch_bounds__(kThreads, 4)
tp_phase2_kernel(const __grid_constant__ tp_params p, int b0)
{
    const int b = b0 + blockIdx.y, N = p.N;
    const int64_t row = (int64_t)b * N;
    const int n0 = blockIdx.x * kTile2 + 4 * threadIdx.x;
    const float *Ab = p.A + (int64_t)(b % p.R) * p.lay.slot_words;
    float4 S[kRounds2];
#pragma unroll
    for (int q = 0; q < kRounds2; q++) {
        const int n = n0 + q * (4 * kThreads);
        S[q] = n < N ? __ldg(reinterpret_cast<const float4 *>(p.x + row + n)) : make_float4(0.f, 0.f, 0.f, 0.f);
    }
#pragma unroll
    for (int q = 0; q < kRounds2; q++) {
        const int n = n0 + q * (4 * kThreads);
        if (n < N) phase2_round<L, OUT>(p, Ab, row, n, S[q]);
    }
}

struct tp_sched {
    int nchunks, ntiles, R;
    tp_layout lay;
};

tp_sched make_sched(const hs_plan *p, int64_t batch)
{
    tp_sched s{};
    const int N = (int)p->nbins;
    s.lay = make_layout(N, p->Hmax);
    s.nchunks = p->Hmax > 1 ? (N + kChunk - 1) / kChunk : 0;
    s.ntiles = (N + kTile2 - 1) / kTile2;
    // groups of spectra whose arrays take up to 1.6 GB: bigger groups mean fewer, longer kernels
    // (B200, eq. 2 on 4096 x 2^18: 256 spectra per group 9.8 ms, 512 9.2 ms, 1024 8.6 ms)
    int64_t G = s.lay.slot_words > 0 ? ((int64_t)1600 << 20) / (s.lay.slot_words * 4) : batch;
    if (G > 65535) G = 65535;                                          // gridDim.y
    if (G > batch) G = batch;
    s.R = G < 1 ? 1 : (int)G;
    return s;
}

template <int VARIANT, int HMAX, int OUT>
int launch(const hs_plan *p, const hs_buffers &buf, int64_t batch, void *ws, cudaStream_t stream)
{
    const tp_sched s = make_sched(p, batch);
    tp_params prm{};
    prm.x = buf.x;
    prm.A = static_cast<float *>(ws);
    prm.sums = buf.sums;
    prm.vmax = buf.vmax;
    prm.amax = buf.amax;
    prm.sink = buf.sink;
    prm.lay = s.lay;
    prm.N = (int)p->nbins;
    prm.B = (int)batch;
    prm.nchunks = s.nchunks;
    prm.ntiles = s.ntiles;
    prm.R = s.R;
    // groups of R spectra, phase 1 then phase 2 in stream order
    constexpr int L = HMAX == 1 ? 1 : HMAX == 2 ? 2 : HMAX == 4 ? 3 : HMAX == 8 ? 4 : HMAX == 16 ? 5 : 6;
    for (int64_t b0 = 0; b0 < batch; b0 += s.R) {
        const int nb = (int)((batch - b0 < s.R) ? batch - b0 : s.R);
        if (s.nchunks > 0) {
            tp_phase1_kernel<VARIANT, HMAX><<<dim3((unsigned)s.nchunks, (unsigned)nb), kThreads, 0, stream>>>(prm, (int)b0);
            HS_CUDA_OK(cudaGetLastError());
        }
        tp_phase2_kernel<L, OUT><<<dim3((unsigned)s.ntiles, (unsigned)nb), kThreads, 0, stream>>>(prm, (int)b0);
        HS_CUDA_OK(cudaGetLastError());
    }
    return HS_OK;
}

template <int VARIANT, int HMAX>
int by_out(const hs_plan *p, const hs_buffers &buf, int64_t batch, void *ws, cudaStream_t stream)
{
    switch (p->out_mode) {
        case HS_OUT_FULL: return launch<VARIANT, HMAX, HS_OUT_FULL>(p, buf, batch, ws, stream);
        case HS_OUT_REDUCED:
            if (buf.sink.cand) return launch<VARIANT, HMAX, HS_OUT_REDUCED | HS_OUT_CAND>(p, buf, batch, ws, stream);
            return launch<VARIANT, HMAX, HS_OUT_REDUCED>(p, buf, batch, ws, stream);
        default: return launch<VARIANT, HMAX, HS_OUT_BOTH>(p, buf, batch, ws, stream);
    }
}

template <int VARIANT>
int by_hmax(const hs_plan *p, const hs_buffers &buf, int64_t batch, void *ws, cudaStream_t stream)
{
    switch (p->Hmax) {
        case 1: return by_out<VARIANT, 1>(p, buf, batch, ws, stream);
        case 2: return by_out<VARIANT, 2>(p, buf, batch, ws, stream);
        case 4: return by_out<VARIANT, 4>(p, buf, batch, ws, stream);
        case 8: return by_out<VARIANT, 8>(p, buf, batch, ws, stream);
        case 16: return by_out<VARIANT, 16>(p, buf, batch, ws, stream);
        default: return by_out<VARIANT, 32>(p, buf, batch, ws, stream);
    }
}

}  // namespace

size_t hs_twophase_workspace_bytes(const hs_plan *p, int64_t batch)
{
    const tp_sched s = make_sched(p, batch);
    return (size_t)s.R * (size_t)s.lay.slot_words * 4 + 256;
}

int hs_twophase_launches(const hs_plan *p, int64_t batch)
{
    const tp_sched s = make_sched(p, batch);
    return (int)((batch + s.R - 1) / s.R) * (s.nchunks > 0 ? 2 : 1);
}

bool hs_twophase_supported(const hs_plan *p, int64_t batch)
{
    (void)batch;
    return p->variant == HS_MAX || p->variant == HS_FREQBIN;
}

int hs_twophase_launch(const hs_plan *p, const hs_buffers &buf, int64_t batch, void *ws, cudaStream_t stream)
{
    if (!ws) HS_FAIL(HS_ERR_WORKSPACE);
    if (p->variant == HS_FREQBIN) return by_hmax<HS_FREQBIN>(p, buf, batch, ws, stream);
    return by_hmax<HS_MAX>(p, buf, batch, ws, stream);
}

// ------------------------------------------------------------------------ hs_execute_static: scratch inside the library
// For callers that cannot hand the library a workspace because they cannot allocate device memory at all (a search loop
// that has banned cudaMalloc after start-up, a plug-in that is only ever given input and output buffers, a process whose
// framework holds all of the device's memory): the same two kernels, their per-harmonic arrays kept in an array that is
// part of this module's image.  See include/hs.h for the contract.  Nothing above this line is touched by it.

namespace {

// The scratch itself.  Device code may use the name; in HOST code `g_static_scratch` is only a handle for the runtime's
// symbol table (its host address is NOT where the data lives), so the launcher below asks the runtime for the device
// address and hands that to the kernels.  Each device has its own copy, allocated when this module is loaded there.
static __device__ __align__(256) unsigned char g_static_scratch[HS_STATIC_SCRATCH_BYTES];

constexpr int kMaxCachedDevices = 64;
std::mutex g_static_mutex;
void *g_static_addr[kMaxCachedDevices];   // device address of g_static_scratch per device ordinal, nullptr = not looked up

// Device address of the array on device `dev`, which must be current.  The first call per device does the look-up
// (cudaGetSymbolAddress loads the module if need be: keep it out of stream capture); later calls read the cache.
int static_scratch_address(int dev, void **out)
{
    const bool cached = dev >= 0 && dev < kMaxCachedDevices;
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (cached && g_static_addr[dev]) {
        *out = g_static_addr[dev];
        return HS_OK;
    }
    void *ptr = nullptr;
    HS_CUDA_OK(cudaGetSymbolAddress(&ptr, g_static_scratch));
    if (!ptr || (reinterpret_cast<uintptr_t>(ptr) % 256) != 0) HS_FAIL(HS_ERR_CUDA);
    if (cached) g_static_addr[dev] = ptr;
    *out = ptr;
    return HS_OK;
}

// launch<> above with the slot ring at `A` holding R spectra (instead of a caller's workspace sized by make_sched)
template <int VARIANT, int HMAX, int OUT>
int launch_in(const hs_plan *p, const hs_buffers &buf, float *A, int R, cudaStream_t stream)
{
    const int N = (int)p->nbins;
    tp_params prm{};
    prm.x = buf.x;
    prm.A = A;
    prm.sums = buf.sums;
    prm.vmax = buf.vmax;
    prm.amax = buf.amax;
    prm.sink = buf.sink;
    prm.lay = make_layout(N, p->Hmax);
    prm.N = N;
    prm.B = (int)p->batch;
    prm.nchunks = p->Hmax > 1 ? (N + kChunk - 1) / kChunk : 0;
    prm.ntiles = (N + kTile2 - 1) / kTile2;
    prm.R = R;
    constexpr int L = HMAX == 1 ? 1 : HMAX == 2 ? 2 : HMAX == 4 ? 3 : HMAX == 8 ? 4 : HMAX == 16 ? 5 : 6;
    // groups of R spectra in stream order: phase 2 of a group has read the slots before phase 1 of the next refills them
    for (int64_t b0 = 0; b0 < p->batch; b0 += R) {
        const int nb = (int)((p->batch - b0 < R) ? p->batch - b0 : R);
        if (prm.nchunks > 0) {
            tp_phase1_kernel<VARIANT, HMAX><<<dim3((unsigned)prm.nchunks, (unsigned)nb), kThreads, 0, stream>>>(prm, (int)b0);
            HS_CUDA_OK(cudaGetLastError());
        }
        tp_phase2_kernel<L, OUT><<<dim3((unsigned)prm.ntiles, (unsigned)nb), kThreads, 0, stream>>>(prm, (int)b0);
        HS_CUDA_OK(cudaGetLastError());
    }
    return HS_OK;
}

template <int VARIANT, int HMAX>
int in_by_out(const hs_plan *p, const hs_buffers &buf, float *A, int R, cudaStream_t stream)
{
    switch (p->out_mode) {
        case HS_OUT_FULL: return launch_in<VARIANT, HMAX, HS_OUT_FULL>(p, buf, A, R, stream);
        case HS_OUT_REDUCED: return launch_in<VARIANT, HMAX, HS_OUT_REDUCED>(p, buf, A, R, stream);
        default: return launch_in<VARIANT, HMAX, HS_OUT_BOTH>(p, buf, A, R, stream);
    }
}

template <int VARIANT>
int in_by_hmax(const hs_plan *p, const hs_buffers &buf, float *A, int R, cudaStream_t stream)
{
    switch (p->Hmax) {
        case 1: return in_by_out<VARIANT, 1>(p, buf, A, R, stream);
        case 2: return in_by_out<VARIANT, 2>(p, buf, A, R, stream);
        case 4: return in_by_out<VARIANT, 4>(p, buf, A, R, stream);
        case 8: return in_by_out<VARIANT, 8>(p, buf, A, R, stream);
        case 16: return in_by_out<VARIANT, 16>(p, buf, A, R, stream);
        default: return in_by_out<VARIANT, 32>(p, buf, A, R, stream);
    }
}

bool aligned16(const void *q) { return (reinterpret_cast<uintptr_t>(q) % 16) == 0; }

}  // namespace

extern "C" size_t hs_static_scratch_bytes(void) { return (size_t)HS_STATIC_SCRATCH_BYTES; }

extern "C" int hs_execute_static(const hs_plan *p, const float *d_x, float *d_sums, float *d_max, uint8_t *d_argmax,
                                 void *stream)
{
    if (!p) HS_FAIL(HS_ERR_NULL_POINTER);
    if ((p->variant != HS_MAX && p->variant != HS_FREQBIN) || p->nz != 1 || p->levels_mode != HS_LEVELS_DYADIC ||
        p->window != HS_WINDOW_C2)
        HS_FAIL(HS_ERR_INVALID_ARG);
    // how many spectra's arrays the built-in array holds; a spectrum that does not fit on its own is refused here,
    // before anything is enqueued (Hmax = 1 has no arrays: one group)
    const int64_t slot_bytes = make_layout((int)p->nbins, p->Hmax).slot_words * 4;
    int64_t R = slot_bytes > 0 ? (int64_t)HS_STATIC_SCRATCH_BYTES / slot_bytes : p->batch;
    if (R < 1) HS_FAIL(HS_ERR_SCRATCH_LIMIT);
    if (R > 65535) R = 65535;                                           // gridDim.y
    if (R > p->batch) R = p->batch;
    if (!d_x) HS_FAIL(HS_ERR_NULL_POINTER);
    if ((p->out_mode & HS_OUT_FULL) && !d_sums) HS_FAIL(HS_ERR_NULL_POINTER);
    if ((p->out_mode & HS_OUT_REDUCED) && (!d_max || !d_argmax)) HS_FAIL(HS_ERR_NULL_POINTER);
    if (!aligned16(d_x) || !aligned16(d_sums) || !aligned16(d_max) || !aligned16(d_argmax)) HS_FAIL(HS_ERR_MISALIGNED);
    int dev = -1;
    HS_CUDA_OK(cudaGetDevice(&dev));
    if (dev != p->device) HS_FAIL(HS_ERR_INVALID_ARG);
    void *scratch = nullptr;
    const int rc = static_scratch_address(dev, &scratch);
    if (rc != HS_OK) return rc;
    p->n_last_ctrl = 0;                                                 // (no control block: hs_plan_device_status -> HS_OK)
    hs_buffers buf{d_x, (p->out_mode & HS_OUT_FULL) ? d_sums : nullptr, (p->out_mode & HS_OUT_REDUCED) ? d_max : nullptr,
                   (p->out_mode & HS_OUT_REDUCED) ? d_argmax : nullptr, nullptr, {}, false, 0.0f};
    float *A = static_cast<float *>(scratch);
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    if (p->variant == HS_FREQBIN) return in_by_hmax<HS_FREQBIN>(p, buf, A, (int)R, s);
    return in_by_hmax<HS_MAX>(p, buf, A, (int)R, s);
}
