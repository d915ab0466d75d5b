// hs_twophase.cu — eqs. 2 and 3 (CONVENTIONS.md C2, C3, C5) in two phases through a small ring of
// workspace slots that stays resident in the 126 MB L2, run by ONE persistent kernel.
//
// Both variants have the form S_H(n) = sum_{i<=H} A_i(n) with a per-harmonic array that depends on x only:
//     freq-bin  A_i(n) = x~(i n)                      the stride-i decimation of the spectrum
//     Max       A_i(n) = max x~[i n .. i n + i - 1]   the maximum of the aligned block of size i
// A_i has ceil(N/i) non-zero entries, sum_{i=2..32} N/i = 3.06 N words in all.  Gathering x(i n) per output touches one
// 32-byte sector per word for i >= 8 and, for Max, re-reads the spectrum once per harmonic; instead
//   phase 1 (item = one 4096-word input chunk) reads the chunk ONCE, coalesced, into shared memory and writes every
//           A_i segment it owns;
//   phase 2 (item = 4096 outputs) reads x and the A_i with unit stride (float4), accumulates the levels, normalises and
//           emits the outputs.
// Work items are handed out in order from one global counter: [phase 1 of spectrum b][phase 2 of spectrum b - D] for
// b = 0, 1, ...  A phase-2 item waits (acquire load on a per-spectrum counter) until all chunks of its spectrum are
// written; a phase-1 item waits until phase 2 of the spectrum that last used its ring slot (b - R) is finished.  Items
// only ever wait for items handed out EARLIER, so the schedule cannot deadlock, and with D of a few spectra the waits
// are never actually exercised: the lag hides them.  The ring has R = 2 D slots, a few tens of MB: the A traffic
// (3.06 N words written, 3.06 N read per spectrum) stays in L2 and HBM sees x once and the outputs once.
//
// Max, phase 1: for odd j the blocks of size j are reduced by one thread each (lane stride j words: conflict-free);
// the blocks of size 2j, 4j, .. <= Hmax are unions of aligned pairs, so they come from a shuffle-xor pyramid over
// neighbouring lanes (M_2j(n) = max(M_j(2n), M_j(2n+1))).  A chunk owns the super-blocks (size j*K_j, K_j the largest
// power of two with j*K_j <= Hmax) that START inside it, and reads a 32-word halo for those that run past its end.
#include <cstdlib>

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
    int *ctrl;       // [0] work counter, [1] error flag, [2..5] wait statistics, [16 + b] phase-1 chunks done, [16 + B + b] phase-2 tiles done
    tp_layout lay;
    int N;
    int B;
    int nchunks;     // phase-1 items per spectrum (0 when Hmax == 1)
    int ntiles;      // phase-2 items per spectrum
    int D;           // phase 2 lags phase 1 by D spectra
    int R;           // ring slots
    int discard;     // drop consumed A lines from L2 without write-back
};

constexpr int chain_len(int j, int hmax)  // K_j: largest power of two with j*K <= hmax
{
    int k = 1;
    while (j * k * 2 <= hmax) k *= 2;
    return k;
}

__device__ __forceinline__ int ld_acquire(const int *p)
{
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void red_release_add(int *p, int v)
{
    asm volatile("red.release.gpu.global.add.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// thread 0 only: wait until *cnt >= target (bounded: a bug must not hang the GPU; the error flag makes it visible)
__device__ __forceinline__ void wait_count(const int *cnt, int target, int *err, int *stat)
{
    unsigned spins = 0;
    while (ld_acquire(cnt) < target) {
        __nanosleep(64);
        if (++spins > (1u << 22) || ld_acquire(err) != 0) {
            atomicExch(err, 1);
            break;
        }
    }
    if (spins) {                      // statistics for tuning the lag: [stat] waits that had to spin, [stat+1] spins
        atomicAdd(stat, 1);
        atomicAdd(stat + 1, (int)spins);
    }
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
                    // This 128-byte line of A_i is read by exactly these 8 lanes and never again: drop it from L2 so
                    // that the dead data is not written back to HBM.  The test on v.x makes the discard wait for the load.
                    if (p.discard && (threadIdx.x & 7) == 0 && v.x == v.x)
                        asm volatile("discard.global.L2 [%0], 128;" ::"l"(An + p.lay.off[i]) : "memory");
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

// ---------------------------------------------------------------------------------------------- persistent kernel
struct tp_item {
    int kind;   // 0 = nothing to do, 1 = phase 1, 2 = phase 2
    int b;      // spectrum
    int idx;    // chunk (phase 1) or tile (phase 2)
};

__device__ __forceinline__ tp_item decode_item(const tp_params &p, int item, int64_t total)
{
    tp_item it{0, 0, 0};
    if (item >= total) return it;
    const int per_round = p.nchunks + p.ntiles;
    const int r = item / per_round, rem = item - r * per_round;
    if (rem < p.nchunks) {
        if (r < p.B) it = tp_item{1, r, rem};
    } else {
        const int b = r - p.D;
        if (b >= 0 && b < p.B) it = tp_item{2, b, rem - p.nchunks};
    }
    return it;
}

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

template <int VARIANT, int HMAX, int OUT>
__global__ void __launch_bounds__(kThreads, kMinCtasPerSm)
tp_persistent_kernel(const __grid_constant__ tp_params p)
{
    static_assert(kChunk == kTile2, "preload() addresses both phases the same way");
    constexpr int L = HMAX == 1 ? 1 : HMAX == 2 ? 2 : HMAX == 4 ? 3 : HMAX == 8 ? 4 : HMAX == 16 ? 5 : 6;
    __shared__ __align__(16) float sm[kChunk + kHalo + 16];        // + zero pad read by the table builds
    __shared__ int2 s_bounds[33];
    __shared__ int s_item[2];
    int *queue = p.ctrl, *err = p.ctrl + 1;
    int *cnt1 = p.ctrl + 16, *cnt2 = p.ctrl + 16 + p.B;
    const int64_t total = (int64_t)(p.B + p.D) * (p.nchunks + p.ntiles);
    const int N = p.N;

    if (threadIdx.x < 16) sm[kChunk + kHalo + threadIdx.x] = 0.0f;
    if (threadIdx.x == 0) {
        s_item[0] = atomicAdd(queue, 1);
        s_item[1] = atomicAdd(queue, 1);
    }
    __syncthreads();
    int item = s_item[0], next = s_item[1];
    __syncthreads();
    tp_item cur = decode_item(p, item, total);
    tp_pre pre;
    preload(p, cur, pre);
    int flip = 0;
    while (item < total) {
        int after = 0;
        if (threadIdx.x == 0) after = atomicAdd(queue, 1);           // consumed only at the end of this iteration
        const tp_item nxt = decode_item(p, next, total);
        if (cur.kind == 1) {                                         // ---- phase 1: chunk cur.idx of spectrum cur.b
            const int b = cur.b, k0 = cur.idx * kChunk;
#pragma unroll
            for (int q = 0; q < kChunk / (4 * kThreads); q++)
                reinterpret_cast<float4 *>(sm)[q * kThreads + threadIdx.x] = pre.v[q];
            if (threadIdx.x < kHalo / 4) reinterpret_cast<float4 *>(sm)[kChunk / 4 + threadIdx.x] = pre.halo;
            if (threadIdx.x >= 2 && threadIdx.x <= HMAX) {
                const int i = threadIdx.x;
                s_bounds[i] = make_int2((k0 + i - 1) / i, min((k0 + kChunk + i - 1) / i, p.lay.len[i]));
            }
            preload(p, nxt, pre);                                    // in flight while this item computes
            // the ring slot is free once phase 2 of the spectrum that used it last (b - R) has finished
            if (threadIdx.x == 0 && b >= p.R) wait_count(cnt2 + (b - p.R), p.ntiles, err, p.ctrl + 2);
            __syncthreads();
            float *Ab = p.A + (int64_t)(b % p.R) * p.lay.slot_words;
            if (VARIANT == HS_FREQBIN) decimate_chunk<HMAX>(p, sm - k0, s_bounds, Ab);
            else blockmax_chunk<HMAX>(p, sm, s_bounds, Ab, k0);
            if (threadIdx.x == 0) s_item[flip] = after;
            __syncthreads();                                         // all stores of the CTA are ordered before ...
            if (threadIdx.x == 0) red_release_add(cnt1 + b, 1);      // ... thread 0's release (cumulative, gpu scope)
        } else if (cur.kind == 2) {                                  // ---- phase 2: 4096 outputs of spectrum cur.b
            const int b = cur.b;
            const int64_t row = (int64_t)b * N;
            const int n0 = cur.idx * kTile2 + 4 * threadIdx.x;
            float4 S[kRounds2];
#pragma unroll
            for (int q = 0; q < kRounds2; q++) S[q] = pre.v[q];
            preload(p, nxt, pre);
            if (threadIdx.x == 0 && p.nchunks > 0) wait_count(cnt1 + b, p.nchunks, err, p.ctrl + 4);
            __syncthreads();
            const float *Ab = p.A + (int64_t)(b % p.R) * p.lay.slot_words;
#pragma unroll
            for (int q = 0; q < kRounds2; q++) {
                const int n = n0 + q * (4 * kThreads);
                if (n < N) phase2_round<L, OUT>(p, Ab, row, n, S[q]);
            }
            if (threadIdx.x == 0) s_item[flip] = after;
            __syncthreads();
            if (threadIdx.x == 0) red_release_add(cnt2 + b, 1);
        } else {
            preload(p, nxt, pre);
            if (threadIdx.x == 0) s_item[flip] = after;
            __syncthreads();
        }
        item = next;
        cur = nxt;
        next = s_item[flip];
        flip ^= 1;
    }
}

// ---------------------------------------------------------------------------------------------- plain two-launch path
// The same phase bodies as two ordinary kernels over a group of spectra (one CTA per item, the hardware scheduler
// instead of the work counter, stream order instead of the dependency counters).  Each kernel has its own register
// budget, so more CTAs fit per SM than in the fused persistent kernel.
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

// tuning knobs for experiments (environment, read when the schedule is built); defaults are the tuned values
int tune_int(const char *name, int dflt)
{
    const char *v = getenv(name);
    return v && *v ? atoi(v) : dflt;
}

struct tp_sched {
    int nchunks, ntiles, D, R, grid;
    bool plain;
    tp_layout lay;
};

tp_sched make_sched(const hs_plan *p, int64_t batch)
{
    tp_sched s{};
    const int N = (int)p->nbins;
    s.lay = make_layout(N, p->Hmax);
    s.nchunks = p->Hmax > 1 ? (N + kChunk - 1) / kChunk : 0;
    s.ntiles = (N + kTile2 - 1) / kTile2;
    s.grid = p->sm_count * tune_int("HS_TP_CTAS", kMinCtasPerSm);
    const int per_round = s.nchunks + s.ntiles;
    // lag: enough rounds that the CTAs in flight never reach a phase-2 item before its phase-1 items have finished
    (void)per_round;
    // Items are claimed in order but finish out of order: a CTA holds up to three claimed items (running, preloaded,
    // prefetched index), and a phase-2 item that has to spin delays the phase-1 items queued behind it in the same CTA,
    // which in turn makes later phase-2 items spin (a convoy).  Measured on B200 (profiles/r01_twophase_lag.md): with
    // 4 CTAs/SM the spinning only vanishes once phase 2 lags by about six times the items in flight, and the ring
    // needs as much slack again.  That is ~0.8 GB of workspace whatever the spectrum length; it no longer fits L2.
    const int in_flight = s.nchunks > 0 ? (6 * s.grid + s.nchunks - 1) / s.nchunks : 0;
    int D = tune_int("HS_TP_LAG", in_flight + 1);
    if (D > batch) D = (int)batch;
    if (D < 1) D = 1;
    int R = tune_int("HS_TP_RING", 4 * D);
    if (R > batch) R = (int)batch;
    if (R < D) R = D;          // (R >= D keeps slot b-R's phase 2 strictly before phase 1 of b in the item order)
    s.D = D;
    s.R = R < 1 ? 1 : R;
    s.plain = tune_int("HS_TP_MODE", 1) == 1;
    if (s.plain) {
        // plain two-launch mode: groups of up to 512 spectra (1.6 GB of A arrays at 2^18 bins); bigger groups mean
        // fewer, longer kernels (B200: 256 -> 9.8 ms, 512 -> 9.2 ms, 1024 -> 8.6 ms for eq. 2 on 4096 x 2^18)
        int64_t G = tune_int("HS_TP_RING", 0);
        if (G <= 0) {
            G = s.lay.slot_words > 0 ? ((int64_t)1600 << 20) / (s.lay.slot_words * 4) : batch;
            if (G > 65535) G = 65535;
        }
        if (G > batch) G = batch;
        s.R = G < 1 ? 1 : (int)G;
    }
    return s;
}

size_t ctrl_bytes(int64_t batch) { return (size_t)((16 + 2 * batch) * sizeof(int) + 255) / 256 * 256; }

template <int VARIANT, int HMAX, int OUT>
int launch(const hs_plan *p, const hs_buffers &buf, int64_t batch, void *ws, cudaStream_t stream)
{
    const tp_sched s = make_sched(p, batch);
    tp_params prm{};
    prm.x = buf.x;
    prm.ctrl = static_cast<int *>(ws);
    prm.A = reinterpret_cast<float *>(static_cast<char *>(ws) + ctrl_bytes(batch));
    prm.sums = buf.sums;
    prm.vmax = buf.vmax;
    prm.amax = buf.amax;
    prm.sink = buf.sink;
    prm.lay = s.lay;
    prm.N = (int)p->nbins;
    prm.B = (int)batch;
    prm.nchunks = s.nchunks;
    prm.ntiles = s.ntiles;
    prm.D = s.D;
    prm.R = s.R;
    prm.discard = tune_int("HS_TP_DISCARD", 0);
    if (s.plain) {
        // plain path: groups of R spectra, phase 1 then phase 2 in stream order
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
    HS_CUDA_OK(cudaMemsetAsync(ws, 0, ctrl_bytes(batch), stream));
    const int64_t total = (int64_t)(batch + s.D) * (s.nchunks + s.ntiles);
    const unsigned grid = (unsigned)(total < s.grid ? total : s.grid);
    tp_persistent_kernel<VARIANT, HMAX, OUT><<<grid, kThreads, 0, stream>>>(prm);
    HS_CUDA_OK(cudaGetLastError());
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
    // The work/dependency counters need batch <= 2^30 spectra and fewer than 2^31 items.
    const tp_sched s = make_sched(p, batch);
    return ctrl_bytes(batch) + (size_t)s.R * (size_t)s.lay.slot_words * 4 + 256;
}

int hs_twophase_launches(const hs_plan *p, int64_t batch)
{
    const tp_sched s = make_sched(p, batch);
    if (!s.plain) return 2;  // one memset node + one persistent kernel
    return (int)((batch + s.R - 1) / s.R) * (s.nchunks > 0 ? 2 : 1);
}

bool hs_twophase_supported(const hs_plan *p, int64_t batch)
{
    const tp_sched s = make_sched(p, batch);
    return (batch + s.D) * (int64_t)(s.nchunks + s.ntiles) < ((int64_t)1 << 31) - (int64_t)s.grid * 4;
}

int hs_twophase_launch(const hs_plan *p, const hs_buffers &buf, int64_t batch, void *ws, cudaStream_t stream)
{
    if (!ws) HS_FAIL(HS_ERR_WORKSPACE);
    if (p->variant == HS_FREQBIN) return by_hmax<HS_FREQBIN>(p, buf, batch, ws, stream);
    return by_hmax<HS_MAX>(p, buf, batch, ws, stream);
}
