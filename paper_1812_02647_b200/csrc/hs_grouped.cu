// hs_grouped.cu — eqs. 2 and 3 (CONVENTIONS.md C2, C3, C5) in two phases per spectrum, each spectrum
// handled by a static GROUP of co-resident CTAs whose per-harmonic arrays never leave the 126 MB L2.
//
// Both variants have the form S_H(n) = sum_{i<=H} A_i(n) with a per-harmonic array that depends on x only:
//     freq-bin  A_i(n) = x~(i n)                      the stride-i decimation of the spectrum
//     Max       A_i(n) = max x~[i n .. i n + i - 1]   the maximum of the aligned block of size i
// sum_{i=2..32} |A_i| = 3.06 N words (at Hmax = 32 the arrays of sizes 2, 3, 4 are not kept: phase B takes those terms
// from the spectrum itself, 1.98 N words remain -- `stored()` below).  One persistent, cooperatively launched kernel; CTA c belongs to group
// c % groups with rank c / groups.  A group owns ONE workspace slot (3.06 N words) and walks through the spectra
// g, g + groups, g + 2 groups, ..:
//   phase A  the GS CTAs of the group share the spectrum's 4096-word chunks: chunk -> shared memory by one TMA bulk
//            copy (double buffered, the next chunk is in flight while this one is reduced), then every A_i segment
//            the chunk owns is written to the slot;
//   barrier  (group-wide: one counter in global memory, release/acquire at gpu scope)
//   phase B  the warps of the group share the spectrum's 128-bin output tiles: x and the A_i are read with unit stride
//            (float4, straight from L2), the levels accumulated, normalised and the outputs emitted;
//   barrier  before the slot is overwritten by the next spectrum's phase A.
// The two group barriers per spectrum are waited for as LATE as possible: a CTA takes its chunks top-down, so the first
// chunk of a spectrum is an upper one whose TMA wait, tables and upper-half outputs come before the wait for "slot free"
// (which sits just before the first store to the slot), and each warp waits for the phase-A arrivals inside its first
// phase-B tile, after the terms it takes from x itself (6.69 -> 5.94 ms on 4096 x 2^18).
// groups x slot is sized to the L2 budget (make_sched: 18 groups of 32 CTAs = 37 MB of slots at 2^18 bins, Hmax 32), so the A traffic (3.06 N words written, 3.06 N read per spectrum) stays in L2 and
// HBM sees x once and the outputs once: 9 B/bin in reduced mode.  No CTA ever waits for a CTA outside its group, the
// schedule is static (no work queue), and a waiting CTA shares its SM with a CTA of another group.
//
// Max, phase A.  Power-of-two block sizes: a thread reduces 8 aligned words (sizes 16 and 32 by shuffles).  Odd sizes
// j = 3, 5, 7 with their doublings: a thread reduces one whole super-block (j K_j <= 28 words) in registers.  Odd sizes
// j >= 9: the block maximum is the maximum of two overlapping sliding-window maxima of width w = 8 or 16 (tables T8,
// T16 in shared memory, built in one pass from 28 raw words per thread): max(T_w[o], T_w[o + j - w]); lane stride j
// words is conflict-free for odd j; size 2j is the union of an aligned pair of j-blocks: one shuffle-xor.
// A chunk owns the super-blocks (size j K_j, K_j the largest power of two with j K_j <= Hmax) that START inside it and
// reads a 32-word halo for those that run past its end.
#include <utility>

#include "hs_internal.cuh"
#include "hs_ptx.cuh"
#include "hs_sync.cuh"

namespace {

constexpr int kThreads = 256;
constexpr int kWarps = kThreads / 32;
constexpr int kChunk = 4096;              // phase-A input words per chunk (= 8 words per thread)
constexpr int kHalo = 32;
constexpr int kRaw = kChunk + kHalo + 32; // raw buffer: chunk + halo + zero pad read by the table build
constexpr int kTab = kChunk + kHalo;      // table entries per width
constexpr int kTileB = 128;               // phase-B outputs per warp tile (float4 per lane)
constexpr size_t kL2Budget = (size_t)56 << 20;

// Which per-harmonic arrays A_i exist.  HYB = 0: every i = 2..Hmax.  HYB = 2 (Hmax >= 8): the sizes 2, 3, 4 are evaluated
// by phase B straight from the spectrum (a window of i words per output costs no more L2 traffic than writing and
// re-reading A_i while i is small, and the slot shrinks from 3.06 N to 1.98 N words).
__host__ __device__ constexpr bool stored(int variant, int hyb, int i)
{
    (void)variant;
    if (!hyb) return true;
    return i > 4;                                // hyb == 2: phase B takes sizes 2, 3, 4 from the spectrum
}

struct gr_layout {
    int off[33];  // word offset of A_i inside a slot (multiple of 32: 128-byte rows), i = 2..Hmax
    int len[33];  // ceil(N / i): entries of A_i that can be non-zero
    int64_t slot_words;
};

gr_layout make_layout(int N, int Hmax, int variant = HS_MAX, int hyb = 0)
{
    gr_layout lay{};
    int64_t o = 0;
    for (int i = 2; i <= Hmax; i++) {
        lay.off[i] = (int)o;
        lay.len[i] = (N + i - 1) / i;
        if (!stored(variant, hyb, i)) continue;
        o += (lay.len[i] + 8 + 31) & ~31;  // padded: vector stores/loads at any n < len stay inside the row
    }
    lay.slot_words = (o + 63) & ~(int64_t)63;
    return lay;
}

struct gr_params {
    const float *x;
    float *A;        // `groups` slots of slot_words each
    float *sums;
    float *vmax;
    uint8_t *amax;
    int *ctrl;       // control block (hs_internal.cuh): [1] error flag, [2] spinning waits, [3] polls; [32 + 64 g] phase-A
                     // arrivals, [64 + 64 g] phase-B arrivals of group g
    gr_layout lay;
    int N, B;
    int groups, GS;  // number of groups, CTAs per group
    int nchunks;     // phase-A chunks per spectrum
    int ntiles;      // phase-B warp tiles per spectrum: they cover the bins below n_split
    int n_split;     // multiple of kChunk, >= N/2: the outputs of bins n >= n_split are emitted by phase A
    hs_cand_sink sink;
    unsigned spin_limit;
    float scale;     // CPLX (hs_execute_complex): x holds (re, im) pairs, x(k) = hs_power(F_k, scale)
};

constexpr int chain_len(int j, int hmax)  // K_j: largest power of two with j*K <= hmax
{
    int k = 1;
    while (j * k * 2 <= hmax) k *= 2;
    return k;
}
constexpr int ilog2c(int v) { return v <= 1 ? 0 : 1 + ilog2c(v >> 1); }

using hssync::red_release_add;

// ---------------------------------------------------------------------------------------------- phase A
// Shared-memory view of one chunk: raw[kRaw] holds x[k0 .. k0 + kChunk + kHalo) (zero beyond the spectrum, C5) and
// a zero pad; T8/T16[kTab] are the sliding-window maxima T_w[p] = max raw[p .. p + w - 1].
struct gr_smem {
    float *raw;
    float *T8, *T16;
    int2 *bounds;  // [33]: for odd j, (first, one-past-last) j-block owned by the chunk; .y already clamped to the spectrum
};

// Max: the sliding-maximum tables.  Thread t reduces the run raw[12 t .. 12 t + 27] into 12 entries of each table:
// with a lane stride of 48 bytes the 16-byte shared-memory accesses of a quarter-warp fall into distinct banks.
constexpr int kRun = 12;
static_assert(kTab % kRun == 0, "whole runs cover the tables");
static_assert(kTab + 15 < kRaw, "the last run reads inside the zero pad");
template <int HMAX>
__device__ __forceinline__ void max_tables(const gr_smem &sm)
{
#pragma unroll 1
    for (int r = threadIdx.x; r < kTab / kRun; r += kThreads) {
    const int p0 = kRun * r;
    float v[28];
#pragma unroll
    for (int q = 0; q < 7; q++) {
        const float4 t = *reinterpret_cast<const float4 *>(sm.raw + p0 + 4 * q);
        v[4 * q] = t.x, v[4 * q + 1] = t.y, v[4 * q + 2] = t.z, v[4 * q + 3] = t.w;
    }
    float a[26], b[24], c[20], d[12];
#pragma unroll
    for (int k = 0; k < 26; k++) a[k] = fmaxf(v[k], v[k + 1]);
#pragma unroll
    for (int k = 0; k < 24; k++) b[k] = fmaxf(a[k], a[k + 2]);
#pragma unroll
    for (int k = 0; k < 20; k++) c[k] = fmaxf(b[k], b[k + 4]);
#pragma unroll
    for (int k = 0; k < 12; k++) d[k] = fmaxf(c[k], c[k + 8]);
#pragma unroll
    for (int q = 0; q < 3; q++) {
        *reinterpret_cast<float4 *>(sm.T8 + p0 + 4 * q) = make_float4(c[4 * q], c[4 * q + 1], c[4 * q + 2], c[4 * q + 3]);
        if (HMAX >= 32)
            *reinterpret_cast<float4 *>(sm.T16 + p0 + 4 * q) = make_float4(d[4 * q], d[4 * q + 1], d[4 * q + 2], d[4 * q + 3]);
    }
    }
}

// Max: the power-of-two block sizes from the thread's 8 aligned raw words (sizes 16 and 32 by shuffles).
template <int HMAX, int HYB>
__device__ __forceinline__ void max_pow2(const gr_params &p, const gr_smem &sm, float *__restrict__ Ab, int k0)
{
    const int lane = threadIdx.x & 31;
#pragma unroll
    for (int h = 0; h < kChunk / (8 * kThreads); h++) {
    const int p0 = 8 * (threadIdx.x + kThreads * h), k = k0 + p0;   // k: global bin of the first word, a multiple of 8
    const float4 u = *reinterpret_cast<const float4 *>(sm.raw + p0);
    const float4 w = *reinterpret_cast<const float4 *>(sm.raw + p0 + 4);
    const float m0 = fmaxf(u.x, u.y), m1 = fmaxf(u.z, u.w), m2 = fmaxf(w.x, w.y), m3 = fmaxf(w.z, w.w);
    const float q0 = fmaxf(m0, m1), q1 = fmaxf(m2, m3);
    const float e8 = fmaxf(q0, q1);
    const float e16 = fmaxf(e8, __shfl_xor_sync(0xffffffffu, e8, 1));
    const float e32 = fmaxf(e16, __shfl_xor_sync(0xffffffffu, e16, 2));
    if (k >= p.N) continue;
    const bool whole = k + 8 <= p.N;                          // else exactly 4 bins are left (N % 4 == 0)
    if constexpr (stored(HS_MAX, HYB, 2)) {
        float *A2 = Ab + ((unsigned)p.lay.off[2] + (unsigned)(k >> 1));
        if (whole) *reinterpret_cast<float4 *>(A2) = make_float4(m0, m1, m2, m3);
        else *reinterpret_cast<float2 *>(A2) = make_float2(m0, m1);
    }
    if constexpr (HMAX >= 4 && stored(HS_MAX, HYB, 4)) {
        float *A4 = Ab + ((unsigned)p.lay.off[4] + (unsigned)(k >> 2));
        if (whole) *reinterpret_cast<float2 *>(A4) = make_float2(q0, q1);
        else A4[0] = q0;
    }
    if constexpr (HMAX >= 8 && stored(HS_MAX, HYB, 8)) Ab[(unsigned)p.lay.off[8] + (unsigned)(k >> 3)] = e8;
    if (HMAX >= 16 && (lane & 1) == 0) Ab[(unsigned)p.lay.off[16] + (unsigned)(k >> 4)] = e16;
    if (HMAX >= 32 && (lane & 3) == 0) Ab[(unsigned)p.lay.off[32] + (unsigned)(k >> 5)] = e32;
    }
}

// freq-bin: the power-of-two decimations straight from the raw words.
template <int HMAX, int HYB>
__device__ __forceinline__ void dec_pow2(const gr_params &p, const gr_smem &sm, float *__restrict__ Ab, int k0)
{
    const int lane = threadIdx.x & 31;
#pragma unroll
    for (int h = 0; h < kChunk / (8 * kThreads); h++) {
    const int p0 = 8 * (threadIdx.x + kThreads * h), k = k0 + p0;
    if (k >= p.N) continue;
    const float4 u = *reinterpret_cast<const float4 *>(sm.raw + p0);
    const float4 w = *reinterpret_cast<const float4 *>(sm.raw + p0 + 4);
    const bool whole = k + 8 <= p.N;
    if constexpr (stored(HS_FREQBIN, HYB, 2)) {
        float *A2 = Ab + ((unsigned)p.lay.off[2] + (unsigned)(k >> 1));
        if (whole) *reinterpret_cast<float4 *>(A2) = make_float4(u.x, u.z, w.x, w.z);
        else *reinterpret_cast<float2 *>(A2) = make_float2(u.x, u.z);
    }
    if constexpr (HMAX >= 4 && stored(HS_FREQBIN, HYB, 4)) {
        float *A4 = Ab + ((unsigned)p.lay.off[4] + (unsigned)(k >> 2));
        if (whole) *reinterpret_cast<float2 *>(A4) = make_float2(u.x, w.x);
        else A4[0] = u.x;
    }
    if constexpr (HMAX >= 8 && stored(HS_FREQBIN, HYB, 8)) Ab[(unsigned)p.lay.off[8] + (unsigned)(k >> 3)] = u.x;
    if (HMAX >= 16 && (lane & 1) == 0) Ab[(unsigned)p.lay.off[16] + (unsigned)(k >> 4)] = u.x;
    if (HMAX >= 32 && (lane & 3) == 0) Ab[(unsigned)p.lay.off[32] + (unsigned)(k >> 5)] = u.x;
    }
}

// store the CNT entries of size JD held in m[0..CNT) for super-block q, then halve (pairwise maxima) and recurse
template <int JD, int CNT, int HYB>
__device__ __forceinline__ void direct_levels(const gr_params &p, float *__restrict__ Ab, int q, float *m)
{
    const int n0 = CNT * q;
    const int len = p.lay.len[JD];
    float *__restrict__ g = Ab + ((unsigned)p.lay.off[JD] + (unsigned)n0);
    if constexpr (!stored(HS_MAX, HYB, JD)) {                                 // (size JD is not kept: phase B reads the spectrum)
        (void)len, (void)g;
    } else if (n0 + CNT <= len) {
        if constexpr (CNT == 8) {
            *reinterpret_cast<float4 *>(g) = make_float4(m[0], m[1], m[2], m[3]);
            *reinterpret_cast<float4 *>(g + 4) = make_float4(m[4], m[5], m[6], m[7]);
        } else if constexpr (CNT == 4) {
            *reinterpret_cast<float4 *>(g) = make_float4(m[0], m[1], m[2], m[3]);
        } else if constexpr (CNT == 2) {
            *reinterpret_cast<float2 *>(g) = make_float2(m[0], m[1]);
        } else {
            g[0] = m[0];
        }
    } else {
#pragma unroll
        for (int k = 0; k < CNT; k++)
            if (n0 + k < len) g[k] = m[k];
    }
    if constexpr (CNT > 1) {
#pragma unroll
        for (int k = 0; k < CNT / 2; k++) m[k] = fmaxf(m[2 * k], m[2 * k + 1]);
        direct_levels<JD * 2, CNT / 2, HYB>(p, Ab, q, m);
    }
}

// ---- odd sizes J = 3, 5, .., and their doublings 2J, 4J, .. <= HMAX ------------------------------------------------
// Max, J < 8: one thread reduces one whole super-block (J K words, K = chain_len) held in registers: K maxima of
// size J, then the pairwise pyramid, stored as vectors.  No table needed, ~1.6 instructions per input word.
template <int J, int HMAX, int W0, int HYB>
__device__ __forceinline__ void max_direct(const gr_params &p, const gr_smem &sm, float *__restrict__ Ab, int k0)
{
    constexpr int K = chain_len(J, HMAX), D = ilog2c(K), SB = J * K;
    constexpr int VW = SB % 4 == 0 ? 4 : SB % 2 == 0 ? 2 : 1;             // widest aligned shared-memory load
    const int tid = (threadIdx.x - 32 * W0) & (kThreads - 1);
    const int2 bd = sm.bounds[J];                                         // in blocks of size J; multiples of K
#pragma unroll 1
    for (int q = bd.x / K + tid; q < bd.y / K; q += kThreads) {           // this thread's super-blocks (one if K >= 4)
    const float *__restrict__ s = sm.raw + (SB * q - k0);
    float v[SB];
    if (VW == 4) {
#pragma unroll
        for (int t = 0; t < SB / 4; t++) {
            const float4 u = *reinterpret_cast<const float4 *>(s + 4 * t);
            v[4 * t] = u.x, v[4 * t + 1] = u.y, v[4 * t + 2] = u.z, v[4 * t + 3] = u.w;
        }
    } else if (VW == 2) {
#pragma unroll
        for (int t = 0; t < SB / 2; t++) {
            const float2 u = *reinterpret_cast<const float2 *>(s + 2 * t);
            v[2 * t] = u.x, v[2 * t + 1] = u.y;
        }
    } else {
#pragma unroll
        for (int t = 0; t < SB; t++) v[t] = s[t];
    }
    float m[K];
#pragma unroll
    for (int k = 0; k < K; k++) {
        m[k] = v[J * k];
#pragma unroll
        for (int t = 1; t < J; t++) m[k] = fmaxf(m[k], v[J * k + t]);
    }
    direct_levels<J, K, HYB>(p, Ab, q, m);
    }
}

// predicated scalar store without a branch: if (n < lim) base[idx] = v   (idx: 32-bit word offset, BYTES: immediate)
template <int BYTES>
__device__ __forceinline__ void stg_lt(int n, int lim, float *base, unsigned idx, float v)
{
    asm volatile(
        "{\n\t.reg .pred q;\n\t.reg .u64 a;\n\t"
        "setp.lt.s32 q, %0, %1;\n\t"
        "mad.wide.u32 a, %3, 4, %2;\n\t"
        "@q st.global.f32 [a+%5], %4;\n\t}" ::"r"(n),
        "r"(lim), "l"(base), "r"(idx), "f"(v), "n"(BYTES)
        : "memory");
}

// A lane per entry: NW warps (W0 .. W0 + NW - 1) take the chunk's entries of size I in rounds of 32, every address is
// base + immediate.  freq-bin: A_I[n] = raw[I n - k0] (any I that is not a power of two).  Max: odd I >= 9, the block
// maximum from two table entries, and for 2 I <= HMAX the maximum of the lane pair as A_2I[n / 2].
template <int VARIANT, int I, int HMAX, int W0, int NW>
__device__ __forceinline__ void row_pass(const gr_params &p, const gr_smem &sm, float *__restrict__ Ab, int k0)
{
    constexpr int K = VARIANT == HS_MAX ? chain_len(I, HMAX) : 1;
    static_assert(K <= 2, "row_pass handles at most one doubling");
    constexpr int W = VARIANT == HS_FREQBIN ? 1 : I < 16 ? 8 : 16;
    constexpr int ROUNDS = (kChunk / I + K + 31) / 32, TMAX = (ROUNDS + NW - 1) / NW;
    const int lane = threadIdx.x & 31;
    const int wq = ((threadIdx.x >> 5) - W0) & (kWarps - 1);
    if (wq >= NW) return;
    const int2 bd = sm.bounds[I];                                         // entries [bd.x, bd.y) belong to the chunk
    const int n = bd.x + 32 * wq + lane;
    const float *__restrict__ s = (W == 1 ? sm.raw : W == 8 ? sm.T8 : sm.T16) + (I * n - k0);
    const unsigned g1 = (unsigned)p.lay.off[I] + (unsigned)n;
    const int lim1 = min(bd.y, p.lay.len[I]);
    unsigned g2 = 0;
    int lim2 = 0;
    if (K == 2) {
        g2 = (unsigned)p.lay.off[2 * I <= 32 ? 2 * I : 32] + (unsigned)(n >> 1);
        lim2 = (lane & 1) ? 0 : min(bd.y, 2 * p.lay.len[2 * I <= 32 ? 2 * I : 32]);
    }
#pragma unroll
    for (int t = 0; t < TMAX; t++) {
            const int nt = n + 32 * NW * t;
        if (nt - lane >= bd.y) break;                                     // warp-uniform
        float v = 0.f;
        if (nt < bd.y) {
            if (VARIANT == HS_FREQBIN) v = s[I * 32 * NW * t];
            else v = fmaxf(s[I * 32 * NW * t], s[I * 32 * NW * t + I - W]);
        }
        switch (t) {   // (the byte offset must be an immediate)
#define HS_ROW_CASE(T)                                                                        \
    case T:                                                                                   \
        stg_lt<4 * 32 * NW * T>(nt, lim1, Ab, g1, v);                                        \
        if (K == 2) {                                                                         \
            const float w = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, 1));                     \
            stg_lt<4 * 16 * NW * T>(nt, lim2, Ab, g2, w);                                    \
        }                                                                                     \
        break;
            HS_ROW_CASE(0) HS_ROW_CASE(1) HS_ROW_CASE(2) HS_ROW_CASE(3) HS_ROW_CASE(4) HS_ROW_CASE(5) HS_ROW_CASE(6)
            HS_ROW_CASE(7) HS_ROW_CASE(8) HS_ROW_CASE(9) HS_ROW_CASE(10) HS_ROW_CASE(11) HS_ROW_CASE(12)
            HS_ROW_CASE(13) HS_ROW_CASE(14) HS_ROW_CASE(15)
#undef HS_ROW_CASE
            default: break;
        }
    }
    static_assert(TMAX <= 16, "more rounds per warp than row_pass unrolls");
}

// static spread of the sizes over the CTA's warps: size I gets NW warps starting at warp W0 (cumulative, modulo 16)
constexpr bool is_pow2(int v) { return (v & (v - 1)) == 0; }
constexpr bool is_direct(int variant, int I) { return variant == HS_MAX && (I & 1) && I < 8; }
constexpr bool is_row(int variant, int I) { return variant == HS_MAX ? ((I & 1) && I >= 9) : !is_pow2(I); }
constexpr int nw_of(int variant, int I, int hmax)
{
    if (is_direct(variant, I)) return (kChunk / (I * chain_len(I, hmax)) + 1 + 31) / 32;   // one super-block per thread
    if (!is_row(variant, I)) return 0;
    const int rounds = (kChunk / I + 2 + 31) / 32;
    const int r = (rounds + 3) / 6;
    return r < 1 ? 1 : r;
}
constexpr int w0_of(int variant, int I, int hmax)
{
    int w = 0;
    for (int i = 3; i < I; i++) w += nw_of(variant, i, hmax);
    return w % kWarps;
}

template <int VARIANT, int HMAX, int HYB, int I = 3>
__device__ __forceinline__ void other_sizes(const gr_params &p, const gr_smem &sm, float *__restrict__ Ab, int k0)
{
    if constexpr (I <= HMAX) {
        constexpr int W0 = w0_of(VARIANT, I, HMAX), NW = nw_of(VARIANT, I, HMAX);
        if constexpr (is_direct(VARIANT, I)) max_direct<I, HMAX, W0, HYB>(p, sm, Ab, k0);
        else if constexpr (is_row(VARIANT, I) && stored(VARIANT, HYB, I)) row_pass<VARIANT, I, HMAX, W0, NW>(p, sm, Ab, k0);
        other_sizes<VARIANT, HMAX, HYB, I + 1>(p, sm, Ab, k0);
    }
}

// Bins n >= N/2 have no harmonic but the first in range: S_H(n) = x(n) for every H, so their outputs are emitted here
// from the chunk in shared memory instead of in phase B.  h_l = x c_l is monotone in l: level 0 wins for x >= 0
// (ties included, C8), the last level for x < 0.
template <int L, int OUT>
__device__ __forceinline__ void emit_upper(const gr_params &p, const gr_smem &sm, int64_t row, int k0)
{
    const int N = p.N;
#pragma unroll
    for (int h = 0; h < kChunk / (4 * kThreads); h++) {
        const int p0 = 4 * threadIdx.x + 4 * kThreads * h, n = k0 + p0;
        if (n >= N) continue;
        const float4 x4 = *reinterpret_cast<const float4 *>(sm.raw + p0);
        if (OUT & HS_OUT_FULL) {
#pragma unroll
            for (int l = 0; l < L; l++) {
                const float c = hs_norm(l);
                hsptx::st_cs(reinterpret_cast<float4 *>(p.sums + (row * L + (int64_t)l * N + n)),
                             make_float4(x4.x * c, x4.y * c, x4.z * c, x4.w * c));
            }
        }
        if (OUT & HS_OUT_REDUCED) {
            const float c = hs_norm(L - 1);
            const float4 m = make_float4(x4.x < 0.f ? x4.x * c : x4.x, x4.y < 0.f ? x4.y * c : x4.y,
                                         x4.z < 0.f ? x4.z * c : x4.z, x4.w < 0.f ? x4.w * c : x4.w);
            const uint32_t a = (x4.x < 0.f ? (uint32_t)(L - 1) : 0u) | (x4.y < 0.f ? (uint32_t)(L - 1) << 8 : 0u) |
                               (x4.z < 0.f ? (uint32_t)(L - 1) << 16 : 0u) | (x4.w < 0.f ? (uint32_t)(L - 1) << 24 : 0u);
            if (OUT & HS_OUT_CAND) {
                if (fmaxf(fmaxf(m.x, m.y), fmaxf(m.z, m.w)) > p.sink.thr) {
                    const int64_t b = row / N;
                    hs_push(p.sink, b, n, m.x, (int)(a & 255u));
                    hs_push(p.sink, b, n + 1, m.y, (int)((a >> 8) & 255u));
                    hs_push(p.sink, b, n + 2, m.z, (int)((a >> 16) & 255u));
                    hs_push(p.sink, b, n + 3, m.w, (int)(a >> 24));
                }
            } else {
                hsptx::st_cs(reinterpret_cast<float4 *>(p.vmax + row + n), m);
                hsptx::st_cs(reinterpret_cast<uint32_t *>(p.amax + row + n), a);
            }
        }
    }
}

// all A_i segments owned by the chunk at k0 (raw is complete and zero padded; bounds are set)
template <int VARIANT, int HMAX, int HYB>
__device__ __forceinline__ void phaseA_chunk(const gr_params &p, const gr_smem &sm, float *__restrict__ Ab, int k0)
{
    if (VARIANT == HS_MAX) {
        if (HMAX >= 16) max_tables<HMAX>(sm);
        max_pow2<HMAX, HYB>(p, sm, Ab, k0);
        if (HMAX >= 16) __syncthreads();                       // tables complete
    } else {
        dec_pow2<HMAX, HYB>(p, sm, Ab, k0);
    }
    other_sizes<VARIANT, HMAX, HYB>(p, sm, Ab, k0);
}

// ---------------------------------------------------------------------------------------------- phase B
// One warp tile = 128 consecutive outputs below n_split: lane holds bins n_first + 4 lane .. +3 as one float4.
// The loads of a level are issued in batches of up to 8 float4 before they are consumed (memory-level parallelism).
// Terms of harmonic I for the outputs n .. n + 3 straight from the spectrum: the window x[I n .. I n + 4 I) as I aligned
// float4 loads (`whole`: warp-uniform, every element of the warp's windows in range), else element-wise with zero padding.
template <int VARIANT, int I, bool CPLX>
__device__ __forceinline__ void add_from_x(float4 &S, const float *__restrict__ xrow, int n, int N, bool whole, float scale)
{
    float v[4 * I];
    if (whole) {
#pragma unroll
        for (int q = 0; q < I; q++) {
            const float4 t = hs_ldx4<CPLX>(xrow, I * n + 4 * q, scale);
            v[4 * q] = t.x, v[4 * q + 1] = t.y, v[4 * q + 2] = t.z, v[4 * q + 3] = t.w;
        }
    } else {
#pragma unroll
        for (int k = 0; k < 4 * I; k++) v[k] = I * n + k < N ? hs_ldx<CPLX>(xrow, I * n + k, scale) : 0.0f;   // zero padding (C5)
    }
    float t[4];
#pragma unroll
    for (int o = 0; o < 4; o++) {
        t[o] = v[I * o];
        if (VARIANT == HS_MAX) {
#pragma unroll
            for (int k = 1; k < I; k++) t[o] = fmaxf(t[o], v[I * o + k]);
        }
    }
    S.x += t[0];
    S.y += t[1];
    S.z += t[2];
    S.w += t[3];
}

// `before_slot()` is called once, before the tile's first read from the slot (after the terms taken from x when HYB = 2):
// the warp's first tile of a spectrum waits for the group's phase-A arrivals THERE, with its x-only part already done.
template <int L, int OUT, int VARIANT = HS_MAX, int HYB = 0, bool CPLX = false, class W>
__device__ __forceinline__ void phaseB_tile(const gr_params &p, const float *__restrict__ Ab, int64_t row, int n_first, W &before_slot)
{
    const int N = p.N;
    const int n = n_first + 4 * (threadIdx.x & 31);
    const bool live = n < N;                                       // (N % 4 == 0: a float4 is wholly inside or outside)
    const float *__restrict__ xrow = p.x + row * (CPLX ? 2 : 1);
    float4 S = live ? hs_ldx4<CPLX>(xrow, n, p.scale) : make_float4(0.f, 0.f, 0.f, 0.f);
    hs_emit<OUT> e0, e1, e2, e3;
    const float *__restrict__ An = Ab + ((unsigned)n);       // A_i[n] = An[off_i]
    auto emit = [&](int l) {
        const float c = hs_norm(l);
        const float4 h = make_float4(S.x * c, S.y * c, S.z * c, S.w * c);
        if ((OUT & HS_OUT_FULL) && live) hsptx::st_cs(reinterpret_cast<float4 *>(p.sums + (row * L + (int64_t)l * N + n)), h);
        if (OUT & HS_OUT_REDUCED) {
            e0.reduce(l, h.x);
            e1.reduce(l, h.y);
            e2.reduce(l, h.z);
            e3.reduce(l, h.w);
        }
    };
    emit(0);
    bool tail = false;   // levels skipped because no harmonic of theirs is in range (reduced-only output)
    if (HYB != 2 || L <= 3) before_slot();
#pragma unroll
    for (int l = 1; l < L; l++) {
        constexpr int kBatch = 8;
        const int lo = (1 << (l - 1)) + 1, hi = 1 << l;
        if (HYB == 2 && L > 3 && l == 3) before_slot();                // (levels 1 and 2 came from the spectrum itself)
        if ((int64_t)lo * n_first < N) {                           // warp-uniform: the level has a harmonic in range
            if (HYB == 2 && l <= 2) {                              // sizes 2, 3, 4 are not kept: straight from the spectrum
                if (l == 1) {
                    add_from_x<VARIANT, 2, CPLX>(S, xrow, n, N, 2 * (n_first + kTileB) <= N, p.scale);
                } else {
                    add_from_x<VARIANT, 3, CPLX>(S, xrow, n, N, 3 * (n_first + kTileB) <= N, p.scale);
                    add_from_x<VARIANT, 4, CPLX>(S, xrow, n, N, 4 * (n_first + kTileB) <= N, p.scale);
                }
            } else if ((int64_t)hi * (n_first + kTileB) <= N) {    // warp-uniform: every element of the level in range
#pragma unroll
                for (int i0 = lo; i0 <= hi; i0 += kBatch) {
                    float4 v[kBatch];
#pragma unroll
                    for (int k = 0; k < kBatch; k++)
                        if (i0 + k <= hi) v[k] = hsptx::ld_cg(reinterpret_cast<const float4 *>(An + p.lay.off[i0 + k]));
#pragma unroll
                    for (int k = 0; k < kBatch; k++) {
                        if (i0 + k <= hi) {
                            S.x += v[k].x;
                            S.y += v[k].y;
                            S.z += v[k].z;
                            S.w += v[k].w;
                        }
                    }
                }
            } else {
#pragma unroll
                for (int i = lo; i <= hi; i++) {
                    const int len = p.lay.len[i];
                    if (n < len) {
                        const float4 v = hsptx::ld_cg(reinterpret_cast<const float4 *>(An + p.lay.off[i]));
                        S.x += v.x;                                // n < len
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
    if ((OUT & HS_OUT_REDUCED) && live && (OUT & HS_OUT_CAND)) {
        if (fmaxf(fmaxf(e0.m, e1.m), fmaxf(e2.m, e3.m)) > p.sink.thr) {
            const int64_t b = row / N;
            hs_push(p.sink, b, n, e0.m, e0.a);
            hs_push(p.sink, b, n + 1, e1.m, e1.a);
            hs_push(p.sink, b, n + 2, e2.m, e2.a);
            hs_push(p.sink, b, n + 3, e3.m, e3.a);
        }
    } else if ((OUT & HS_OUT_REDUCED) && live) {
        hsptx::st_cs(reinterpret_cast<float4 *>(p.vmax + row + n), make_float4(e0.m, e1.m, e2.m, e3.m));
        hsptx::st_cs(reinterpret_cast<uint32_t *>(p.amax + row + n),
                     (uint32_t)e0.a | ((uint32_t)e1.a << 8) | ((uint32_t)e2.a << 16) | ((uint32_t)e3.a << 24));
    }
}

// ---------------------------------------------------------------------------------------------- persistent kernel
struct gr_pos {
    int b, c;  // spectrum, chunk
};

// CPLX (hs_execute_complex): x holds the complex Fourier series.  Phase A loads the chunk with ordinary vector loads and
// forms the normalised power while writing it to shared memory (no TMA: the copy engine cannot compute); phase B forms
// the few values it reads from the spectrum on the fly.  x itself is never written to global memory.
template <int VARIANT, int HMAX, int OUT, int HYB, bool CPLX = false>
__global__ void __launch_bounds__(kThreads, 4)
gr_kernel(const __grid_constant__ gr_params p)
{
    constexpr int L = ilog2c(HMAX) + 1;
    constexpr bool kTables = VARIANT == HS_MAX && HMAX >= 16;
    constexpr int kRawBufs = kTables ? 1 : 2;     // with tables the next chunk is fetched after this one is done (other
                                                  // CTAs of the SM cover the latency); without, while it is reduced
    extern __shared__ __align__(128) float dyn[];
    __shared__ __align__(8) uint64_t bar[2];
    __shared__ int2 s_bounds[33];
    __shared__ int s_next;

    const int grp = blockIdx.x % p.groups, rank = blockIdx.x / p.groups;
    const int N = p.N;
    gr_smem sm;
    sm.T8 = dyn + kRawBufs * kRaw;
    sm.T16 = sm.T8 + (kTables && HMAX >= 32 ? kTab : 0);
    sm.bounds = s_bounds;
    float *__restrict__ Ab = p.A + (int64_t)grp * p.lay.slot_words;   // the group's slot
    int *cntA = p.ctrl + 32 + 64 * grp, *cntB = cntA + 32;

    if (threadIdx.x == 0) {
        hsptx::mbar_init(&bar[0], 1);
        hsptx::mbar_init(&bar[1], 1);
        hsptx::mbar_fence_init();
    }
    __syncthreads();

    // thread 0: start the TMA bulk copy of chunk `at` into buffer `buf` (the part that lies inside the spectrum)
    auto issue = [&](gr_pos at, int buf) {
        if (CPLX) return;                                                 // (loaded by all threads in the chunk loop)
        const int k0 = at.c * kChunk;
        const int words = min(kChunk + kHalo, N - k0);
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");     // the buffer was last written by ordinary stores
        hsptx::mbar_arrive_expect_tx(&bar[buf], (uint32_t)words * 4u);
        hsptx::bulk_g2s(dyn + buf * kRaw, p.x + (int64_t)at.b * N + k0, (uint32_t)words * 4u, &bar[buf]);
    };
    // a CTA takes the chunks rank, rank + GS, .. of a spectrum from the TOP down: the upper chunks (bins >= n_split) also
    // emit outputs, which needs nothing but x -- work that is done before the CTA waits for the slot
    const int c_top = rank + (p.nchunks - 1 - rank) / p.GS * p.GS;
    auto advance = [&](gr_pos at) {
        at.c -= p.GS;
        if (at.c < 0) {
            at.b += p.groups;
            at.c = c_top;
        }
        return at;
    };

    gr_pos cur{grp, c_top};
    int buf = 0;
    uint32_t parity = 0u;                                                 // bit `buf`: phase of that buffer's barrier
    if (threadIdx.x == 0 && cur.b < p.B) issue(cur, 0);

    for (int it = 0; cur.b < p.B; it++) {
        const int b = cur.b;
        // ---- phase A: this CTA's chunks of spectrum b.  The slot is free once every CTA of the group has finished phase B
        // of the previous spectrum: the CTA waits for that as late as possible -- after the first chunk has arrived, its
        // sliding-maximum tables are built and (upper chunks) its outputs are emitted, just before the first store to the slot.
        bool slot_free = it == 0;
        while (cur.b == b) {
            const gr_pos nxt = advance(cur);
            if (kRawBufs == 2 && threadIdx.x == 0 && nxt.b < p.B) issue(nxt, buf ^ 1);   // in flight while this chunk is reduced
            const int k0 = cur.c * kChunk;
            if (threadIdx.x >= 3 && threadIdx.x <= HMAX) {
                // entries of size i owned by the chunk: those whose super-block (i K words) starts inside it
                const int i = threadIdx.x, K = VARIANT == HS_MAX ? chain_len(i, HMAX) : 1, sb = i * K;
                const int first = K * ((k0 + sb - 1) / sb), last = K * ((k0 + kChunk + sb - 1) / sb);
                const int lenK = (p.lay.len[i] + K - 1) / K * K;          // whole super-blocks that start in the spectrum
                s_bounds[i] = make_int2(first, min(last, lenK));
            }
            sm.raw = dyn + buf * kRaw;
            const int valid = min(kChunk + kHalo, N - k0);                // words the copy delivered (multiple of 4)
            if (CPLX) {
                const float *__restrict__ frow = p.x + ((int64_t)b * N + k0) * 2;
                for (int w = 4 * threadIdx.x; w < valid; w += 4 * kThreads)
                    *reinterpret_cast<float4 *>(sm.raw + w) = hs_ldx4<true>(frow, w, p.scale);
            } else {
                hsptx::mbar_wait(&bar[buf], (parity >> buf) & 1u);
                parity ^= 1u << buf;
            }
            for (int w = valid + threadIdx.x; w < kRaw; w += kThreads) sm.raw[w] = 0.0f;   // zero padding (C5)
            __syncthreads();
            constexpr bool kTabs = VARIANT == HS_MAX && HMAX >= 16;
            if (kTabs) max_tables<HMAX>(sm);
            if (k0 >= p.n_split) emit_upper<L, OUT>(p, sm, (int64_t)b * N, k0);
            if (!slot_free) {
                if (threadIdx.x == 0) hssync::wait_count(cntB, p.GS * it, p.ctrl, p.ctrl + HS_CTRL_STATS, p.spin_limit);
                slot_free = true;
                __syncthreads();                                          // the slot is free (and the tables are complete)
            } else if (kTabs) {
                __syncthreads();                                          // tables complete
            }
            if (VARIANT == HS_MAX) max_pow2<HMAX, HYB>(p, sm, Ab, k0);
            else dec_pow2<HMAX, HYB>(p, sm, Ab, k0);
            other_sizes<VARIANT, HMAX, HYB>(p, sm, Ab, k0);
            __syncthreads();                                              // raw/tables/bounds are reused
            if (kRawBufs == 1 && threadIdx.x == 0 && nxt.b < p.B) issue(nxt, 0);
            cur = nxt;
            if (kRawBufs == 2) buf ^= 1;
        }
        if (threadIdx.x == 0) {
            s_next = 0;
            red_release_add(cntA, 1);                                     // (cumulative: ordered after the CTA's stores)
        }
        __syncthreads();
        // ---- phase B: the group's warps share the tiles; a CTA takes tiles rank, rank + GS, .. heavy (low n) first.
        // Every A_i of the spectrum is in the slot once all CTAs of the group have arrived: each WARP waits for that inside
        // its first tile, after the part of the tile that reads only x.
        const int64_t row = (int64_t)b * N;
        bool arrived = false;
        auto wait_arrivals = [&]() {
            if (arrived) return;
            if ((threadIdx.x & 31) == 0) hssync::wait_count(cntA, p.GS * (it + 1), p.ctrl, p.ctrl + HS_CTRL_STATS, p.spin_limit);
            __syncwarp();
            arrived = true;
        };
        for (;;) {
            int j = 0;
            if ((threadIdx.x & 31) == 0) j = atomicAdd(&s_next, 1);
            j = __shfl_sync(0xffffffffu, j, 0);
            const int tile = rank + p.GS * j;
            if (tile >= p.ntiles) break;
            phaseB_tile<L, OUT, VARIANT, HYB, CPLX>(p, Ab, row, tile * kTileB, wait_arrivals);
        }
        __syncthreads();                                                  // every load of the slot has returned
        if (threadIdx.x == 0) red_release_add(cntB, 1);
    }
}

// ---------------------------------------------------------------------------------------------- host side
struct gr_sched {
    int groups, GS, nchunks, ntiles, n_split;
    gr_layout lay;
};

constexpr int kCtasPerSm = 4;

// Hmax >= 8: the arrays of sizes 2, 3, 4 (1.08 N of the 3.06 N words at Hmax = 32) are not kept, phase B takes those terms
// from the spectrum (HS_GR_HYB=0 keeps every array).  eq. 2 on 4096 x 2^18: Hmax 32 6.85 -> 6.72 ms, Hmax 16 5.45 -> 4.75 ms
int gr_hyb(const hs_plan *p)
{
    if (p->Hmax < 8) return 0;
    return hs_knob("HS_GR_HYB", 2);   // measured: eq. 2 6.85 -> 6.72 ms, eq. 3 5.76 -> 4.96 ms
}

gr_sched make_sched(const hs_plan *p, int64_t batch)
{
    gr_sched s{};
    const int N = (int)p->nbins;
    s.lay = make_layout(N, p->Hmax, p->variant, gr_hyb(p));
    s.nchunks = (N + kChunk - 1) / kChunk;
    s.n_split = p->Hmax == 1 ? 0 : (int)(((int64_t)(N + 1) / 2 + kChunk - 1) / kChunk * kChunk);   // bins >= n_split: emitted by phase A
    s.ntiles = ((s.n_split < N ? s.n_split : N) + kTileB - 1) / kTileB;
    const int64_t slots = (int64_t)p->sm_count * kCtasPerSm;
    const size_t slot_bytes = (size_t)s.lay.slot_words * 4;
    // CTAs per group: the smallest power of two for which all the groups' slots together fit the L2 budget
    int GS = 1;
    while ((slots / GS) * slot_bytes > kL2Budget + kL2Budget / 8 && GS * 2 <= slots) GS *= 2;
    if (hs_knob("HS_GR_GS", 0) > 0) GS = hs_knob("HS_GR_GS", 0);
    while (GS > 1 && (GS > s.nchunks || GS > s.ntiles)) GS /= 2;
    int64_t groups = slots / GS;
    if (groups > batch) groups = batch;
    s.GS = GS;
    s.groups = (int)groups;
    return s;
}

size_t ctrl_bytes(int groups) { return (size_t)(32 + 64 * (size_t)groups) * sizeof(int); }

size_t smem_bytes(int variant, int Hmax)
{
    int tabs = 0;
    if (variant == HS_MAX) tabs = Hmax >= 32 ? 2 : Hmax >= 16 ? 1 : 0;
    return (size_t)((tabs ? 1 : 2) * kRaw + tabs * kTab) * sizeof(float);
}

template <int VARIANT, int HMAX, int OUT, int HYB, bool CPLX>
int launch_hyb_c(const hs_plan *p, const hs_buffers &buf, int64_t batch, void *ws, cudaStream_t stream)
{
    const gr_sched s = make_sched(p, batch);
    gr_params prm{};
    prm.x = buf.x;
    prm.ctrl = static_cast<int *>(ws);
    prm.A = reinterpret_cast<float *>(static_cast<char *>(ws) + (ctrl_bytes(s.groups) + 255) / 256 * 256);
    prm.sums = buf.sums;
    prm.vmax = buf.vmax;
    prm.amax = buf.amax;
    prm.sink = buf.sink;
    prm.lay = s.lay;
    prm.N = (int)p->nbins;
    prm.B = (int)batch;
    prm.groups = s.groups;
    prm.GS = s.GS;
    prm.nchunks = s.nchunks;
    prm.ntiles = s.ntiles;
    prm.n_split = s.n_split;
    prm.spin_limit = hs_spin_limit();
    prm.scale = buf.scale;
    auto kern = gr_kernel<VARIANT, HMAX, OUT, HYB, CPLX>;
    const size_t smem = smem_bytes(VARIANT, HMAX);
    // (function attributes are per device: set on every launch rather than once per process)
    HS_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int occ = 0;
    HS_CUDA_OK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, kThreads, smem));
    if (occ < kCtasPerSm) HS_FAIL(HS_ERR_CUDA);           // the groups' CTAs wait for one another: all must be resident
    HS_CUDA_OK(cudaMemsetAsync(ws, 0, ctrl_bytes(s.groups), stream));
    void *args[] = {&prm};
    // cooperative launch: fails instead of deadlocking if the grid cannot be co-resident
    HS_CUDA_OK(cudaLaunchCooperativeKernel(reinterpret_cast<const void *>(kern), dim3((unsigned)(s.groups * s.GS)),
                                           dim3(kThreads), args, smem, stream));
    return HS_OK;
}

template <int VARIANT, int HMAX, int OUT, int HYB>
int launch_hyb(const hs_plan *p, const hs_buffers &buf, int64_t batch, void *ws, cudaStream_t stream)
{
    if constexpr (VARIANT == HS_MAX && HMAX >= 8) {                      // (the complex front end: where this kernel is a default)
        if (buf.cplx) return launch_hyb_c<VARIANT, HMAX, OUT, HYB, true>(p, buf, batch, ws, stream);
    }
    if (buf.cplx) HS_FAIL(HS_ERR_INVALID_ARG);
    return launch_hyb_c<VARIANT, HMAX, OUT, HYB, false>(p, buf, batch, ws, stream);
}

template <int VARIANT, int HMAX, int OUT>
int launch(const hs_plan *p, const hs_buffers &buf, int64_t batch, void *ws, cudaStream_t stream)
{
    if constexpr (HMAX >= 8) {
        if (gr_hyb(p) == 2) return launch_hyb<VARIANT, HMAX, OUT, 2>(p, buf, batch, ws, stream);
    }
    return launch_hyb<VARIANT, HMAX, OUT, 0>(p, buf, batch, ws, stream);
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
        case 2: return by_out<VARIANT, 2>(p, buf, batch, ws, stream);
        case 4: return by_out<VARIANT, 4>(p, buf, batch, ws, stream);
        case 8: return by_out<VARIANT, 8>(p, buf, batch, ws, stream);
        case 16: return by_out<VARIANT, 16>(p, buf, batch, ws, stream);
        default: return by_out<VARIANT, 32>(p, buf, batch, ws, stream);
    }
}

}  // namespace

// One slot per group must fit the L2 budget: spectra of up to ~2^22 bins; Hmax = 1 has no phase A at all.
bool hs_grouped_supported(const hs_plan *p)
{
    if (p->variant != HS_MAX && p->variant != HS_FREQBIN) return false;
    if (p->Hmax < 2 || p->nbins > ((int64_t)1 << 23)) return false;   // (the contract of HS_ALGO_GROUPED, include/hs.h)
    const gr_sched s = make_sched(p, p->batch);
    return (size_t)s.groups * (size_t)s.lay.slot_words * 4 <= 2 * kL2Budget;
}

size_t hs_grouped_workspace_bytes(const hs_plan *p, int64_t batch)
{
    const gr_sched s = make_sched(p, batch);
    return (ctrl_bytes(s.groups) + 255) / 256 * 256 + (size_t)s.groups * (size_t)s.lay.slot_words * 4 + 256;
}

int hs_grouped_launches(const hs_plan *p, int64_t batch)
{
    (void)p;
    (void)batch;
    return 2;   // one memset node + one persistent kernel
}

int hs_grouped_launch(const hs_plan *p, const hs_buffers &buf, int64_t batch, void *ws, cudaStream_t stream)
{
    if (!ws) HS_FAIL(HS_ERR_WORKSPACE);
    if (p->variant == HS_FREQBIN) return by_hmax<HS_FREQBIN>(p, buf, batch, ws, stream);
    return by_hmax<HS_MAX>(p, buf, batch, ws, stream);
}
