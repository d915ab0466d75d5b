// hs_interleaved.cu — eq. 3 (CONVENTIONS.md C3, C5) as a gather from a spectrum-interleaved copy of a
// small group of spectra that lives in L2, run by ONE persistent kernel.
//
// Eq. 3 reads x(i n) for i = 1..Hmax: a stride-i gather.  From the [batch][nbins] layout a warp of 32 consecutive n
// touches one 128-byte L1 line (and one 32-byte sector) per lane for large i, and the L1 of an SM looks up about one
// line per clock (profiles/r02_microbench_b200.txt): that, not HBM, bounds the plain gather (hs_greedy_gather.cu).
// Loop inversion over the batch fixes it: G = 16 spectra are first copied into a ring slot as xT[k][g] (bin-major, the
// 16 spectra of a group side by side: one 64-byte row per bin), and the gather runs with four lanes across a row
// (float4 = 4 spectra each): whole sectors whatever the stride, 4.06 words per bin between L2 and the SMs.  A group's
// copy is 16 N floats (16 MiB at 2^18 bins) in a ring of R slots that stays in L2: HBM sees x once (streamed,
// evict-first) and the outputs once (streaming stores).
// (Eq. 4 was tried on this layout in round 2, with max(x(k), x(k+1)) and the comparison bit packed into one word so
// that a harmonic costs ONE load: parity green, but 10.9 ms against the plain gather's 5.3 ms.  Greedy's 31 dependent
// loads per bin make a group's gather phase ~31 L2 latencies long whatever the item size, and a ring that covers
// throughput x that latency (Little's law: 1.4 TB/s x 50 us = 70 MB) does not fit the ~30 MB of L2 that stay dirty:
// DESIGN.md section 7.)
//
// Work items and scheduling.  Two kinds of items, each kind handed out in order from its own global counter:
//     T item: copy 512 bins x 16 spectra of a group into its ring slot; bins n >= N/2 have no harmonic but the first in
//             range (S_H(n) = x(n) for every H), so their outputs are emitted right here, in the natural layout;
//     G item: the gather for 256 bins (x 1 below N/8, x 3 above) x 16 spectra of a group, low (= long) bins first.
// A CTA is eight worker warps and one SCHEDULER warp (one active lane).  The scheduler holds up to one ticket of each
// queue (fetch-and-add) and picks whichever is runnable, gathers first: a G ticket once ALL T items of its group are
// complete, a T ticket once the gather of the group that used its ring slot last (g - R) is complete; a ticket that is
// not runnable is kept while the other kind of work goes on.  It does this WHILE the workers run the previous item:
// it publishes item k + 1 in a shared-memory mailbox, draws the replacement ticket, starts the TMA bulk copies of a T
// ticket's input rows into one of two shared-memory tiles (x is read only, so this needs nothing but the ticket
// number), and when the workers report item k done it releases its completion at gpu scope (fence + the group's
// counter).  Measured with thread 0 doing all of this between items: release 0.7 - 0.8 us + choice 1.0 us per item on
// top of item bodies of 2.6 us (T) and 6.5 us (G); with the scheduler warp 3.92 -> 3.63 ms (profiles/r02_il_items.md).
//
// Gather thread = (4 spectra of the group, C = 4 consecutive bins): one 16-byte load per bin and harmonic serves four
// spectra, the outputs of a thread are four float4 and four 4-byte stores; a warp owns 32 consecutive bins.  Range
// handling is warp-uniform: harmonic i is in range for every lane iff i (n_hi + 1) <= N.  The loads of harmonic i + 2
// are issued (cp.async into a per-thread shared-memory FIFO) before harmonic i is consumed: no staging registers.
#include "hs_internal.cuh"
#include "hs_ptx.cuh"
#include "hs_sync.cuh"

namespace {

#ifndef HS_IL_CTAS
#define HS_IL_CTAS 2
#endif
#ifndef HS_IL_G
#define HS_IL_G 16
#endif
constexpr int G = HS_IL_G;                                   // spectra per group = floats per row of xT
constexpr int C = 4;                                    // consecutive bins per gather thread (times 4 spectra)
constexpr int kThreads = 256;
constexpr int kWarps = kThreads / 32;
constexpr int kLPR = G / 4;                              // lanes per row of xT (one float4 = 4 spectra each)
constexpr int kWarpBins = (32 / kLPR) * C;              // bins per warp
constexpr int kGTile = kWarps * kWarpBins;              // 256 bins per gather tile
constexpr int kGSub = 3;                                // tiles per G item above the heavy region (bins >= N/8), 1 below
                                                        // (B200: 1 -> 4.03 ms, 2 -> 3.84, 3 -> 3.76, 4 -> 3.73 with waits, 8 -> 5.2)
#ifndef HS_IL_TBINS
#define HS_IL_TBINS 512
#endif
constexpr int kTBins = HS_IL_TBINS * 16 / G;            // bins per T item (32 KiB of input)
constexpr int kTStride = kTBins + 4;                    // shared-memory row stride (floats) of the copy tile
constexpr int kMaxRing = 3;
#ifndef HS_IL_DEPTH
#define HS_IL_DEPTH 2
#endif
constexpr int kDepth = HS_IL_DEPTH;                     // harmonics in flight per gather thread (cp.async into a per-thread FIFO)
constexpr size_t kFifoBytes = (size_t)kDepth * C * kThreads * sizeof(float4);

struct il_params {
    const float *x;
    float *xT;          // ring of R slots, slot_words each
    float *sums;
    float *vmax;
    uint8_t *amax;
    int *ctrl;          // control block (hs_internal.cuh): [0] T tickets drawn, [1] error flag, [2] times a CTA found neither of
                        // its tickets runnable, [3] polls of those, [8] G tickets drawn; [16 + g] T items done, [16 + groups + g] G items done
    unsigned spin_limit;
    int64_t slot_words;
    int N, B, groups, R;
    float scale;        // CPLX (hs_execute_complex): x holds (re, im) pairs, the copy items form x = |F|^2 scale - 1
    hs_cand_sink sink;
    int nT, nG;         // items per group
    int nHeavy;         // the first nHeavy G items are single tiles (bins below ~N/8: 8 to 32 harmonics per bin)
    int gsub;           // tiles per G item above the heavy region
    int n_split;        // G items cover bins [0, n_split); T items emit the outputs of [n_split, N)
};

// Ring data: ordinary weak loads (L1-allocating).  Coherent here because a CTA's first read of a group follows its own
// acquire of the group's counter (LDG.E.STRONG.GPU + CCTL.IVALL: the SM's L1 is invalidated) and a __syncthreads.
__device__ __forceinline__ float4 ld_ring(const float4 *p) { return *p; }

__device__ __forceinline__ float4 ld_stream(const float4 *p)   // read-once input: evict-first in L1 and L2
{
    float4 v;
    asm volatile("ld.global.cs.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
    return v;
}
// 16 bytes global -> shared, asynchronously; `bytes` = 16, or 0 to store zeros instead (the source is then not read)
__device__ __forceinline__ void cp_async16(void *dst, const void *src, int bytes)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(hsptx::smem_u32(dst)), "l"(src), "r"(bytes) : "memory");
}
__device__ __forceinline__ void cp_async16(void *dst, const void *src)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(hsptx::smem_u32(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait()
{
    asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory");
}
// ------------------------------------------------------------------------------------------------ T item
// Shared-memory tile of a copy item: row g (spectrum b0 + g) holds its kTBins bins at tile + row_off(g).  The upper
// eight rows start 8 floats later, which makes the transposed reads below conflict-free (rows are 516 floats apart).
__device__ __forceinline__ int row_off(int g) { return g * kTStride + (g & 8); }
constexpr int kTileFloats = G * kTStride + 8;

// Start the TMA bulk copies of the input of T item (group grp, bins from k0) into `tile`: one copy per spectrum row that
// exists, the part of it below N; completion on `bar`.  One thread.  x is read only: this may run long before the item.
__device__ __forceinline__ void prefetch_item(const il_params &p, float *tile, uint64_t *bar, int grp, int k0)
{
    const int64_t b0 = (int64_t)grp * G;
    const int nb = (int)min((int64_t)G, (int64_t)p.B - b0);
    const int cols = min(kTBins, p.N - k0);                              // multiple of 4 (N % 4 == 0)
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");         // the tile was last read by ordinary loads
    hsptx::mbar_arrive_expect_tx(bar, (uint32_t)nb * (uint32_t)cols * 4u);
    const uint64_t pol = hsptx::policy_evict_first();                    // read once: must not push the ring out of L2
    for (int g = 0; g < nb; g++)
        hsptx::bulk_g2s_hint(tile + row_off(g), p.x + (b0 + g) * p.N + k0, (uint32_t)cols * 4u, bar, pol);
}

// xT[k][g] = x[b0 + g][k] for g < nb, 0 for nb <= g < G, k in [k0, k0 + 512) below N; outputs of the bins >= n_split.
// The input is in `tile` already (prefetch_item, waited for by the caller) unless CPLX: the fused front end forms
// x = |F|^2 scale - 1 here while loading, and x is never written to HBM.
template <int L, int OUT, bool CPLX, class F>
__device__ __forceinline__ void copy_item(const il_params &p, float *tile, int grp, int k0, float *__restrict__ xT, F &redraw)
{
    const int N = p.N;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t b0 = (int64_t)grp * G;
    const int nb = (int)min((int64_t)G, (int64_t)p.B - b0);
    constexpr int SPW = G / kWarps;                      // spectra per warp (2)
    constexpr int Q = kTBins / 128;                      // float4 per lane per spectrum (4)
    float4 v[SPW][Q];
#pragma unroll
    for (int s = 0; s < SPW; s++) {
        const int g = warp * SPW + s;
#pragma unroll
        for (int q = 0; q < Q; q++) {
            const int kk = 4 * (lane + 32 * q), k = k0 + kk;
            v[s][q] = make_float4(0.f, 0.f, 0.f, 0.f);
            if (g < nb && k < N) {
                if (CPLX) {
                    const float4 *f = reinterpret_cast<const float4 *>(p.x + ((b0 + g) * N + k) * 2);
                    const float4 a = ld_stream(f), c = ld_stream(f + 1);
                    v[s][q] = make_float4(hs_power(a.x, a.y, p.scale), hs_power(a.z, a.w, p.scale),
                                          hs_power(c.x, c.y, p.scale), hs_power(c.z, c.w, p.scale));
                } else {
                    v[s][q] = *reinterpret_cast<const float4 *>(tile + row_off(g) + kk);
                }
            }
        }
    }
    redraw();                                           // (thread 0: the next item, while the loads are in flight)
#pragma unroll
    for (int s = 0; s < SPW; s++) {
        const int g = warp * SPW + s;
#pragma unroll
        for (int q = 0; q < Q; q++) {
            const int kk = 4 * (lane + 32 * q);
            if (CPLX) *reinterpret_cast<float4 *>(tile + row_off(g) + kk) = v[s][q];
            const int k = k0 + kk;
            if (k >= p.n_split && k < N && g < nb) {     // S_H(n) = x(n) for every H: emit in the natural layout
                const int64_t row = (b0 + g) * N;
                hs_emit<OUT> e0, e1, e2, e3;
#pragma unroll
                for (int l = 0; l < L; l++) {
                    // h_l = x c_l is monotone in l: in reduced-only mode the first and the last level decide
                    if ((OUT & 3) == HS_OUT_REDUCED && l != 0 && l != L - 1) continue;
                    const float4 h = make_float4(v[s][q].x * hs_norm(l), v[s][q].y * hs_norm(l), v[s][q].z * hs_norm(l),
                                                 v[s][q].w * hs_norm(l));
                    if (OUT & HS_OUT_FULL) hsptx::st_cs(reinterpret_cast<float4 *>(p.sums + (row * L + (int64_t)l * N + k)), h);
                    if (OUT & HS_OUT_REDUCED) {
                        e0.reduce(l, h.x);
                        e1.reduce(l, h.y);
                        e2.reduce(l, h.z);
                        e3.reduce(l, h.w);
                    }
                }
                if ((OUT & HS_OUT_REDUCED) && (OUT & HS_OUT_CAND)) {
                    if (fmaxf(fmaxf(e0.m, e1.m), fmaxf(e2.m, e3.m)) > p.sink.thr) {
                        hs_push(p.sink, b0 + g, k, e0.m, e0.a);
                        hs_push(p.sink, b0 + g, k + 1, e1.m, e1.a);
                        hs_push(p.sink, b0 + g, k + 2, e2.m, e2.a);
                        hs_push(p.sink, b0 + g, k + 3, e3.m, e3.a);
                    }
                } else if (OUT & HS_OUT_REDUCED) {
                    hsptx::st_cs(reinterpret_cast<float4 *>(p.vmax + row + k), make_float4(e0.m, e1.m, e2.m, e3.m));
                    hsptx::st_cs(reinterpret_cast<uint32_t *>(p.amax + row + k),
                                 (uint32_t)e0.a | ((uint32_t)e1.a << 8) | ((uint32_t)e2.a << 16) | ((uint32_t)e3.a << 24));
                }
            }
        }
    }
    if (CPLX) asm volatile("bar.sync 1, %0;" ::"n"(kThreads) : "memory");   // (the worker warps; the scheduler warp is not part of it)
    // thread t writes the float4 of spectra 4 (t % 4) .. +3 at bins k0 + t / 4 + 64 q; rows the group does not have are zero
    const int g4 = (threadIdx.x & (kLPR - 1)) * 4;
    const float *t0 = tile + row_off(g4);
    const int have = nb - g4;                            // rows g4 .. g4 + have - 1 exist
#pragma unroll
    for (int q = 0; q < kTBins / (kThreads / kLPR); q++) {
        const int kk = q * (kThreads / kLPR) + (threadIdx.x / kLPR);
        if (k0 + kk < N) {
            const float *t = t0 + kk;
            const float4 o = make_float4(have > 0 ? t[0] : 0.f, have > 1 ? t[kTStride] : 0.f, have > 2 ? t[2 * kTStride] : 0.f,
                                         have > 3 ? t[3 * kTStride] : 0.f);
            *reinterpret_cast<float4 *>(xT + (int64_t)(k0 + kk) * G + g4) = o;
        }
    }
}

// ------------------------------------------------------------------------------------------------ G item
// One tile of 256 bins x 16 spectra.  Thread = (4 spectra, 4 consecutive bins): one 16-byte load per bin and harmonic
// serves four spectra; a warp owns 32 consecutive bins, and per output row it stores 128 contiguous bytes of maxima
// and 32 of best levels.
template <int L, int OUT, class F>
__device__ __forceinline__ void gather_item(const il_params &p, int grp, int n_cta, const float *xT, float4 *fifo, F &redraw)
{
    const int N = p.N;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int q4 = lane & (kLPR - 1);                                           // spectra 4 q4 .. 4 q4 + 3 of the group
    const int n_w = n_cta + warp * kWarpBins;                          // first bin of this warp
    const int n_end = min(N, p.n_split);                               // bins [n_end, N) belong to the T items
    if (n_w >= n_end) {                                                // (warp-uniform)
        redraw();
        return;
    }
    const int n0 = n_w + (lane / kLPR) * C;                              // first bin of this thread
    const int n_hi1 = min(n_w + kWarpBins, n_end);                     // one past the warp's last bin
    const bool whole = n_w + kWarpBins <= n_end;                       // every lane's C bins exist
    const int64_t b0 = (int64_t)grp * G + 4 * q4;                      // first of this thread's spectra
    const float4 *xq = reinterpret_cast<const float4 *>(xT) + q4;                // row k: xq[k * (G / 4)]
    constexpr int RS = G / 4;                                          // float4 per row

    float4 S[C];
    hs_emit<OUT> e[C][4];

    auto emit = [&](int l) {
        const float c = hs_norm(l);
#pragma unroll
        for (int k = 0; k < C; k++) {
            if (OUT & HS_OUT_REDUCED) {
                e[k][0].reduce(l, S[k].x * c);
                e[k][1].reduce(l, S[k].y * c);
                e[k][2].reduce(l, S[k].z * c);
                e[k][3].reduce(l, S[k].w * c);
            }
        }
        if (OUT & HS_OUT_FULL) {
#pragma unroll
            for (int q = 0; q < 4; q++) {
                if (b0 + q < p.B) {
                    float *pl = p.sums + ((b0 + q) * L + l) * N + n0;
                    const float h0 = (q == 0 ? S[0].x : q == 1 ? S[0].y : q == 2 ? S[0].z : S[0].w) * c;
                    const float h1 = (q == 0 ? S[1].x : q == 1 ? S[1].y : q == 2 ? S[1].z : S[1].w) * c;
                    const float h2 = (q == 0 ? S[2].x : q == 1 ? S[2].y : q == 2 ? S[2].z : S[2].w) * c;
                    const float h3 = (q == 0 ? S[3].x : q == 1 ? S[3].y : q == 2 ? S[3].z : S[3].w) * c;
                    if (whole) {
                        hsptx::st_cs(reinterpret_cast<float4 *>(pl), make_float4(h0, h1, h2, h3));
                    } else {
                        if (n0 + 0 < n_end) hsptx::st_cs(pl + 0, h0);
                        if (n0 + 1 < n_end) hsptx::st_cs(pl + 1, h1);
                        if (n0 + 2 < n_end) hsptx::st_cs(pl + 2, h2);
                        if (n0 + 3 < n_end) hsptx::st_cs(pl + 3, h3);
                    }
                }
            }
        }
    };
    auto add = [](float4 &a, const float4 &b) {
        a.x += b.x;
        a.y += b.y;
        a.z += b.z;
        a.w += b.w;
    };
    const float4 zero = make_float4(0.f, 0.f, 0.f, 0.f);

    // The harmonics 2 .. imax (the last one in range for some lane of the warp) are fetched kDepth ahead of their use by
    // cp.async into a FIFO of this thread's own (stage d, bin k) -> fifo[(d C + k) kThreads + thread]: the loads in flight
    // cost no registers, and a thread only ever reads what it copied itself (no barrier; cp.async.wait_group orders it).
    constexpr int HM = 1 << (L - 1);
    int imax = 1;
    if (n_w > 0) {
        const int q = (N - 1) / n_w;                                   // harmonic i has a bin below N for the warp iff i n_w < N
        imax = q < HM ? q : HM;
    } else {
        imax = HM;
    }
    float4 *mine = fifo + threadIdx.x;
    auto fetch = [&](int i) {                                          // harmonic i -> stage i % kDepth (one commit group)
        if (i <= imax) {
            float4 *dst = mine + (i % kDepth) * (C * kThreads);
            const int base = i * n0;
            if (whole && i * n_hi1 <= N) {                             // in range for every lane: no bounds checks
#pragma unroll
                for (int k = 0; k < C; k++) cp_async16(dst + k * kThreads, xq + (base + k * i) * RS);
            } else {                                                   // straddling the end of the spectrum: zero padding (C5)
#pragma unroll
                for (int k = 0; k < C; k++) {
                    const int r = base + k * i;
                    cp_async16(dst + k * kThreads, xq + (r < N ? r : 0) * RS, r < N ? 16 : 0);
                }
            }
        }
        cp_async_commit();
    };
#pragma unroll
    for (int d = 0; d < kDepth; d++) fetch(2 + d);

    // harmonic 1
#pragma unroll
    for (int k = 0; k < C; k++) S[k] = (whole || n0 + k < N) ? ld_ring(xq + (n0 + k) * RS) : zero;
    redraw();                                                        // (thread 0: the next item, while the loads are in flight)
    emit(0);

    bool tail = false;   // levels skipped because none of their harmonics is in range for the warp (reduced only)
#pragma unroll
    for (int l = 1; l < L; l++) {
        const int lo = (1 << (l - 1)) + 1, hi = 1 << l;
        if (lo <= imax) {
            for (int i = lo; i <= hi && i <= imax; i++) {
                cp_async_wait<kDepth - 1>();                           // harmonic i has landed
                const float4 *src = mine + (i % kDepth) * (C * kThreads);
                float4 v[C];
#pragma unroll
                for (int k = 0; k < C; k++) v[k] = src[k * kThreads];
#pragma unroll
                for (int k = 0; k < C; k++) add(S[k], v[k]);
                fetch(i + kDepth);                                     // refill the stage
            }
            emit(l);
        } else if ((OUT & 3) != HS_OUT_REDUCED) {
            emit(l);
        } else {
            tail = true;
        }
    }
    cp_async_wait<0>();
    // With S unchanged over the skipped levels h_l = S c_l is monotone in l: testing the last level alone is enough.
    if ((OUT & 3) == HS_OUT_REDUCED && tail) emit(L - 1);

    if (OUT & HS_OUT_REDUCED) {
#pragma unroll
        for (int q = 0; q < 4; q++) {
            if (b0 + q < p.B && (OUT & HS_OUT_CAND)) {
#pragma unroll
                for (int k = 0; k < C; k++)
                    if (n0 + k < n_end) hs_push(p.sink, b0 + q, n0 + k, e[k][q].m, e[k][q].a);
            } else if (b0 + q < p.B) {
                float *pm = p.vmax + (b0 + q) * N + n0;
                uint8_t *pa = p.amax + (b0 + q) * N + n0;
                if (whole) {
                    hsptx::st_cs(reinterpret_cast<float4 *>(pm), make_float4(e[0][q].m, e[1][q].m, e[2][q].m, e[3][q].m));
                    hsptx::st_cs(reinterpret_cast<uint32_t *>(pa), (uint32_t)e[0][q].a | ((uint32_t)e[1][q].a << 8) |
                                                                       ((uint32_t)e[2][q].a << 16) | ((uint32_t)e[3][q].a << 24));
                } else {
#pragma unroll
                    for (int k = 0; k < C; k++) {
                        if (n0 + k < n_end) {
                            hsptx::st_cs(pm + k, e[k][q].m);
                            hsptx::st_cs(pa + k, (uint8_t)e[k][q].a);
                        }
                    }
                }
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------ persistent kernel
using hssync::kNoTicket;
using il_tickets = hssync::tickets;
constexpr int kItemG = 1 << 30;

// CTA = 8 worker warps + 1 scheduler warp (one active lane).  The scheduler owns the tickets: while the workers run item
// k it draws replacement tickets, starts the TMA prefetch of a T ticket's input, and picks item k + 1 (whichever ticket in
// hand is runnable, gathers first) and publishes it; when the workers report item k done it releases the item's
// completion at gpu scope (fence + counter) -- after the workers have already gone on to item k + 1.  None of the
// latencies of scheduling (ticket atomics, polls of the groups' counters, the release fence: ~2 us per item, a third
// of an item's time when thread 0 of the CTA did this between items) is on the workers' path any more.
// If no ticket is runnable while item k is still running, the scheduler first waits for item k and releases it (item
// k + 1 may depend on it) and only then waits for a ticket to become runnable.
template <int L, int OUT, bool CPLX>
__global__ void __launch_bounds__(kThreads + 32, HS_IL_CTAS)
il_persistent_kernel(const __grid_constant__ il_params p)
{
    // dynamic shared memory: the gather items' FIFO, then two tiles for the copy items (the input of the T ticket in
    // hand is prefetched into the tile that is not in use while the CTA is busy with another item)
    extern __shared__ __align__(128) unsigned char dyn_smem[];
    float4 *fifo = reinterpret_cast<float4 *>(dyn_smem);
    float *tiles = reinterpret_cast<float *>(dyn_smem + kFifoBytes);
    __shared__ __align__(8) uint64_t tbar[2];      // a tile's input has landed (TMA)
    // Mailboxes between the scheduler and the workers: monotonic counters (no phase parity that could be lapped)
    __shared__ int s_done[4];                      // worker warps that have finished item k: slot k & 3 (the workers are never more
                                                   // than one item apart, but NOT in lockstep: one counter per item, not a running sum)
    __shared__ int s_pub;                          // items the scheduler has published
    __shared__ int s_item[2], s_buf[2];            // item k is in slot k & 1
    if (threadIdx.x == 0) {
        hsptx::mbar_init(&tbar[0], 1);
        hsptx::mbar_init(&tbar[1], 1);
        hsptx::mbar_fence_init();
        s_done[0] = s_done[1] = s_done[2] = s_done[3] = 0;
        s_pub = 0;
    }
    __syncthreads();

    if (threadIdx.x >= kThreads) {                                      // ---------------- scheduler warp
        if (threadIdx.x != kThreads) return;
        il_tickets q;
        q.tq = p.ctrl + HS_CTRL_QUEUE;
        q.gq = p.ctrl + 8;
        q.doneT = p.ctrl + 16;
        q.doneG = p.ctrl + 16 + p.groups;
        q.nT = p.nT;
        q.nG = p.nG;
        q.R = p.R;
        q.totalT = p.groups * p.nT;
        q.totalG = p.groups * p.nG;
        q.readyT = -1;
        q.freeG = -1;                                                   // (groups below R have a fresh slot: ts - R <= -1)
        q.gt = q.tt = kNoTicket;
        int pft[2] = {kNoTicket, kNoTicket};                            // the T ticket whose input is in tile b (or on its way)
        int nft[2] = {0, 0};                                            // prefetches started into tile b (phase of tbar[b] = count - 1)
        // start the TMA copies for T ticket `t` unless it has a tile already; returns its tile, or -1 if none is free
        auto fetch = [&](int t) -> int {
            if (pft[0] == t) return 0;
            if (pft[1] == t) return 1;
            const int bsel = pft[0] == kNoTicket ? 0 : pft[1] == kNoTicket ? 1 : -1;
            if (bsel < 0) return -1;
            const int s = t / p.nT, idx = t - s * p.nT;
            if (!CPLX) prefetch_item(p, tiles + bsel * kTileFloats, &tbar[bsel], s, idx * kTBins);
            nft[bsel]++;
            pft[bsel] = t;
            return bsel;
        };
        auto publish = [&](int k, int it) {                             // item number k (its parity selects the mailbox)
            int bsel = 0;
            if (it >= 0 && !(it & kItemG)) bsel = fetch(it);            // (a tile is free: at most one other T item is in flight)
            *(volatile int *)&s_item[k & 1] = it;
            *(volatile int *)&s_buf[k & 1] = bsel;
            __threadfence_block();
            *(volatile int *)&s_pub = k + 1;
            q.draw_g();                                                 // replacement tickets, and the held T ticket's input
            q.draw_t();
            if (q.tt >= 0) (void)fetch(q.tt);
        };
        int cur = q.next(p.ctrl, p.spin_limit, kItemG);                 // kNoTicket: nothing to do at all
        publish(0, cur);
        for (int k = 0; cur != kNoTicket; k++) {
            int nxt = q.try_next(kItemG);
            bool published = false;
            if (nxt != kNoTicket) {
                if (nxt == hssync::kExhausted) nxt = kNoTicket;
                publish(k + 1, nxt);
                published = true;
            }
            while (*(volatile int *)&s_done[k & 3] < kWarps) {          // every worker warp has finished item k
            }
            *(volatile int *)&s_done[k & 3] = 0;                        // (item k + 4 is published three iterations from now)
            __threadfence();                                            // their stores, cumulatively, before the release at gpu scope
            if (!(cur & kItemG)) {
                atomicAdd(q.doneT + cur / p.nT, 1);
                pft[pft[0] == cur ? 0 : 1] = kNoTicket;                 // (the tile has been read by everybody)
            } else {
                atomicAdd(q.doneG + (cur & (kItemG - 1)) / p.nG, 1);
            }
            if (!published) {
                nxt = q.next(p.ctrl, p.spin_limit, kItemG);
                publish(k + 1, nxt);
            } else if (q.tt >= 0) {
                (void)fetch(q.tt);                                      // (a tile may have become free)
            }
            cur = nxt;
        }
        // Every published item has been finished by the workers, but a T ticket still in hand (a bounded wait gave up
        // before it became runnable) may have its input on the way: the CTA must not exit with a bulk copy in flight into
        // its shared memory, so wait for that copy to land (it always does; nobody reads it).
        if (!CPLX) {
#pragma unroll
            for (int b = 0; b < 2; b++)
                if (pft[b] != kNoTicket) hsptx::mbar_wait(&tbar[b], (uint32_t)(nft[b] - 1) & 1u);
        }
        return;
    }

    // ---------------- worker warps
    auto nothing = []() {};
    uint32_t tphase = 0u;                                               // bit b: parity of the next wait on tbar[b]
    for (int k = 0;; k++) {
        while (*(volatile int *)&s_pub <= k) {
        }
        __threadfence_block();
        const int item = *(volatile int *)&s_item[k & 1], tb = *(volatile int *)&s_buf[k & 1];
        if (item == kNoTicket) break;
        if (!(item & kItemG)) {                                         // ---- T item
            const int s = item / p.nT, idx = item - s * p.nT;
            float *xT = p.xT + (int64_t)(s % p.R) * p.slot_words;
            if (!CPLX) {
                hsptx::mbar_wait(&tbar[tb], (tphase >> tb) & 1u);
                tphase ^= 1u << tb;
            }
            copy_item<L, OUT, CPLX>(p, tiles + tb * kTileFloats, s, idx * kTBins, xT, nothing);
        } else {                                                        // ---- G item
            const int gi = item & (kItemG - 1);
            const int grp = gi / p.nG, qi = gi - grp * p.nG;
            const float *xT = p.xT + (int64_t)(grp % p.R) * p.slot_words;
            if (qi < p.nHeavy) {
                gather_item<L, OUT>(p, grp, qi * kGTile, xT, fifo, nothing);
            } else {
#pragma unroll 1
                for (int sub = 0; sub < p.gsub; sub++) {
                    const int t = p.nHeavy + (qi - p.nHeavy) * p.gsub + sub;
                    gather_item<L, OUT>(p, grp, t * kGTile, xT, fifo, nothing);
                }
            }
        }
        // every load of this warp from the ring / the tile has returned (their values were consumed) and its stores are
        // issued: one arrival per warp (release at CTA scope; the scheduler's fence makes them visible at gpu scope)
        __syncwarp();
        if ((threadIdx.x & 31) == 0) {
            __threadfence_block();
            atomicAdd(&s_done[k & 3], 1);
        }
    }
}

struct il_sched {
    int groups, R, nT, nG, nHeavy, gsub, n_split;
    int64_t slot_words;
};
constexpr int kCtasPerSm = HS_IL_CTAS;                                  // (__launch_bounds__ of the kernel)

il_sched make_sched(const hs_plan *p, int64_t batch)
{
    il_sched s{};
    const int N = (int)p->nbins;
    s.groups = (int)((batch + G - 1) / G);
    s.nT = (N + kTBins - 1) / kTBins;
    // bins n >= N/2 have S_H(n) = x(n): the T items emit them.  The split is a multiple of the T tile.
    const int half = (N + 1) / 2;
    int split = (half + kTBins - 1) / kTBins * kTBins;
    if (p->Hmax == 1) split = 0;                                       // nothing to gather at all
    const int gt = kGTile;
    if (split > N) split = (N + gt - 1) / gt * gt;                      // (only spectra shorter than a T tile)
    s.n_split = split;
    const int tiles = (((split < N) ? split : N) + gt - 1) / gt;
    s.nHeavy = (N / 8 + gt - 1) / gt;
    if (s.nHeavy > tiles) s.nHeavy = tiles;
    s.gsub = hs_knob("HS_IL_GSUB", kGSub);
    if (s.gsub < 1) s.gsub = 1;
    s.nG = s.nHeavy + (tiles - s.nHeavy + s.gsub - 1) / s.gsub;
    s.slot_words = ((int64_t)N * G + 63) & ~(int64_t)63;
    // Ring slots: the copies run ahead of the gathers by at most R groups.  Three 16 MiB slots (2^18 bins) keep the
    // resident CTAs busy; shorter spectra need more groups in flight for that (about two items per resident CTA),
    // within the same 48 MiB.
    const int64_t slot_bytes = s.slot_words * 4;
    // (measured with the scheduler warp: as many slots as fit 48 MiB -- 2^16 bins: 5 slots 4.3 ms, 12 slots 3.51 ms;
    // 2^17 bins: 4 slots 4.06 ms, 6 slots 3.54 ms on 2^30 bins)
    const int64_t cap = ((int64_t)48 << 20) / slot_bytes;
    int64_t R = cap;
    if (R < kMaxRing) R = slot_bytes > ((int64_t)16 << 20) ? 2 : kMaxRing;   // (2^19-bin spectra: two 32 MiB slots)
    R = hs_knob("HS_IL_RING", (int)R);
    if (R < 2) R = 2;
    s.R = (int)(s.groups < R ? s.groups : R);
    return s;
}

size_t ctrl_bytes(int groups) { return ((size_t)(16 + 2 * (size_t)groups) * sizeof(int) + 255) / 256 * 256; }

template <int L, int OUT, bool CPLX>
int launch_c(const hs_plan *p, const hs_buffers &buf, int64_t batch, void *ws, cudaStream_t stream)
{
    const il_sched s = make_sched(p, batch);
    il_params prm{};
    prm.x = buf.x;
    prm.ctrl = static_cast<int *>(ws);
    prm.xT = reinterpret_cast<float *>(static_cast<char *>(ws) + ctrl_bytes(s.groups));
    prm.sums = buf.sums;
    prm.vmax = buf.vmax;
    prm.amax = buf.amax;
    prm.sink = buf.sink;
    prm.slot_words = s.slot_words;
    prm.N = (int)p->nbins;
    prm.B = (int)batch;
    prm.groups = s.groups;
    prm.R = s.R;
    prm.scale = buf.scale;
    prm.spin_limit = hs_spin_limit();
    prm.nT = s.nT;
    prm.nG = s.nG;
    prm.nHeavy = s.nHeavy;
    prm.gsub = s.gsub;
    prm.n_split = s.n_split;
    auto kern = il_persistent_kernel<L, OUT, CPLX>;
    const size_t smem = kFifoBytes + 2 * (size_t)kTileFloats * sizeof(float);
    HS_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int occ = 0;                                                        // (per device: asked on every launch)
    HS_CUDA_OK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, kThreads + 32, smem));
    const int ctas_per_sm = occ > 0 ? occ : 1;
    HS_CUDA_OK(cudaMemsetAsync(ws, 0, ctrl_bytes(s.groups), stream));
    const int64_t total = (int64_t)s.groups * (s.nT + s.nG);
    const int64_t slots = (int64_t)p->sm_count * ctas_per_sm;
    kern<<<(unsigned)(total < slots ? total : slots), kThreads + 32, smem, stream>>>(prm);
    HS_CUDA_OK(cudaGetLastError());
    return HS_OK;
}

template <int L, int OUT>
int launch(const hs_plan *p, const hs_buffers &buf, int64_t batch, void *ws, cudaStream_t stream)
{
    if (buf.cplx) return launch_c<L, OUT, true>(p, buf, batch, ws, stream);
    return launch_c<L, OUT, false>(p, buf, batch, ws, stream);
}

template <int L>
int by_out(const hs_plan *p, const hs_buffers &buf, int64_t batch, void *ws, cudaStream_t stream)
{
    switch (p->out_mode) {
        case HS_OUT_FULL: return launch<L, HS_OUT_FULL>(p, buf, batch, ws, stream);
        case HS_OUT_REDUCED:
            if (buf.sink.cand) return launch<L, HS_OUT_REDUCED | HS_OUT_CAND>(p, buf, batch, ws, stream);
            return launch<L, HS_OUT_REDUCED>(p, buf, batch, ws, stream);
        default: return launch<L, HS_OUT_BOTH>(p, buf, batch, ws, stream);
    }
}

int by_level(const hs_plan *p, const hs_buffers &buf, int64_t batch, void *ws, cudaStream_t stream)
{
    switch (p->L) {
        case 2: return by_out<2>(p, buf, batch, ws, stream);
        case 3: return by_out<3>(p, buf, batch, ws, stream);
        case 4: return by_out<4>(p, buf, batch, ws, stream);
        case 5: return by_out<5>(p, buf, batch, ws, stream);
        default: return by_out<6>(p, buf, batch, ws, stream);
    }
}

}  // namespace

// The interleaved copies of a ring of groups have to stay in L2 (126 MB): three slots of up to 16 MiB (spectra of up to
// 2^18 bins) or two of 32 MiB (2^19 bins: 8.66 ms against the plain gather's 9.80 ms on 4096 x 2^19); longer spectra take
// the plain gather kernel.  Item numbers are 32-bit.
bool hs_interleaved_supported(const hs_plan *p)
{
    if (p->variant != HS_FREQBIN) return false;
    if (p->Hmax < 2 || p->nbins > ((int64_t)1 << 19)) return false;
    const il_sched s = make_sched(p, p->batch);
    return (int64_t)s.groups * (s.nT > s.nG ? s.nT : s.nG) < ((int64_t)1 << 30);   // (item codes: bit 30 marks a G item)
}

size_t hs_interleaved_workspace_bytes(const hs_plan *p, int64_t batch)
{
    const il_sched s = make_sched(p, batch);
    return ctrl_bytes(s.groups) + (size_t)s.R * (size_t)s.slot_words * sizeof(float) + 256;
}

int hs_interleaved_launches(const hs_plan *p, int64_t batch)
{
    (void)p;
    (void)batch;
    return 2;   // one memset node + one persistent kernel
}

int hs_interleaved_launch(const hs_plan *p, const hs_buffers &buf, int64_t batch, void *ws, cudaStream_t stream)
{
    if (!ws) HS_FAIL(HS_ERR_WORKSPACE);
    return by_level(p, buf, batch, ws, stream);
}
