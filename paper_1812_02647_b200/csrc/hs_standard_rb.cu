// hs_standard_rb.cu — eq. 1 (CONVENTIONS.md C1) at Hmax = 32, reduced output, register blocked.
//
// The term of harmonic i = 1..32 at output n is x[(n i + 16) >> 5].  With n = 32 m + r the index is m i + c(r, i),
// c(r, i) = (r i + 16) >> 5 in [0, i]: a THREAD that owns the 32 consecutive outputs 32 m .. 32 m + 31 reads, for
// harmonic i, only the i + 1 words x[m i .. m i + i], and every one of its 1024 (r, i) terms has a compile-time register
// index.  That is 17.5 shared-memory words per output instead of the 32 of a lane-per-output mapping (hs_standard_tiled.cu),
// which is what bounds eq. 1: the path is limited by shared-memory bandwidth and L2 -> SM fill, not by HBM.
//
// A CTA of 128 threads takes tiles of 4096 consecutive outputs (lane = m) and streams the 32 harmonics through a ring
// of shared-memory slots in dyadic level order 32 | 16 | 8 24 | 4 12 20 28 | 2 6 .. 30 | 1 3 .. 31, so that one running
// sum per output serves all six levels (eq. 1 is cumulative over dyadic H).  The window of harmonic i for the tile is
// the contiguous range x[n0 i / 32 .. (n0 + 4096) i / 32]: 128 i + 1 words.
//   * i not a multiple of 8: one TMA bulk copy per window (cp.async.bulk, UBLKCP) onto the slot's mbarrier.  Lane stride
//     is i words: conflict-free 4-byte loads for odd i, 8-byte loads for i = 2 (mod 4), 16-byte loads for i = 4 (mod 8).
//   * i = 8, 16, 24, 32: a lane stride of i words would hit the same banks, so the window is copied by cp.async
//     (16 bytes per thread) into rows of i + 4 words: one pad unit per thread row makes the 16-byte loads conflict-free.
// The warp that finishes with a slot last refills it with the window three stages ahead (a counter per slot in shared
// memory, one mbarrier per slot for the arrival of the data: no CTA-wide barrier anywhere); the ring runs across tiles.
// The reduced outputs of a thread (32 consecutive floats = one 128-byte line) are stored straight from registers
// (a transposition through shared memory for fully coalesced stores measured the same time).
#include <utility>

#include "hs_internal.cuh"
#include "hs_ptx.cuh"

namespace {

constexpr int kT = 4096;                  // outputs per tile
constexpr int kNT = 128;                  // threads per CTA: one per 32 outputs
constexpr int kSlot = 5128;               // words per ring slot: the largest stage (padded windows of i = 8 and 24)
constexpr int kSlots = 3;
constexpr int kCtasPerSm = 3;
constexpr int kStages = 17;

// A stage brings the windows of one or two harmonics (about 4100 words, so the stages are evenly sized), in dyadic
// level order: 32 | 16 | 8 24 | 4 28, 12 20 | 2 30, 6 26, 10 22, 14 18 | 1 31, 3 29, .., 15 17
__host__ __device__ constexpr int stream_a(int s)
{
    return s == 0 ? 32 : s == 1 ? 16 : s == 2 ? 8 : s == 3 ? 4 : s == 4 ? 12 : s < 9 ? 2 + 4 * (s - 5) : 1 + 2 * (s - 9);
}
__host__ __device__ constexpr int stream_b(int s) { return s < 2 ? 0 : 32 - stream_a(s); }
// level completed by stage s, or -1
__host__ __device__ constexpr int level_after(int s)
{
    return s == 0 ? 0 : s == 1 ? 1 : s == 2 ? 2 : s == 4 ? 3 : s == 8 ? 4 : s == 16 ? 5 : -1;
}
__host__ __device__ constexpr bool is_padded(int i) { return (i & 7) == 0; }
__host__ __device__ constexpr int cidx(int r, int i) { return (r * i + 16) >> 5; }
// words the window of harmonic i occupies in a slot (padded rows of i + 4 words, or 128 i + 1 words rounded up to 16 bytes)
__host__ __device__ constexpr int slot_words(int i) { return is_padded(i) ? 128 * (i + 4) + (i <= 16 ? 4 : 0) : 128 * i + 4; }

struct rb_params {
    const float *x;
    float *vmax;
    uint8_t *amax;
    int *counter;    // tile queue (zeroed before the launch)
    hs_cand_sink sink;
    int N;
    int tiles_per_spectrum;
    int tiles;       // total (< 2^31: checked on the host)
    int Z;           // rows of an f-fdot plane (hs_plan_create_2d): a "spectrum" is then one plane row zi, and harmonic i of
                     // drift z = zi - (Z-1)/2 reads row floor((z i + 16)/32) of the same plane; 1 = the one-dimensional sum
};

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

// S[r] (+)= x[m i + c(r, i)] for the thread's 32 outputs, window of harmonic I staged in `slot` (lane = tile-local m)
template <int I>
__device__ __forceinline__ void accumulate(const float *__restrict__ slot, int mloc, float (&S)[32])
{
    float w[I + 4];
    if constexpr (is_padded(I)) {
        const float *__restrict__ row = slot + mloc * (I + 4);
#pragma unroll
        for (int q = 0; q < I / 4; q++) {
            const float4 u = *reinterpret_cast<const float4 *>(row + 4 * q);
            w[4 * q] = u.x, w[4 * q + 1] = u.y, w[4 * q + 2] = u.z, w[4 * q + 3] = u.w;
        }
        if constexpr (I <= 16) w[I] = row[I + 4];               // first word of the next thread's row
    } else if constexpr (I % 4 == 0) {
        const float *__restrict__ row = slot + mloc * I;
#pragma unroll
        for (int q = 0; q <= I / 4; q++) {
            const float4 u = *reinterpret_cast<const float4 *>(row + 4 * q);
            w[4 * q] = u.x, w[4 * q + 1] = u.y, w[4 * q + 2] = u.z, w[4 * q + 3] = u.w;
        }
    } else if constexpr (I % 2 == 0) {
        const float *__restrict__ row = slot + mloc * I;
#pragma unroll
        for (int q = 0; q <= I / 2; q++) {
            const float2 u = *reinterpret_cast<const float2 *>(row + 2 * q);
            w[2 * q] = u.x, w[2 * q + 1] = u.y;
        }
    } else {
        const float *__restrict__ row = slot + mloc * I;
#pragma unroll
        for (int k = 0; k <= I; k++) w[k] = row[k];
    }
#pragma unroll
    for (int r = 0; r < 32; r += 2) {
        if constexpr (I == 32) {                                 // first harmonic of a tile: starts the running sums
            S[r] = w[cidx(r, I)];
            S[r + 1] = w[cidx(r + 1, I)];
        } else {
            asm("{\n\t.reg .b64 a, b, d;\n\tmov.b64 a, {%0, %1};\n\tmov.b64 b, {%2, %3};\n\tadd.rn.f32x2 d, a, b;\n\tmov.b64 {%0, %1}, d;\n\t}"
                : "+f"(S[r]), "+f"(S[r + 1])
                : "f"(w[cidx(r, I)]), "f"(w[cidx(r + 1, I)]));
        }
    }
}

// level l complete: h = S c_l, running maximum and best level (C8: a later level wins only if strictly greater)
template <int LV>
__device__ __forceinline__ void emit_level(const float (&S)[32], float (&m)[32], int (&a)[32])
{
#pragma unroll
    for (int r = 0; r < 32; r += 2) {
        // two outputs per multiply: mul.f32x2 (FMUL2) is the same IEEE fp32 product in each half
        float h0, h1;
        if (LV == 0) {
            h0 = S[r], h1 = S[r + 1];
        } else {
            asm("{\n\t.reg .b64 a, c, d;\n\tmov.b64 a, {%2, %3};\n\tmov.b64 c, {%4, %4};\n\tmul.rn.f32x2 d, a, c;\n\tmov.b64 {%0, %1}, d;\n\t}"
                : "=f"(h0), "=f"(h1)
                : "f"(S[r]), "f"(S[r + 1]), "f"(hs_norm(LV)));
        }
        if (LV == 0) {
            m[r] = h0, m[r + 1] = h1;
            a[r] = 0, a[r + 1] = 0;
        } else {
            if (h0 > m[r]) {
                m[r] = h0;
                a[r] = LV;
            }
            if (h1 > m[r + 1]) {
                m[r + 1] = h1;
                a[r + 1] = LV;
            }
        }
    }
}

template <class F, int... s>
__device__ __forceinline__ void for_each_stage(F &f, std::integer_sequence<int, s...>)
{
    (f(std::integral_constant<int, s>{}), ...);
}

// PLANE: the two-dimensional sum (p.Z > 1); a compile-time switch so that the one-dimensional kernel carries none of the
// row arithmetic (it cost 11 % there when it was a run-time test).
template <bool CAND, bool PLANE>
__global__ void __launch_bounds__(kNT, kCtasPerSm)
rb_kernel(const __grid_constant__ rb_params p)
{
    extern __shared__ __align__(128) float smem[];
    __shared__ __align__(8) uint64_t full[kSlots];
    float *ring = smem;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int N = p.N;

    if (threadIdx.x == 0) {
#pragma unroll
        for (int s = 0; s < kSlots; s++) hsptx::mbar_init(&full[s], 1);
        hsptx::mbar_fence_init();
    }
    __syncthreads();

    // Tiles are handed out in order from one global counter: the CTAs in flight always work on ~gridDim.x consecutive
    // tiles, so the windows a tile shares with its neighbours (the low harmonics of tile t lie where tile t i / 32 read
    // its own bins) are still in L2.  A static stride lets the CTAs drift apart by many rounds and re-reads x from HBM
    // (ncu: 1.5x the algorithmic reads at 2^18 bins, 3.5x at 2^20).  The first tile is blockIdx.x; a CTA asks for its
    // next tile at the start of the current one (the ring prefetches across tiles).
    const int tps = p.tiles_per_spectrum;
    __shared__ int s_next[2];
    int cur = (int)blockIdx.x;
    int cb = (int)((unsigned)cur / (unsigned)tps), ct = (int)((unsigned)cur % (unsigned)tps);

    // start the copies of stage SC of tile (spectrum ib, tile it) into slot `islot` (the stage is a compile-time
    // constant: the stage that issues it is known); every thread commits one cp.async group per stage
    auto issue = [&](auto sc, int ib, int it, int islot, bool live) {
        constexpr int SC = decltype(sc)::value, IA = stream_a(SC), IB = stream_b(SC);
        if (live) {
            float *dst = ring + islot * kSlot;
            // the row harmonic IA (and IB) of "spectrum" ib is read from: ib itself, or in the 2-D sum the plane row at
            // drift floor((z i + 16) / 32) (arithmetic shift: floor toward minus infinity)
            auto src_row = [&](int i) -> int64_t {
                if constexpr (!PLANE) return ib;
                const int Zc = (p.Z - 1) >> 1, pl = ib / p.Z, z = ib - pl * p.Z - Zc;
                return (int64_t)pl * p.Z + ((z * i + 16) >> 5) + Zc;
            };
            const float *xb = p.x + (src_row(IA) * N + (int64_t)it * (kT / 32 * IA));        // x[n0 IA / 32]: 16-byte aligned
            const float *xb2 = PLANE ? p.x + (src_row(IB == 0 ? IA : IB) * N + (int64_t)it * (kT / 32 * (IB == 0 ? IA : IB)))
                                     : xb + (int64_t)it * (kT / 32 * (IB - IA));
            if constexpr (is_padded(IA)) {
                auto copy_padded = [&](auto ic, float *d, const float *src) {
                    constexpr int I = decltype(ic)::value, units = 32 * I + (I <= 16 ? 1 : 0), rowu = I / 4;
#pragma unroll
                    for (int u0 = 0; u0 < units; u0 += kNT) {
                        const int u = u0 + threadIdx.x;
                        if (u0 + kNT <= units || u < units) cp_async16(d + 4 * (u + u / rowu), src + 4 * u);
                    }
                };
                copy_padded(std::integral_constant<int, IA>{}, dst, xb);
                if constexpr (IB != 0)
                    copy_padded(std::integral_constant<int, IB == 0 ? 8 : IB>{}, dst + slot_words(IA), xb2);
            } else if (threadIdx.x == 0) {
                constexpr uint32_t bytesA = (uint32_t)slot_words(IA) * 4u, bytesB = (uint32_t)slot_words(IB) * 4u;
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");  // the slot was last read by ordinary loads
                hsptx::mbar_arrive_expect_tx(&full[islot], bytesA + bytesB);
                hsptx::bulk_g2s(dst, xb, bytesA, &full[islot]);
                hsptx::bulk_g2s(dst + slot_words(IA), xb2, bytesB, &full[islot]);
            }
        }
        cp_async_commit();
    };

    issue(std::integral_constant<int, 0>{}, cb, ct, 0, cur < p.tiles);
    issue(std::integral_constant<int, 1>{}, cb, ct, 1, cur < p.tiles);
    issue(std::integral_constant<int, 2>{}, cb, ct, 2, cur < p.tiles);
    if constexpr (kSlots > 3) issue(std::integral_constant<int, 3>{}, cb, ct, 3, cur < p.tiles);

    uint32_t phase = 0u;                                                  // bit s: parity of the next wait on full[s]
    float S[32], m[32];
    int a[32];
    int slot = 0;
    for (int k = 0; cur < p.tiles; k++) {
        const int64_t b = cb;
        const int n0 = ct * kT;
        if (threadIdx.x == 0) s_next[k & 1] = (int)gridDim.x + atomicAdd(p.counter, 1);
        int nxt = 0, nb = 0, nt = 0;                                      // the CTA's next tile: known from stage 1 on
        bool more = false;
        auto stage = [&](auto sc) {
            constexpr int s = decltype(sc)::value, IA = stream_a(s), IB = stream_b(s), LV = level_after(s);
            if constexpr (is_padded(IA)) {
                cp_async_wait<kSlots - 1>();
                __syncthreads();
            } else {
                hsptx::mbar_wait(&full[slot], (phase >> slot) & 1u);
                phase ^= 1u << slot;
            }
            if constexpr (s == 1) {                                       // (a CTA barrier separates this from the write)
                nxt = s_next[k & 1];
                more = nxt < p.tiles;
                nb = (int)((unsigned)nxt / (unsigned)tps);
                nt = (int)((unsigned)nxt % (unsigned)tps);
            }
            accumulate<IA>(ring + slot * kSlot, threadIdx.x, S);
            if constexpr (IB != 0) accumulate<IB == 0 ? 1 : IB>(ring + slot * kSlot + slot_words(IA), threadIdx.x, S);
            if constexpr (LV >= 0) emit_level<LV>(S, m, a);
            __syncthreads();                                              // the slot is free: refill it with stage s + 3
            constexpr int s3 = (s + kSlots) % kStages;
            if constexpr (s + kSlots < kStages) issue(std::integral_constant<int, s3>{}, cb, ct, slot, true);
            else issue(std::integral_constant<int, s3>{}, nb, nt, slot, more);
            slot = slot == kSlots - 1 ? 0 : slot + 1;
        };
        for_each_stage(stage, std::make_integer_sequence<int, kStages>{});
        cur = nxt;
        cb = nb;
        ct = nt;

        // ---- outputs of the tile: thread holds bins nw0 + 32 lane + [0, 32)
        const int64_t base = b * N + n0 + warp * 1024;
        if constexpr (CAND) {   // hs_execute_candidates: no stores, rare appends
            float mm = m[0];
#pragma unroll
            for (int r = 1; r < 32; r++) mm = fmaxf(mm, m[r]);
            if (mm > p.sink.thr) {
#pragma unroll
                for (int r = 0; r < 32; r++) hs_push(p.sink, b, n0 + warp * 1024 + 32 * lane + r, m[r], a[r]);
            }
            continue;
        }
        {
            float *pv = p.vmax + base + 32 * lane;
#pragma unroll
            for (int q = 0; q < 8; q++)
                hsptx::st_cs(reinterpret_cast<float4 *>(pv + 4 * q), make_float4(m[4 * q], m[4 * q + 1], m[4 * q + 2], m[4 * q + 3]));
#pragma unroll
            for (int h = 0; h < 2; h++) {
                uint32_t pk[4];
#pragma unroll
                for (int q = 0; q < 4; q++)
                    pk[q] = (uint32_t)a[16 * h + 4 * q] | ((uint32_t)a[16 * h + 4 * q + 1] << 8) |
                            ((uint32_t)a[16 * h + 4 * q + 2] << 16) | ((uint32_t)a[16 * h + 4 * q + 3] << 24);
                asm volatile("st.global.cs.v4.u32 [%0], {%1,%2,%3,%4};" ::"l"(p.amax + base + 32 * lane + 16 * h), "r"(pk[0]),
                             "r"(pk[1]), "r"(pk[2]), "r"(pk[3])
                             : "memory");
            }
        }
    }
    asm volatile("cp.async.wait_all;" ::: "memory");
}

}  // namespace

// Hmax = 32, reduced output only, spectra made of whole 4096-bin tiles; everything else takes hs_standard_tiled.cu
// (or, for the 2-D sum, hs_general.cu).
bool hs_standard_rb_supported(const hs_plan *p)
{
    return p->variant == HS_STANDARD && p->Hmax == 32 && p->out_mode == HS_OUT_REDUCED && p->nbins % kT == 0 &&
           p->levels_mode == HS_LEVELS_DYADIC && p->batch * p->nz * (p->nbins / kT) < ((int64_t)1 << 30);
}

size_t hs_standard_rb_workspace_bytes(const hs_plan *) { return 512; }   // the tile counter (one 256-byte line, padded)

int hs_standard_rb_launch(const hs_plan *p, const hs_buffers &buf, int64_t batch, void *ws, cudaStream_t stream)
{
    if (!ws) HS_FAIL(HS_ERR_WORKSPACE);
    rb_params prm{};
    prm.x = buf.x;
    prm.vmax = buf.vmax;
    prm.amax = buf.amax;
    prm.N = (int)p->nbins;
    prm.tiles_per_spectrum = (int)(p->nbins / kT);
    prm.tiles = (int)(batch * p->nz * prm.tiles_per_spectrum);
    prm.Z = (int)p->nz;
    prm.counter = static_cast<int *>(ws);
    prm.sink = buf.sink;
    const size_t smem = (size_t)(kSlots * kSlot) * sizeof(float);
    // (function attributes are per device: set on every launch rather than once per process)
    const bool plane = p->nz > 1;
    auto kern = buf.sink.cand ? (plane ? rb_kernel<true, true> : rb_kernel<true, false>)
                              : (plane ? rb_kernel<false, true> : rb_kernel<false, false>);
    HS_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const int64_t slots = (int64_t)p->sm_count * kCtasPerSm;
    const unsigned grid = (unsigned)(prm.tiles < slots ? prm.tiles : slots);
    HS_CUDA_OK(cudaMemsetAsync(ws, 0, 256, stream));
    kern<<<grid, kNT, smem, stream>>>(prm);
    HS_CUDA_OK(cudaGetLastError());
    return HS_OK;
}
