// hs_internal.cuh — plan layout, error plumbing and the shared device-side epilogue (normalise, full planes,
// running max/argmax).  Product code: shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>
#ifdef HS_TUNING
#include <cstdlib>
#endif

#include "../../include/hs.h"

#define HS_MAX_LEVELS 6
#define HS_OUT_CAND 8   // internal OUT template bit: reduced output goes to the candidate sink (hs_execute_candidates)
#define HS_HOST_LANES 3

// Control block at the start of every workspace that a persistent kernel synchronises through (zeroed by a memset
// node before each launch): word 0 = work counter, word 1 = error flag (a bounded wait gave up, hs_plan_device_status),
// words 2.. = wait statistics of the kernel family.
#define HS_CTRL_QUEUE 0
#define HS_CTRL_ERROR 1
#define HS_CTRL_STATS 2
#define HS_SPIN_LIMIT_DEFAULT (1u << 23)

// Tuning knobs are compiled out of the product: only a -DHS_TUNING build (the builder's sweeps and the forced-timeout
// test, libhs_tuning.so) reads the environment.
inline int hs_knob(const char *name, int dflt)
{
#ifdef HS_TUNING
    const char *v = getenv(name);
    return v ? atoi(v) : dflt;
#else
    (void)name;
    return dflt;
#endif
}
inline unsigned hs_spin_limit() { return (unsigned)hs_knob("HS_SPIN_LIMIT", (int)HS_SPIN_LIMIT_DEFAULT); }

struct hs_plan {
    int64_t nbins, batch;
    int64_t nz;        // rows of the f - fdot plane per batch entry (1: the one-dimensional sum)
    int levels_mode;   // enum hs_levels
    int window;        // enum hs_window (eq. 2 only)
    int Hmax, L, variant, out_mode;
    int algo_req;  // what the caller asked for (enum hs_algo)
    int algo;      // resolved family, never AUTO
    int device;    // ordinal of the device the plan was created on (checked at execute)
    int sm_count;
    size_t smem_optin;  // max dynamic shared memory per block
    // control blocks (device) the last execute launched with, for hs_plan_device_status; written by hs_execute*
    mutable const void *last_ctrl[3];
    mutable int n_last_ctrl;
    // workspace for the resolved algorithm (device, caller-owned)
    void *ws;
    size_t ws_bytes;
    // host-buffer path (hs_execute_host)
    void *staging;
    size_t staging_bytes;
    int64_t slab;
    cudaStream_t lane_stream[HS_HOST_LANES];
    cudaEvent_t lane_done[HS_HOST_LANES];
    cudaEvent_t fork;
    bool lanes_ready;
};

// ---- error plumbing (hs_api.cu) ---------------------------------------------------------------------------------
void hs_set_error(int code);
#define HS_FAIL(code)          \
    do {                       \
        hs_set_error(code);    \
        return (code);         \
    } while (0)
#define HS_CUDA_OK(expr)                        \
    do {                                        \
        if ((expr) != cudaSuccess) {            \
            (void)cudaGetLastError();           \
            HS_FAIL(HS_ERR_CUDA);               \
        }                                       \
    } while (0)

// ---- launch entry points of the kernel families -------------------------------------------------------------------
// Each enqueues on `stream` for spectra [0, batch) of the given buffers and returns an hs_status.
// Candidate sink of hs_execute_candidates: when `cand` is set a kernel appends the bins whose reduced maximum exceeds
// `thr` instead of storing vmax / amax (which are then nullptr).  `b0` = batch index of the first spectrum of the launch.
struct hs_cand_sink {
    hs_candidate *cand;
    unsigned long long *count;
    long long cap;
    float thr;
    int b0;
};
struct hs_buffers {
    const float *x;  // the spectra, or (cplx) the complex Fourier series [..][2] they are formed from on the fly
    float *sums;
    float *vmax;
    uint8_t *amax;
    uint8_t *jdbg;  // Greedy debug paths or nullptr
    hs_cand_sink sink;
    bool cplx;      // hs_execute_complex: x holds (re, im) pairs, x(k) = hs_power(F_k, scale)
    float scale;
};
int hs_launch_direct(const hs_plan *p, const hs_buffers &buf, int64_t batch, void *ws, cudaStream_t stream);
int hs_launch_general(const hs_plan *p, const hs_buffers &buf, int64_t batch, void *ws, cudaStream_t stream);   // hs_general.cu
size_t hs_general_workspace_bytes(const hs_plan *p);
int hs_general_launches(const hs_plan *p);
int hs_launch_tiled(const hs_plan *p, const hs_buffers &buf, int64_t batch, void *ws, cudaStream_t stream);
size_t hs_tiled_workspace_bytes(const hs_plan *p, int64_t batch);
int hs_tiled_launches(const hs_plan *p, int64_t batch);
bool hs_tiled_supported(const hs_plan *p);
// per-variant tuned kernels
int hs_standard_tiled_launch(const hs_plan *p, const hs_buffers &buf, int64_t batch, cudaStream_t stream);
int hs_standard_tiled_launches(const hs_plan *p, int64_t batch);
int hs_standard_rb_launch(const hs_plan *p, const hs_buffers &buf, int64_t batch, void *ws, cudaStream_t stream);
size_t hs_standard_rb_workspace_bytes(const hs_plan *p);
bool hs_standard_rb_supported(const hs_plan *p);
int hs_twophase_launch(const hs_plan *p, const hs_buffers &buf, int64_t batch, void *ws, cudaStream_t stream);
int hs_twophase_launches(const hs_plan *p, int64_t batch);
size_t hs_twophase_workspace_bytes(const hs_plan *p, int64_t batch);
bool hs_twophase_supported(const hs_plan *p, int64_t batch);
int hs_greedy_gather_launch(const hs_plan *p, const hs_buffers &buf, int64_t batch, cudaStream_t stream);
int hs_greedy_gather_launches(const hs_plan *p, int64_t batch);
int hs_interleaved_launch(const hs_plan *p, const hs_buffers &buf, int64_t batch, void *ws, cudaStream_t stream);
int hs_interleaved_launches(const hs_plan *p, int64_t batch);
size_t hs_interleaved_workspace_bytes(const hs_plan *p, int64_t batch);
bool hs_interleaved_supported(const hs_plan *p);
int hs_grouped_launch(const hs_plan *p, const hs_buffers &buf, int64_t batch, void *ws, cudaStream_t stream);
int hs_grouped_launches(const hs_plan *p, int64_t batch);
size_t hs_grouped_workspace_bytes(const hs_plan *p, int64_t batch);
bool hs_grouped_supported(const hs_plan *p);
bool hs_tiled_has_ctrl(const hs_plan *p);
bool hs_tiled_supports_complex(const hs_plan *p);   // the resolved kernel starts its workspace with a control block

// ---- fused front end (hs_execute_complex) ----------------------------------------------------
// x(k) = (re^2 + im^2) * scale - 1, fp32, every operation rounded on its own (the _rn intrinsics are never contracted
// into a fused multiply-add): bit-identical to the definition the parity tests check against (separately rounded fp32 operations), so that the comparisons the
// harmonic sum takes on x (Greedy's drift, the best level) are the same on both sides.
__device__ __forceinline__ float hs_power(float re, float im, float scale)
{
    return __fsub_rn(__fmul_rn(__fadd_rn(__fmul_rn(re, re), __fmul_rn(im, im)), scale), 1.0f);
}
// element k of a spectrum whose storage starts at `row` (CPLX: `row` points at the spectrum's first (re, im) pair)
template <bool CPLX>
__device__ __forceinline__ float hs_ldx(const float *__restrict__ row, int k, float scale)
{
    if (CPLX) {
        const float2 f = __ldg(reinterpret_cast<const float2 *>(row) + k);
        return hs_power(f.x, f.y, scale);
    }
    return __ldg(row + k);
}
// elements k .. k + 3 (k % 4 == 0 and the row 16-byte aligned)
template <bool CPLX>
__device__ __forceinline__ float4 hs_ldx4(const float *__restrict__ row, int k, float scale)
{
    if (CPLX) {
        const float4 a = __ldg(reinterpret_cast<const float4 *>(row) + (k >> 1));
        const float4 b = __ldg(reinterpret_cast<const float4 *>(row) + (k >> 1) + 1);
        return make_float4(hs_power(a.x, a.y, scale), hs_power(a.z, a.w, scale), hs_power(b.x, b.y, scale), hs_power(b.z, b.w, scale));
    }
    return __ldg(reinterpret_cast<const float4 *>(row + k));
}

// ---- device-side epilogue ---------------------------------------------------------------------------------------
// c_H = fp32(1/sqrt(H)) for H = 1,2,4,8,16,32 (CONVENTIONS.md C7; "1/sqrt(H)").
__device__ __forceinline__ constexpr float hs_norm(int l)
{
    return l == 0 ? 1.0f
         : l == 1 ? 0.70710678118654752440f
         : l == 2 ? 0.5f
         : l == 3 ? 0.35355339059327376220f
         : l == 4 ? 0.25f
                  : 0.17677669529663688110f;
}

// hs_execute_candidates: append (b, n, m, a) if m > thr.  Bins above a sensible threshold are rare, so one atomic each.
__device__ __forceinline__ void hs_push(const hs_cand_sink &s, int64_t b, int n, float m, int a)
{
    if (m > s.thr) {
        const unsigned long long pos = atomicAdd(s.count, 1ULL);
        if (pos < (unsigned long long)s.cap) {
            int4 rec = make_int4((int)(b + s.b0), n, __float_as_int(m), a);
            *reinterpret_cast<int4 *>(s.cand + pos) = rec;
        }
    }
}

// Running reduced output of one bin: m = max_l h_l, a = smallest l attaining it (C8).
template <int OUT>
struct hs_emit {
    float m;
    int a;
    // running max over the levels; a level replaces the maximum only if strictly greater
    __device__ __forceinline__ void reduce(int l, float h)
    {
        if (l == 0) {
            m = h;
            a = 0;
        } else if (h > m) {
            m = h;
            a = l;
        }
    }
    // plane0 points at sums[b][0][n]; consecutive levels are `N` floats apart.
    __device__ __forceinline__ void level(int l, float S, float *__restrict__ plane0, int64_t N)
    {
        const float h = S * hs_norm(l);
        if (OUT & HS_OUT_FULL) plane0[(int64_t)l * N] = h;
        if (OUT & HS_OUT_REDUCED) reduce(l, h);
    }
};
