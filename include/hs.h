/*
 * hs.h — C ABI of the batched incoherent harmonic sum for NVIDIA B200 (sm_100a).
 *
 * What is computed: for every spectrum b of a batch and every bin n, the partial harmonic sums
 * h_H(n), H = 1,2,4,..,Hmax, of arXiv 1812.02647 (Adamek & Armour) in one of the paper's four variants
 *     HS_STANDARD  eq. 1, PAPER.md:17      h_H(n) = H^-1/2 sum_{i=1..H} x(floor((n i + H/2)/H))
 *     HS_MAX       eq. 2, PAPER.md:33      h_H(n) = H^-1/2 sum_{i=1..H} max_{0<=j<=i-1} x~(i n + j)
 *     HS_FREQBIN   eq. 3, PAPER.md:38      h_H(n) = H^-1/2 sum_{i=1..H} x~(i n)
 *     HS_GREEDY    eq. 4, PAPER.md:43-46   S_1 = x(n), j = 0; for i = 2..Hmax: l = x~(i n + j), r = x~(i n + j + 1),
 *                                          S_i = S_{i-1} + max(l, r), j += (r > l);  h_H = H^-1/2 S_H
 * with x~(k) = x(k) inside [0, nbins) and 0 outside.  The exact readings (rounding, window, tie and padding
 * rules) are frozen in CONVENTIONS.md (C1..C11); the call names and argument order are fixed by
 * BASELINE.json north_star.  The batch is data-parallel: spectra are independent.
 *
 * Layouts (row-major, all device pointers unless the name says host):
 *     x       [batch][nbins]          float32   input, read-only, must not alias an output
 *     sums    [batch][L][nbins]       float32   full output, plane l holds h_{2^l}; L = log2(Hmax)+1
 *     max     [batch][nbins]          float32   reduced output: max over the L levels
 *     argmax  [batch][nbins]          uint8     reduced output: smallest level index l in [0, L-1] attaining it
 * Arithmetic: fp32 loads, fp32 accumulation, h = S * fp32(1/sqrt(H)); comparisons on raw fp32 values.
 * Inputs must be finite (NaN/Inf: unspecified result, no fault).
 *
 * Ownership: the caller owns every buffer, including the workspace.  A plan owns host metadata only (and, once
 * hs_plan_set_host_staging is called, three CUDA streams and their events).  No function allocates device memory.
 * Errors: functions returning int return HS_OK (0) or an hs_status code; hs_plan_create returns NULL and records the
 * code, readable with hs_last_error() (thread-local).  Nothing is printed, thrown or aborted across this ABI.
 * There is no CPU fallback: without an sm_100 device hs_plan_create fails with HS_ERR_UNSUPPORTED.
 */
#ifndef HS_H
#define HS_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct hs_plan hs_plan; /* opaque */

enum hs_variant { HS_STANDARD = 0, HS_MAX = 1, HS_FREQBIN = 2, HS_GREEDY = 3 };
enum hs_out_mode { HS_OUT_FULL = 1, HS_OUT_REDUCED = 2, HS_OUT_BOTH = 3 };
enum hs_status {
    HS_OK = 0,
    HS_ERR_INVALID_ARG = 1,  /* a size, Hmax, variant, out_mode or option out of range                  */
    HS_ERR_NULL_POINTER = 2, /* a required pointer is NULL                                              */
    HS_ERR_MISALIGNED = 3,   /* a base pointer is not 16-byte aligned                                   */
    HS_ERR_UNSUPPORTED = 4,  /* no CUDA device of compute capability 10.x is current                    */
    HS_ERR_WORKSPACE = 5,    /* the chosen algorithm needs a workspace that was not set or is too small */
    HS_ERR_CUDA = 6,         /* a CUDA runtime call or kernel launch failed                             */
    HS_ERR_DEVICE_TIMEOUT = 7, /* hs_plan_device_status: a kernel of the last execute gave up waiting for another
                                 thread block (its outputs are then not valid)                          */
    HS_ERR_SCRATCH_LIMIT = 8  /* hs_execute_static: one spectrum's per-harmonic arrays do not fit the library's
                                 built-in scratch array (HS_STATIC_SCRATCH_BYTES)                       */
};
/* Kernel family.  HS_ALGO_AUTO picks the fastest one that is valid for the plan. */
enum hs_algo {
    HS_ALGO_AUTO = 0,
    HS_ALGO_DIRECT = 1, /* one thread per output bin, loads straight from global memory; needs no workspace;
                           every variant; kept as the simple on-device reference                              */
    HS_ALGO_TILED = 2,  /* the tuned kernels: eq. 1 register-blocked with TMA-streamed windows
                           (workspace: a tile counter); eq. 2 grouped two-phase through L2-resident workspace slots;
                           eq. 3 gather from a spectrum-interleaved copy of 16 spectra at a time (workspace ring);
                           eq. 4, and eqs. 2-3 where those do not apply, the range-skipping gather                    */
    HS_ALGO_TWOPHASE = 3, /* eqs. 2-3 only: the two-phase kernel (for eq. 2 the same as HS_ALGO_TILED)              */
    HS_ALGO_GATHER = 4,   /* eqs. 3-4 only: the range-skipping gather straight from x (no workspace); what
                             HS_ALGO_TILED itself uses for spectra too long for the interleaved group copy           */
    HS_ALGO_GROUPED = 5,  /* eqs. 2-3 only, Hmax >= 2, nbins <= 2^23: two phases per spectrum by a static group of co-resident CTAs, the
                             per-harmonic arrays of a spectrum live in one L2-resident workspace slot per group
                             (cooperative launch)                                                                   */
    HS_ALGO_GENERAL = 6   /* what plans of hs_plan_create_ex (every integer H, printed window) and hs_plan_create_2d
                             resolve to: one thread per output, no workspace; not selectable for other plans        */
};
/* hs_plan_create_ex options */
enum hs_levels {
    HS_LEVELS_DYADIC = 0, /* H = 1, 2, 4, .., Hmax (BASELINE.json north_star)                                        */
    HS_LEVELS_ALL = 1     /* every integer H = 1 .. Hmax, Hmax <= 64 ("an increasing number of harmonics") */
};
enum hs_window {
    HS_WINDOW_C2 = 0,     /* eq. 2 window j = 0 .. i-1 (CONVENTIONS.md C2: h_1(n) = x(n))                             */
    HS_WINDOW_PRINTED = 1, /* eq. 2 window exactly as printed, j = 1 .. i: h_1(n) = x(n + 1)            */
    HS_TERM_INTERP = 2     /* eq. 1 only: the term x(n i / H) of PAPER.md:17 read on the straight line between the two
                              neighbouring bins instead of at the nearest bin (CONVENTIONS.md C15; PAPER.md:52 is about
                              the power lost between bins): with n i = q H + r, ((H - r) x(q) + r x(q + 1)) / H          */
};

/*
 * hs_plan_create — describe one problem shape (the paper's statement of the problem: a batch of independent
 * spectra; partial sums for an increasing number of harmonics; one algorithm of
 * PAPER.md:17-46).
 *   nbins    bins per spectrum, 4 <= nbins <= 2^25 and nbins % 4 == 0 (16-byte rows for vector/bulk copies; bin indices
 *            up to 32*nbins+32 are int32)
 *   batch    number of spectra, 1 <= batch <= 2^31 - 1 (spectrum indices, also hs_candidate.spectrum, are int32),
 *            batch*nbins <= 2^40
 *   Hmax     largest number of harmonics, one of 1,2,4,8,16,32
 *   variant  enum hs_variant;  out_mode  enum hs_out_mode
 * Does no device work.  The plan belongs to the CUDA device that is current at the call: executing it with another
 * device current fails with HS_ERR_INVALID_ARG.
 * Returns NULL on error: HS_ERR_INVALID_ARG (checked first), HS_ERR_UNSUPPORTED, HS_ERR_CUDA.
 */
hs_plan *hs_plan_create(int64_t nbins, int64_t batch, int Hmax, int variant, int out_mode);

/*
 * hs_plan_create_ex — the variants of the paper's own description beyond the dyadic default:
 *   levels   HS_LEVELS_ALL: partial sums for EVERY integer H = 1..Hmax, 1 <= Hmax <= 64.  Level index l = H - 1, so
 *            sums is [batch][Hmax][nbins], argmax holds H - 1, hs_plan_levels returns Hmax.  eq. 1 uses the nearest
 *            bin, half up, for any H: x(floor((2 n i + H) / (2 H))) (= CONVENTIONS.md C1 for even H); h_H = S_H / sqrt(H).
 *            nbins <= 2^24.  HS_LEVELS_DYADIC with HS_WINDOW_C2 is exactly hs_plan_create.
 *   window   HS_WINDOW_PRINTED (HS_MAX only, else HS_ERR_INVALID_ARG): eq. 2 with 1 <= j <= i as the paper prints it.
 *            HS_TERM_INTERP (HS_STANDARD only, else HS_ERR_INVALID_ARG): eq. 1 with linearly interpolated terms, with
 *            either choice of levels; fp32: w = fp32(r) * fp32(1/H), term = fma(w, x(q+1) - x(q), x(q)).
 * Such plans resolve to HS_ALGO_GENERAL (no workspace); hs_plan_set_algo accepts only HS_ALGO_AUTO for them.
 */
hs_plan *hs_plan_create_ex(int64_t nbins, int64_t batch, int Hmax, int variant, int out_mode, int levels, int window);

/*
 * hs_plan_create_2d — the two-dimensional harmonic sum over the f - fdot plane of a Fourier-domain acceleration search
 * (reading R-2D of DESIGN.md section 16: the paper gives no equation).
 * One batch entry is a plane x[nz][nbins] (row-major); row zi holds drift z = zi - (nz-1)/2, nz odd, 1 <= nz <= 4095.
 * Harmonic i of a signal at (bin n, drift z) sits at (n i/H, z i/H):
 *     HS_STANDARD  S_H(n, z) = sum_{i=1..H} x(floor((z i + H/2)/H), floor((n i + H/2)/H))     (floor toward -infinity)
 *     HS_FREQBIN   S_H(n, z) = sum_{i=1..H} x~(i z, i n)                                       (0 outside the plane)
 * (other variants: HS_ERR_INVALID_ARG), dyadic levels, h_H = S_H / sqrt(H).  Layouts: x [batch][nz][nbins],
 * sums [batch][L][nz][nbins], max / argmax [batch][nz][nbins].  Execute with hs_execute / hs_execute_host.
 */
hs_plan *hs_plan_create_2d(int64_t nbins, int64_t nz, int64_t batch, int Hmax, int variant, int out_mode);

/*
 * hs_execute — enqueue the transform on `stream` (a cudaStream_t; NULL = the legacy default stream) and return
 * without synchronising.  d_x, d_sums, d_max, d_argmax are DEVICE pointers in the layouts above.
 * d_sums may be NULL iff out_mode lacks HS_OUT_FULL; d_max and d_argmax may be NULL iff it lacks HS_OUT_REDUCED;
 * otherwise NULL -> HS_ERR_NULL_POINTER.  Base pointers must be 16-byte aligned -> HS_ERR_MISALIGNED.
 * Every element of every requested output is overwritten.  A plan whose algorithm needs a workspace
 * (hs_plan_workspace_bytes > 0) must have one set -> HS_ERR_WORKSPACE; such a plan must not be executed
 * concurrently with itself.  Launch failure -> HS_ERR_CUDA.
 */
int hs_execute(const hs_plan *plan, const float *d_x, float *d_sums, float *d_max, uint8_t *d_argmax,
               void *stream);

/*
 * hs_execute_complex — the path with the step BEFORE it in the pipeline fused in (the series are "transformed
 * using an FFT into frequency space.  Then the harmonic sum is applied"): instead of a normalised
 * power spectrum the input is the complex Fourier series itself, d_F [batch][nbins][2] float32 (re, im interleaved, DEVICE,
 * 16-byte aligned, read-only), and every kernel forms
 *     x(k) = (re_k^2 + im_k^2) * scale - 1          fp32, each operation rounded separately (no fused multiply-add)
 * while it reads, so that x is never written to (or re-read from) HBM.  Outputs, NULL rules, workspace rule and
 * asynchrony as hs_execute; results are those of hs_execute on that x (bit for bit in h_1 = x).
 * Kernels: the gathers (eqs. 3-4), the interleaved ring's copy items (eq. 3), eq. 2's grouped kernel (phase A forms x while
 * filling shared memory) and the direct family; plans whose tuned kernel stages x with the TMA copy engine (eq. 1; eq. 2 on
 * spectra too long for the grouped kernel) run the direct family here.  Plans of hs_plan_create_ex with non-default
 * options and of hs_plan_create_2d: HS_ERR_INVALID_ARG.
 */
int hs_execute_complex(const hs_plan *plan, const float *d_F, float scale, float *d_sums, float *d_max,
                       uint8_t *d_argmax, void *stream);

/* hs_destroy — free the plan (host memory, and the staging streams if any).  NULL is a no-op returning HS_OK. */
int hs_destroy(hs_plan *plan);

/* ---- helpers ------------------------------------------------------------------------------------------------ */

int hs_last_error(void);                 /* code of the last failed call on this thread (HS_OK if none)          */
const char *hs_error_string(int code);   /* static string, never NULL                                            */
const char *hs_version(void);            /* static string                                                        */

int hs_plan_levels(const hs_plan *plan);                 /* L = log2(Hmax)+1 (HS_LEVELS_ALL plans: Hmax); -1 if NULL */
int hs_plan_set_algo(hs_plan *plan, int algo);           /* enum hs_algo; resets the workspace requirement       */
int hs_plan_algo(const hs_plan *plan);                   /* the resolved family (never HS_ALGO_AUTO), -1 if NULL */
size_t hs_plan_workspace_bytes(const hs_plan *plan);     /* device scratch the resolved algorithm needs (0 = none) */
/* d_ws: DEVICE pointer, 256-byte aligned, at least hs_plan_workspace_bytes(plan) bytes, owned by the caller and
 * kept alive while the plan is executed.  Contents need no initialisation and are undefined afterwards. */
int hs_plan_set_workspace(hs_plan *plan, void *d_ws, size_t bytes);
/* Number of kernel launches (memset nodes included) one hs_execute of this plan enqueues; -1 if plan is NULL. */
int hs_plan_launches(const hs_plan *plan);
/*
 * hs_plan_device_status — SYNCHRONISES `stream`, then reads back the error word of the control block(s) the plan's last
 * hs_execute / hs_execute_candidates / hs_execute_host launched with.  The persistent kernels (HS_ALGO_TILED for eqs. 2-4,
 * HS_ALGO_GROUPED) hand work between thread blocks through counters in the workspace; a thread block that polls such a
 * counter more than a bounded number of times (a scheduling bug, or a debugger / time-slicing stall of seconds) sets
 * the error word and carries on, so that the GPU cannot hang: the outputs of that execute are then NOT valid.
 * Returns HS_OK, HS_ERR_DEVICE_TIMEOUT, or HS_ERR_CUDA if the synchronisation / copy failed.  Plans whose kernels do
 * not synchronise between thread blocks always return HS_OK (after synchronising).  Call it before trusting outputs
 * in tests and benchmarks; hs_execute itself never synchronises.
 */
int hs_plan_device_status(const hs_plan *plan, void *stream);

/*
 * hs_execute_host — the same transform with HOST buffers (pinned memory recommended): h_x, h_sums, h_max, h_argmax
 * are HOST pointers in the layouts above (NULL rules as hs_execute).  The batch is cut into slabs of spectra; each
 * slab is copied to the device, transformed and copied back on one of three internal streams so that host->device
 * copies, kernels and device->host copies overlap.  Work is ordered after what `stream` holds at the call and
 * `stream` waits for it; the call itself does not synchronise.  Requires hs_plan_set_host_staging first.
 */
int hs_execute_host(hs_plan *plan, const float *h_x, float *h_sums, float *h_max, uint8_t *h_argmax,
                    void *stream);
/* Device bytes of staging hs_execute_host needs for slabs of `slab_spectra` spectra (3 slabs in flight, plus the
 * algorithm's workspace per slab).  0 on error. */
size_t hs_plan_host_staging_bytes(const hs_plan *plan, int64_t slab_spectra);
/* d_staging: DEVICE pointer, 256-byte aligned, owned by the caller.  Creates the plan's streams and events. */
int hs_plan_set_host_staging(hs_plan *plan, void *d_staging, size_t bytes, int64_t slab_spectra);

/*
 * hs_execute_candidates — the path with the step that follows it in the pipeline fused in (the harmonic
 * sum feeds SNR detection / candidate selection): instead of writing the reduced pair for every bin (5 bytes/bin), emit
 * only the bins whose maximum over the levels exceeds `threshold`:
 *     for every spectrum b and bin n with m(b, n) = max_l h_{2^l}(b, n) > threshold (strictly):
 *         append { b, n, m(b, n), a(b, n) }          (m and a exactly as d_max / d_argmax of hs_execute, CONVENTIONS.md C8)
 * The plan must have out_mode HS_OUT_REDUCED (else HS_ERR_INVALID_ARG); workspace rules as hs_execute.
 *   d_cand     DEVICE, 16-byte aligned, room for `capacity` records; the ORDER of the records is unspecified
 *   d_count    DEVICE, 8-byte aligned; zeroed by the call on `stream`, afterwards the number of bins above the threshold.
 *              If it exceeds `capacity` only `capacity` records were kept (which ones is unspecified).
 * Asynchronous on `stream` like hs_execute.  A low threshold makes the appends (one atomic each) the bottleneck.
 */
typedef struct hs_candidate {
    int32_t spectrum; /* b */
    int32_t bin;      /* n */
    float value;      /* m(b, n) */
    int32_t level;    /* a(b, n): level index of the best level, smallest on ties: l = log2 H (HS_LEVELS_ALL plans: H - 1) */
} hs_candidate;
int hs_execute_candidates(const hs_plan *plan, const float *d_x, float threshold, hs_candidate *d_cand,
                          int64_t capacity, unsigned long long *d_count, void *stream);

/*
 * hs_execute_static — eqs. 2 and 3 for callers that have no way to get device scratch memory.
 *
 * Every other execute call of this library leaves allocation to the caller: a kernel family that needs scratch wants
 * a workspace from hs_plan_set_workspace.  Some callers cannot provide one.  A real-time search back end typically
 * reserves all of its device memory when the observation starts and bans cudaMalloc / cudaFree inside the observing
 * loop (both synchronise the whole device, and an allocation can still fail hours into a run); a plug-in that a host
 * application hands input and output buffers to owns no allocator at all; and a process whose framework has claimed
 * the device's memory up front gets an out-of-memory error from a raw cudaMalloc.  For those callers this entry
 * point runs the two-phase kernels (the HS_ALGO_TWOPHASE family: phase 1 writes the per-harmonic arrays A_i of a
 * group of spectra, phase 2 sums them) with the arrays kept in a fixed array that is part of the library image:
 * HS_STATIC_SCRATCH_BYTES (32 MiB) of device memory, held by every GPU on which the library's code is loaded, from
 * then until the process exits.  The call allocates nothing: no cudaMalloc, no cudaFree, no library routine that does.
 *
 *   plan     from hs_plan_create with variant HS_MAX or HS_FREQBIN (anything else, and plans of hs_plan_create_ex
 *            with non-default options or of hs_plan_create_2d: HS_ERR_INVALID_ARG).  Any Hmax, any out_mode, any
 *            batch: the batch is processed in groups of as many spectra as fit the array.  The plan's own algorithm
 *            choice and workspace are ignored.
 *   limit    one spectrum's arrays (about 3.06 * nbins floats at Hmax = 32, 1.08 * nbins at Hmax = 4) must fit:
 *            about 2.7 million bins at Hmax = 32 (2^21 fits, 2^22 does not).  Longer spectra fail with HS_ERR_SCRATCH_LIMIT before anything is
 *            enqueued; hs_static_scratch_bytes() returns the size of the array.
 *   buffers  d_x, d_sums, d_max, d_argmax: DEVICE pointers owned by the caller, layouts, NULL and alignment rules and
 *            asynchrony exactly as hs_execute; the outputs are those of hs_execute on a HS_ALGO_TWOPHASE plan.
 *
 * First call on a device: the library looks up the device address of its array (once per device, with that device
 * current) before it launches.  Make that first call outside any stream capture.
 * Sharing: there is ONE array per device, shared by every plan, thread and stream, and it keeps whatever the previous
 * call left in it.  Nothing in it has to start at zero (phase 1 writes every word that phase 2 reads, before it reads
 * it), so a call never sees another call's data as long as calls do not overlap on the GPU; two calls that can run at
 * the same time (different streams with no dependency between them) race on the array and both produce garbage.
 * Order them with events, or use hs_execute with one caller-owned workspace per plan.
 */
#define HS_STATIC_SCRATCH_BYTES (32u << 20)
int hs_execute_static(const hs_plan *plan, const float *d_x, float *d_sums, float *d_max, uint8_t *d_argmax,
                      void *stream);
size_t hs_static_scratch_bytes(void);    /* HS_STATIC_SCRATCH_BYTES of the library that is loaded                 */

/*
 * hs_debug_greedy_paths — test-only: Greedy's drift j after each level, d_j[batch][L][nbins] uint8 (DEVICE),
 * because BASELINE.json north_star asks for bit-exact j paths and the production outputs do not expose j.
 * Valid for HS_GREEDY plans only (else HS_ERR_INVALID_ARG).  Not on the timed path.
 */
int hs_debug_greedy_paths(const hs_plan *plan, const float *d_x, uint8_t *d_j, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* HS_H */
