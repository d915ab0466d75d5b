// hs_api.cu — the C ABI declared in include/hs.h: validation, plan bookkeeping, dispatch to the kernel families and
// the host-buffer pipeline.  No torch types, no allocation of device memory, no output on stdout/stderr.
#include <new>

#include "hs_internal.cuh"

namespace {
thread_local int g_last_error = HS_OK;

bool aligned(const void *p, size_t a) { return (reinterpret_cast<uintptr_t>(p) % a) == 0; }

int levels_of(int Hmax)
{
    switch (Hmax) {
        case 1: return 1;
        case 2: return 2;
        case 4: return 3;
        case 8: return 4;
        case 16: return 5;
        case 32: return 6;
        default: return -1;
    }
}

bool is_general(const hs_plan *p) { return p->nz > 1 || p->levels_mode != HS_LEVELS_DYADIC || p->window != HS_WINDOW_C2; }

void resolve_algo(hs_plan *p)
{
    if (is_general(p)) p->algo = HS_ALGO_GENERAL;
    else if (p->algo_req == HS_ALGO_DIRECT) p->algo = HS_ALGO_DIRECT;
    else if (p->algo_req == HS_ALGO_TILED || p->algo_req == HS_ALGO_TWOPHASE || p->algo_req == HS_ALGO_GATHER ||
             p->algo_req == HS_ALGO_GROUPED)
        p->algo = HS_ALGO_TILED;
    else p->algo = hs_tiled_supported(p) ? HS_ALGO_TILED : HS_ALGO_DIRECT;
    // the workspace and the host staging were sized for the previous algorithm: both have to be set again
    p->ws = nullptr;
    p->ws_bytes = 0;
    p->staging = nullptr;
    p->staging_bytes = 0;
    p->slab = 0;
    p->n_last_ctrl = 0;
}

// the plan's device must be current (function attributes, occupancy and the SM count are per device)
int check_device(const hs_plan *p)
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) {
        (void)cudaGetLastError();
        HS_FAIL(HS_ERR_CUDA);
    }
    if (dev != p->device) HS_FAIL(HS_ERR_INVALID_ARG);
    return HS_OK;
}

// remember which control block a launch used (hs_plan_device_status)
void note_ctrl(const hs_plan *p, const void *ws, bool first)
{
    if (first) p->n_last_ctrl = 0;
    if (ws && p->algo == HS_ALGO_TILED && hs_tiled_has_ctrl(p) && p->n_last_ctrl < HS_HOST_LANES) {
        for (int i = 0; i < p->n_last_ctrl; i++)
            if (p->last_ctrl[i] == ws) return;
        p->last_ctrl[p->n_last_ctrl++] = ws;
    }
}

int check_buffers(const hs_plan *p, const void *x, const void *sums, const void *vmax, const void *amax)
{
    if (!p || !x) HS_FAIL(HS_ERR_NULL_POINTER);
    if ((p->out_mode & HS_OUT_FULL) && !sums) HS_FAIL(HS_ERR_NULL_POINTER);
    if ((p->out_mode & HS_OUT_REDUCED) && (!vmax || !amax)) HS_FAIL(HS_ERR_NULL_POINTER);
    if (!aligned(x, 16) || !aligned(sums, 16) || !aligned(vmax, 16) || !aligned(amax, 16)) HS_FAIL(HS_ERR_MISALIGNED);
    return HS_OK;
}

int launch_family(const hs_plan *p, const hs_buffers &buf, int64_t batch, void *ws, cudaStream_t stream)
{
    if (p->algo == HS_ALGO_TILED && (!buf.cplx || hs_tiled_supports_complex(p))) return hs_launch_tiled(p, buf, batch, ws, stream);
    if (p->algo == HS_ALGO_GENERAL) return hs_launch_general(p, buf, batch, ws, stream);
    return hs_launch_direct(p, buf, batch, ws, stream);
}

size_t round_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// bytes of one slab's device buffers in the host pipeline, each region 256-byte aligned
struct slab_layout {
    size_t x, sums, vmax, amax, ws, total;
};
slab_layout layout_of(const hs_plan *p, int64_t slab)
{
    slab_layout s{};
    const size_t bins = (size_t)slab * (size_t)p->nbins * (size_t)p->nz;
    s.x = round_up(bins * 4, 256);
    s.sums = (p->out_mode & HS_OUT_FULL) ? round_up(bins * 4 * p->L, 256) : 0;
    s.vmax = (p->out_mode & HS_OUT_REDUCED) ? round_up(bins * 4, 256) : 0;
    s.amax = (p->out_mode & HS_OUT_REDUCED) ? round_up(bins, 256) : 0;
    s.ws = p->algo == HS_ALGO_TILED ? round_up(hs_tiled_workspace_bytes(p, slab), 256)
         : p->algo == HS_ALGO_GENERAL ? round_up(hs_general_workspace_bytes(p), 256) : 0;
    s.total = s.x + s.sums + s.vmax + s.amax + s.ws;
    return s;
}
}  // namespace

void hs_set_error(int code) { g_last_error = code; }

extern "C" {

int hs_last_error(void) { return g_last_error; }

const char *hs_error_string(int code)
{
    switch (code) {
        case HS_OK: return "ok";
        case HS_ERR_INVALID_ARG: return "invalid argument";
        case HS_ERR_NULL_POINTER: return "required pointer is NULL";
        case HS_ERR_MISALIGNED: return "pointer is not sufficiently aligned";
        case HS_ERR_UNSUPPORTED: return "no CUDA device of compute capability 10.x (sm_100) is current";
        case HS_ERR_WORKSPACE: return "workspace or staging buffer missing or too small";
        case HS_ERR_CUDA: return "CUDA runtime call or kernel launch failed";
        case HS_ERR_DEVICE_TIMEOUT: return "a kernel gave up waiting for another thread block: outputs are not valid";
        case HS_ERR_SCRATCH_LIMIT:
            return "one spectrum's per-harmonic arrays exceed the library's built-in scratch array (HS_STATIC_SCRATCH_BYTES)";
        default: return "unknown hs_status code";
    }
}

const char *hs_version(void) { return "hs 0.2 (sm_100a)"; }

static hs_plan *create_plan(int64_t nbins, int64_t nz, int64_t batch, int Hmax, int variant, int out_mode, int levels, int window)
{
    const bool all = levels == HS_LEVELS_ALL;
    const int L = all ? Hmax : levels_of(Hmax);
    bool bad = nbins < 4 || nbins > ((int64_t)1 << 25) || (nbins % 4) != 0 || batch < 1 || L < 1 ||
               variant < HS_STANDARD || variant > HS_GREEDY || out_mode < HS_OUT_FULL || out_mode > HS_OUT_BOTH ||
               nz < 1 || batch > ((int64_t)1 << 40) / (nbins * (nz > 0 ? nz : 1)) || batch > (int64_t)0x7fffffff;
    bad = bad || (levels != HS_LEVELS_DYADIC && levels != HS_LEVELS_ALL) ||
          (window != HS_WINDOW_C2 && window != HS_WINDOW_PRINTED && window != HS_TERM_INTERP);
    bad = bad || (window == HS_TERM_INTERP && variant != HS_STANDARD);
    bad = bad || (all && (Hmax < 1 || Hmax > 64 || nbins > ((int64_t)1 << 24)));
    bad = bad || (window == HS_WINDOW_PRINTED && variant != HS_MAX);
    bad = bad || (nz > 1 && ((nz % 2) == 0 || nz > 4095 || all || window != HS_WINDOW_C2 ||
                             (variant != HS_STANDARD && variant != HS_FREQBIN)));
    if (bad) {
        hs_set_error(HS_ERR_INVALID_ARG);
        return nullptr;
    }
    int dev = 0, major = 0, sms = 0, smem = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) {
        (void)cudaGetLastError();
        hs_set_error(HS_ERR_UNSUPPORTED);
        return nullptr;
    }
    if (major != 10) {
        hs_set_error(HS_ERR_UNSUPPORTED);
        return nullptr;
    }
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev) != cudaSuccess) {
        (void)cudaGetLastError();
        hs_set_error(HS_ERR_CUDA);
        return nullptr;
    }
    hs_plan *p = new (std::nothrow) hs_plan();
    if (!p) {
        hs_set_error(HS_ERR_CUDA);
        return nullptr;
    }
    p->nbins = nbins;
    p->batch = batch;
    p->nz = nz;
    p->levels_mode = levels;
    p->window = window;
    p->Hmax = Hmax;
    p->L = L;
    p->variant = variant;
    p->out_mode = out_mode;
    p->algo_req = HS_ALGO_AUTO;
    p->device = dev;
    p->sm_count = sms;
    p->smem_optin = (size_t)smem;
    p->staging = nullptr;
    p->staging_bytes = 0;
    p->slab = 0;
    p->lanes_ready = false;
    resolve_algo(p);
    return p;
}

hs_plan *hs_plan_create(int64_t nbins, int64_t batch, int Hmax, int variant, int out_mode)
{
    return create_plan(nbins, 1, batch, Hmax, variant, out_mode, HS_LEVELS_DYADIC, HS_WINDOW_C2);
}

hs_plan *hs_plan_create_ex(int64_t nbins, int64_t batch, int Hmax, int variant, int out_mode, int levels, int window)
{
    return create_plan(nbins, 1, batch, Hmax, variant, out_mode, levels, window);
}

hs_plan *hs_plan_create_2d(int64_t nbins, int64_t nz, int64_t batch, int Hmax, int variant, int out_mode)
{
    if (nz < 1 || (nz % 2) == 0 || (variant != HS_STANDARD && variant != HS_FREQBIN)) {
        hs_set_error(HS_ERR_INVALID_ARG);
        return nullptr;
    }
    return create_plan(nbins, nz, batch, Hmax, variant, out_mode, HS_LEVELS_DYADIC, HS_WINDOW_C2);
}

int hs_destroy(hs_plan *p)
{
    if (!p) return HS_OK;
    if (p->lanes_ready) {
        for (int i = 0; i < HS_HOST_LANES; i++) {
            cudaEventDestroy(p->lane_done[i]);
            cudaStreamDestroy(p->lane_stream[i]);
        }
        cudaEventDestroy(p->fork);
        (void)cudaGetLastError();
    }
    delete p;
    return HS_OK;
}

int hs_plan_levels(const hs_plan *p) { return p ? p->L : -1; }
int hs_plan_algo(const hs_plan *p) { return p ? p->algo : -1; }

int hs_plan_set_algo(hs_plan *p, int algo)
{
    if (!p) HS_FAIL(HS_ERR_NULL_POINTER);
    if (algo < HS_ALGO_AUTO || algo > HS_ALGO_GROUPED) HS_FAIL(HS_ERR_INVALID_ARG);
    if (is_general(p) && algo != HS_ALGO_AUTO) HS_FAIL(HS_ERR_INVALID_ARG);      // (one family: HS_ALGO_GENERAL)
    if ((algo == HS_ALGO_TWOPHASE || algo == HS_ALGO_GROUPED) && p->variant != HS_MAX && p->variant != HS_FREQBIN)
        HS_FAIL(HS_ERR_INVALID_ARG);
    if (algo == HS_ALGO_GATHER && p->variant != HS_GREEDY && p->variant != HS_FREQBIN &&
        !(p->variant == HS_MAX && p->Hmax <= 4))
        HS_FAIL(HS_ERR_INVALID_ARG);
    const int before = p->algo_req;
    p->algo_req = algo;
    if ((algo == HS_ALGO_TILED || algo == HS_ALGO_TWOPHASE || algo == HS_ALGO_GATHER || algo == HS_ALGO_GROUPED) &&
        !hs_tiled_supported(p)) {
        p->algo_req = before;
        HS_FAIL(HS_ERR_INVALID_ARG);
    }
    resolve_algo(p);
    return HS_OK;
}

size_t hs_plan_workspace_bytes(const hs_plan *p)
{
    if (!p) return 0;
    if (p->algo == HS_ALGO_GENERAL) return hs_general_workspace_bytes(p);
    return p->algo == HS_ALGO_TILED ? hs_tiled_workspace_bytes(p, p->batch) : 0;
}

int hs_plan_set_workspace(hs_plan *p, void *d_ws, size_t bytes)
{
    if (!p) HS_FAIL(HS_ERR_NULL_POINTER);
    const size_t need = hs_plan_workspace_bytes(p);
    if (need == 0) {
        p->ws = d_ws;
        p->ws_bytes = bytes;
        return HS_OK;
    }
    if (!d_ws) HS_FAIL(HS_ERR_NULL_POINTER);
    if (!aligned(d_ws, 256)) HS_FAIL(HS_ERR_MISALIGNED);
    if (bytes < need) HS_FAIL(HS_ERR_WORKSPACE);
    p->ws = d_ws;
    p->ws_bytes = bytes;
    return HS_OK;
}

int hs_plan_launches(const hs_plan *p)
{
    if (!p) return -1;
    if (p->algo == HS_ALGO_TILED) return hs_tiled_launches(p, p->batch);
    if (p->algo == HS_ALGO_GENERAL) return hs_general_launches(p);   // (counted next to the launcher: hs_general.cu)
    const int64_t tiles = (p->nbins + 255) / 256;
    const int64_t max_spectra = ((int64_t)1 << 30) / tiles;
    return (int)((p->batch + max_spectra - 1) / max_spectra);
}

int hs_execute(const hs_plan *p, const float *d_x, float *d_sums, float *d_max, uint8_t *d_argmax, void *stream)
{
    int rc = check_buffers(p, d_x, d_sums, d_max, d_argmax);
    if (rc != HS_OK) return rc;
    if ((rc = check_device(p)) != HS_OK) return rc;
    if (hs_plan_workspace_bytes(p) > 0 && (!p->ws || p->ws_bytes < hs_plan_workspace_bytes(p))) HS_FAIL(HS_ERR_WORKSPACE);
    note_ctrl(p, p->ws, true);
    hs_buffers buf{d_x, (p->out_mode & HS_OUT_FULL) ? d_sums : nullptr, (p->out_mode & HS_OUT_REDUCED) ? d_max : nullptr,
                   (p->out_mode & HS_OUT_REDUCED) ? d_argmax : nullptr, nullptr, {}, false, 0.0f};
    return launch_family(p, buf, p->batch, p->ws, static_cast<cudaStream_t>(stream));
}

int hs_execute_complex(const hs_plan *p, const float *d_F, float scale, float *d_sums, float *d_max, uint8_t *d_argmax,
                       void *stream)
{
    int rc = check_buffers(p, d_F, d_sums, d_max, d_argmax);
    if (rc != HS_OK) return rc;
    if (is_general(p) || !(scale == scale)) HS_FAIL(HS_ERR_INVALID_ARG);
    if ((rc = check_device(p)) != HS_OK) return rc;
    const bool tiled = p->algo == HS_ALGO_TILED && hs_tiled_supports_complex(p);
    if (tiled && hs_plan_workspace_bytes(p) > 0 && (!p->ws || p->ws_bytes < hs_plan_workspace_bytes(p))) HS_FAIL(HS_ERR_WORKSPACE);
    note_ctrl(p, tiled ? p->ws : nullptr, true);
    hs_buffers buf{d_F, (p->out_mode & HS_OUT_FULL) ? d_sums : nullptr, (p->out_mode & HS_OUT_REDUCED) ? d_max : nullptr,
                   (p->out_mode & HS_OUT_REDUCED) ? d_argmax : nullptr, nullptr, {}, true, scale};
    return launch_family(p, buf, p->batch, p->ws, static_cast<cudaStream_t>(stream));
}

int hs_execute_candidates(const hs_plan *p, const float *d_x, float threshold, hs_candidate *d_cand, int64_t capacity,
                          unsigned long long *d_count, void *stream)
{
    if (!p || !d_x || !d_count || (!d_cand && capacity > 0)) HS_FAIL(HS_ERR_NULL_POINTER);
    if (p->out_mode != HS_OUT_REDUCED || capacity < 0 || !(threshold == threshold) || p->nz > 1) HS_FAIL(HS_ERR_INVALID_ARG);
    if (!aligned(d_x, 16) || !aligned(d_cand, 16) || !aligned(d_count, 8)) HS_FAIL(HS_ERR_MISALIGNED);
    const int rcd = check_device(p);
    if (rcd != HS_OK) return rcd;
    if (hs_plan_workspace_bytes(p) > 0 && (!p->ws || p->ws_bytes < hs_plan_workspace_bytes(p))) HS_FAIL(HS_ERR_WORKSPACE);
    note_ctrl(p, p->ws, true);
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    HS_CUDA_OK(cudaMemsetAsync(d_count, 0, sizeof(unsigned long long), s));
    hs_buffers buf{d_x, nullptr, nullptr, nullptr, nullptr, {}, false, 0.0f};
    // a kernel tests `cand` to choose between appending and storing: with no room at all it still has to count
    static hs_candidate *const kNowhere = reinterpret_cast<hs_candidate *>(16);
    buf.sink.cand = capacity > 0 ? d_cand : kNowhere;
    buf.sink.count = d_count;
    buf.sink.cap = capacity;
    buf.sink.thr = threshold;
    buf.sink.b0 = 0;
    return launch_family(p, buf, p->batch, p->ws, s);
}

int hs_debug_greedy_paths(const hs_plan *p, const float *d_x, uint8_t *d_j, void *stream)
{
    if (!p || !d_x || !d_j) HS_FAIL(HS_ERR_NULL_POINTER);
    if (p->variant != HS_GREEDY) HS_FAIL(HS_ERR_INVALID_ARG);
    if (!aligned(d_x, 16) || !aligned(d_j, 16)) HS_FAIL(HS_ERR_MISALIGNED);
    const int rcd = check_device(p);
    if (rcd != HS_OK) return rcd;
    if (hs_plan_workspace_bytes(p) > 0 && (!p->ws || p->ws_bytes < hs_plan_workspace_bytes(p))) HS_FAIL(HS_ERR_WORKSPACE);
    note_ctrl(p, p->ws, true);
    // the plan's own kernel family in its own launch configuration, writing j instead of the outputs
    hs_buffers buf{d_x, nullptr, nullptr, nullptr, d_j, {}, false, 0.0f};
    return launch_family(p, buf, p->batch, p->ws, static_cast<cudaStream_t>(stream));
}

int hs_plan_device_status(const hs_plan *p, void *stream)
{
    if (!p) HS_FAIL(HS_ERR_NULL_POINTER);
    HS_CUDA_OK(cudaStreamSynchronize(static_cast<cudaStream_t>(stream)));
    for (int i = 0; i < p->n_last_ctrl; i++) {
        int words[4] = {0, 0, 0, 0};
        HS_CUDA_OK(cudaMemcpy(words, p->last_ctrl[i], sizeof(words), cudaMemcpyDeviceToHost));
        if (words[HS_CTRL_ERROR] != 0) HS_FAIL(HS_ERR_DEVICE_TIMEOUT);
    }
    return HS_OK;
}

size_t hs_plan_host_staging_bytes(const hs_plan *p, int64_t slab)
{
    if (!p || slab < 1 || slab > p->batch) return 0;
    return layout_of(p, slab).total * HS_HOST_LANES;
}

int hs_plan_set_host_staging(hs_plan *p, void *d_staging, size_t bytes, int64_t slab)
{
    if (!p || !d_staging) HS_FAIL(HS_ERR_NULL_POINTER);
    if (slab < 1 || slab > p->batch) HS_FAIL(HS_ERR_INVALID_ARG);
    if (!aligned(d_staging, 256)) HS_FAIL(HS_ERR_MISALIGNED);
    if (bytes < hs_plan_host_staging_bytes(p, slab)) HS_FAIL(HS_ERR_WORKSPACE);
    if (!p->lanes_ready) {
        for (int i = 0; i < HS_HOST_LANES; i++) {
            HS_CUDA_OK(cudaStreamCreateWithFlags(&p->lane_stream[i], cudaStreamNonBlocking));
            HS_CUDA_OK(cudaEventCreateWithFlags(&p->lane_done[i], cudaEventDisableTiming));
        }
        HS_CUDA_OK(cudaEventCreateWithFlags(&p->fork, cudaEventDisableTiming));
        p->lanes_ready = true;
    }
    p->staging = d_staging;
    p->staging_bytes = bytes;
    p->slab = slab;
    return HS_OK;
}

int hs_execute_host(hs_plan *p, const float *h_x, float *h_sums, float *h_max, uint8_t *h_argmax, void *stream)
{
    if (!p || !h_x) HS_FAIL(HS_ERR_NULL_POINTER);
    if ((p->out_mode & HS_OUT_FULL) && !h_sums) HS_FAIL(HS_ERR_NULL_POINTER);
    if ((p->out_mode & HS_OUT_REDUCED) && (!h_max || !h_argmax)) HS_FAIL(HS_ERR_NULL_POINTER);
    if (!p->lanes_ready || !p->staging) HS_FAIL(HS_ERR_WORKSPACE);
    const int rcd = check_device(p);
    if (rcd != HS_OK) return rcd;
    cudaStream_t user = static_cast<cudaStream_t>(stream);
    const slab_layout lay = layout_of(p, p->slab);
    if (p->staging_bytes < lay.total * HS_HOST_LANES) HS_FAIL(HS_ERR_WORKSPACE);   // (sized for another algorithm)
    p->n_last_ctrl = 0;
    const int64_t N = p->nbins * p->nz;
    HS_CUDA_OK(cudaEventRecord(p->fork, user));
    for (int i = 0; i < HS_HOST_LANES; i++) HS_CUDA_OK(cudaStreamWaitEvent(p->lane_stream[i], p->fork, 0));
    int lane = 0;
    for (int64_t b0 = 0; b0 < p->batch; b0 += p->slab, lane = (lane + 1) % HS_HOST_LANES) {
        const int64_t nb = (p->batch - b0 < p->slab) ? p->batch - b0 : p->slab;
        const size_t bins = (size_t)nb * (size_t)N;                     // (N = elements per batch entry)
        char *base = static_cast<char *>(p->staging) + (size_t)lane * lay.total;
        float *dx = reinterpret_cast<float *>(base);
        float *dsums = lay.sums ? reinterpret_cast<float *>(base + lay.x) : nullptr;
        float *dmax = lay.vmax ? reinterpret_cast<float *>(base + lay.x + lay.sums) : nullptr;
        uint8_t *damax = lay.amax ? reinterpret_cast<uint8_t *>(base + lay.x + lay.sums + lay.vmax) : nullptr;
        void *dws = lay.ws ? base + lay.x + lay.sums + lay.vmax + lay.amax : nullptr;
        cudaStream_t s = p->lane_stream[lane];
        HS_CUDA_OK(cudaMemcpyAsync(dx, h_x + (size_t)b0 * N, bins * 4, cudaMemcpyHostToDevice, s));
        hs_buffers buf{dx, dsums, dmax, damax, nullptr, {}, false, 0.0f};
        note_ctrl(p, dws, false);
        const int rc = launch_family(p, buf, nb, dws, s);
        if (rc != HS_OK) return rc;
        if (dsums)
            HS_CUDA_OK(cudaMemcpyAsync(h_sums + (size_t)b0 * p->L * N, dsums, bins * 4 * p->L, cudaMemcpyDeviceToHost, s));
        if (dmax) {
            HS_CUDA_OK(cudaMemcpyAsync(h_max + (size_t)b0 * N, dmax, bins * 4, cudaMemcpyDeviceToHost, s));
            HS_CUDA_OK(cudaMemcpyAsync(h_argmax + (size_t)b0 * N, damax, bins, cudaMemcpyDeviceToHost, s));
        }
    }
    for (int i = 0; i < HS_HOST_LANES; i++) {
        HS_CUDA_OK(cudaEventRecord(p->lane_done[i], p->lane_stream[i]));
        HS_CUDA_OK(cudaStreamWaitEvent(user, p->lane_done[i], 0));
    }
    return HS_OK;
}

}  // extern "C"
