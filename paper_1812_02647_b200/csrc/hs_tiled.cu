// hs_tiled.cu — HS_ALGO_TILED dispatch (the tuned kernels).  A plan that no tuned kernel covers resolves to
// HS_ALGO_DIRECT.
#include "hs_internal.cuh"

namespace {
// Max always runs two-phase; freq-bin runs two-phase only when asked to (HS_ALGO_TWOPHASE), else the gather kernel.
bool two_phase(const hs_plan *p)
{
    return p->variant == HS_MAX || (p->variant == HS_FREQBIN && p->algo_req == HS_ALGO_TWOPHASE);
}
}  // namespace
bool hs_tiled_supported(const hs_plan *p) { return !two_phase(p) || hs_twophase_supported(p, p->batch); }

size_t hs_tiled_workspace_bytes(const hs_plan *p, int64_t batch)
{
    return two_phase(p) ? hs_twophase_workspace_bytes(p, batch) : 0;
}

int hs_tiled_launches(const hs_plan *p, int64_t batch)
{
    if (p->variant == HS_STANDARD) return hs_standard_tiled_launches(p, batch);
    if (two_phase(p)) return hs_twophase_launches(p, batch);
    return hs_greedy_gather_launches(p, batch);
}

int hs_launch_tiled(const hs_plan *p, const hs_buffers &buf, int64_t batch, void *ws, cudaStream_t stream)
{
    if (p->variant == HS_STANDARD) return hs_standard_tiled_launch(p, buf, batch, stream);
    if (two_phase(p)) return hs_twophase_launch(p, buf, batch, ws, stream);
    return hs_greedy_gather_launch(p, buf, batch, stream);
}
