// hs_tiled.cu — HS_ALGO_TILED dispatch (the tuned kernels).  A plan that no tuned kernel covers resolves to
// HS_ALGO_DIRECT.
#include "hs_internal.cuh"

namespace {
// eq. 2 with few harmonics: block maxima straight from the spectrum (the gather kernel), no workspace
bool max_gather(const hs_plan *p)
{
    if (p->variant != HS_MAX || p->Hmax > 4) return false;   // (Hmax = 8: the grouped kernel is faster)
    return p->algo_req == HS_ALGO_AUTO || p->algo_req == HS_ALGO_TILED || p->algo_req == HS_ALGO_GATHER;
}
// eq. 2 runs grouped when a group's slot fits L2 (else two-phase through HBM); eq. 3 runs grouped only when asked to.
bool grouped(const hs_plan *p)
{
    if (p->variant != HS_MAX && p->variant != HS_FREQBIN) return false;
    if (max_gather(p)) return false;
    if (p->algo_req == HS_ALGO_TWOPHASE || p->algo_req == HS_ALGO_GATHER) return false;
    if (p->variant == HS_FREQBIN && p->algo_req != HS_ALGO_GROUPED) return false;
    if (p->variant == HS_GREEDY) return false;
    return hs_grouped_supported(p);
}
// Max otherwise runs two-phase; freq-bin runs two-phase only when asked to (HS_ALGO_TWOPHASE).
bool two_phase(const hs_plan *p)
{
    if (grouped(p) || max_gather(p)) return false;
    return p->variant == HS_MAX || (p->variant == HS_FREQBIN && p->algo_req == HS_ALGO_TWOPHASE);
}
// freq-bin gathers from the spectrum-interleaved group copies when they fit L2, unless the plain gather is asked for
bool interleaved(const hs_plan *p)
{
    return !grouped(p) && !two_phase(p) && p->algo_req != HS_ALGO_GATHER && p->Hmax == 32 &&
           hs_interleaved_supported(p);
}
}  // namespace
bool hs_tiled_supported(const hs_plan *p)
{
    if (p->algo_req == HS_ALGO_GATHER && p->variant != HS_FREQBIN && p->variant != HS_GREEDY && !max_gather(p)) return false;
    if (p->algo_req == HS_ALGO_GROUPED) return grouped(p);
    return !two_phase(p) || hs_twophase_supported(p, p->batch);
}

size_t hs_tiled_workspace_bytes(const hs_plan *p, int64_t batch)
{
    if (p->variant == HS_STANDARD) return hs_standard_rb_supported(p) ? hs_standard_rb_workspace_bytes(p) : 0;
    if (grouped(p)) return hs_grouped_workspace_bytes(p, batch);
    if (two_phase(p)) return hs_twophase_workspace_bytes(p, batch);
    if (interleaved(p)) return hs_interleaved_workspace_bytes(p, batch);
    return 0;
}

int hs_tiled_launches(const hs_plan *p, int64_t batch)
{
    if (p->variant == HS_STANDARD) return hs_standard_rb_supported(p) ? 2 : hs_standard_tiled_launches(p, batch);   // memset node + kernel
    if (grouped(p)) return hs_grouped_launches(p, batch);
    if (two_phase(p)) return hs_twophase_launches(p, batch);
    if (interleaved(p)) return hs_interleaved_launches(p, batch);
    return hs_greedy_gather_launches(p, batch);
}

int hs_launch_tiled(const hs_plan *p, const hs_buffers &buf, int64_t batch, void *ws, cudaStream_t stream)
{
    if (p->variant == HS_STANDARD)
        return hs_standard_rb_supported(p) ? hs_standard_rb_launch(p, buf, batch, ws, stream) : hs_standard_tiled_launch(p, buf, batch, stream);
    if (grouped(p)) return hs_grouped_launch(p, buf, batch, ws, stream);
    if (two_phase(p)) return hs_twophase_launch(p, buf, batch, ws, stream);
    if (interleaved(p)) return hs_interleaved_launch(p, buf, batch, ws, stream);
    return hs_greedy_gather_launch(p, buf, batch, stream);
}

bool hs_tiled_has_ctrl(const hs_plan *p)
{
    if (p->variant == HS_STANDARD) return hs_standard_rb_supported(p);   // (tile counter; the error word stays zero)
    return grouped(p) || interleaved(p);
}

// hs_execute_complex: which resolved kernels form x from the complex series themselves (the others fall back to the
// direct family, which does): the gathers, the interleaved copy items, and eq. 2's grouped kernel at Hmax >= 8.
bool hs_tiled_supports_complex(const hs_plan *p)
{
    if (p->variant == HS_STANDARD) return false;                        // (both eq. 1 kernels stage x by TMA bulk copies)
    if (p->variant == HS_MAX) return max_gather(p) || (grouped(p) && p->Hmax >= 8);
    if (grouped(p) || two_phase(p)) return false;                       // (eq. 3 through the two-phase families: only when asked for)
    return true;                                                        // interleaved (eq. 3) or the plain gather (eqs. 3-4)
}
