// hs_tiled.cu — HS_ALGO_TILED dispatch (the tuned kernels).  Filled in per variant; a plan that no tuned kernel
// covers resolves to HS_ALGO_DIRECT.
#include "hs_internal.cuh"

bool hs_tiled_supported(const hs_plan *) { return false; }
size_t hs_tiled_workspace_bytes(const hs_plan *, int64_t) { return 0; }
int hs_tiled_launches(const hs_plan *, int64_t) { return 0; }
int hs_launch_tiled(const hs_plan *, const hs_buffers &, int64_t, void *, cudaStream_t) { HS_FAIL(HS_ERR_INVALID_ARG); }
