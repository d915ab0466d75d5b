// hs_sync.cuh — inter-CTA synchronisation through counters in global memory, shared by the persistent kernels.
// A waiter polls with acquire loads; a bounded number of polls so that a scheduling bug cannot hang the GPU: on
// time-out the error word of the control block (HS_CTRL_ERROR) is set, which hs_plan_device_status reports.
#pragma once
#include "hs_internal.cuh"

namespace hssync {

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

// one thread: wait until *cnt >= target.  ctrl = the workspace's control block; stat = two words of wait statistics
// (waits that had to spin, polls) or nullptr.  Returns false if it gave up (the error flag is then set).
__device__ __forceinline__ bool wait_count(const int *cnt, int target, int *ctrl, int *stat, unsigned limit)
{
    unsigned spins = 0;
    bool ok = true;
    while (ld_acquire(cnt) < target) {
        if (++spins > limit || ((spins & 1023u) == 0 && ld_acquire(ctrl + HS_CTRL_ERROR) != 0)) {
            atomicExch(ctrl + HS_CTRL_ERROR, 1);
            ok = false;
            break;
        }
        __nanosleep(40);
    }
    if (spins && stat) {
        atomicAdd(stat, 1);
        atomicAdd(stat + 1, (int)(spins > 0x7fffu ? 0x7fffu : spins));
    }
    return ok;
}

}  // namespace hssync
