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
__device__ __forceinline__ int ld_relaxed(const int *p)
{
    int v;
    asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
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

// ---- producer/consumer ring scheduling: two queues of work items, each handed out in order by fetch-and-add.
// "T" items produce a group's data into ring slot (group % R), "G" items consume it.
// ---- tickets (thread 0 only).  A CTA holds up to one ticket of each queue (fetch-and-add: no retries under contention)
// and runs whichever is runnable, gathers first; a ticket that is not runnable yet is simply kept while the other kind
// of work goes on.  The lowest unfinished ticket of one of the two queues is always runnable (a G ticket of group a needs
// the T tickets of group a, a T ticket of group b needs the G tickets of group b - R: the dependences point strictly
// downwards), and it is held by a CTA that polls it, so the schedule cannot deadlock.
constexpr int kNoTicket = -1, kExhausted = -2;
struct tickets {
    int *tq, *gq, *doneT, *doneG;
    int totalT, totalG, nT, nG, R;
    int readyT, freeG;                                                  // groups already seen complete (acquired)
    int gt, tt;                                                         // the tickets in hand

    __device__ __forceinline__ void draw_g()
    {
        if (gt == kNoTicket) {
            gt = atomicAdd(gq, 1);
            if (gt >= totalG) gt = kExhausted;
        }
    }
    __device__ __forceinline__ void draw_t()
    {
        if (tt == kNoTicket) {
            tt = atomicAdd(tq, 1);
            if (tt >= totalT) tt = kExhausted;
        }
    }
    // polls with relaxed loads; the acquire (which also invalidates the SM's L1) only once the counter is complete
    __device__ __forceinline__ bool g_runnable()
    {
        if (gt < 0) return false;
        const int gs = gt / nG;
        if (gs <= readyT) return true;
        if (ld_relaxed(doneT + gs) < nT) return false;
        (void)ld_acquire(doneT + gs);
        readyT = gs;
        return true;
    }
    __device__ __forceinline__ bool t_runnable()
    {
        if (tt < 0) return false;
        const int fs = tt / nT - R;
        if (fs <= freeG) return true;
        if (ld_relaxed(doneG + fs) < nG) return false;
        (void)ld_acquire(doneG + fs);
        freeG = fs;
        return true;
    }
    // Without waiting: the next item to run (kind | index); kNoTicket if neither ticket in hand is runnable right now;
    // kExhausted when both queues are exhausted.
    __device__ __forceinline__ int try_next(int kItemG)
    {
        draw_g();
        draw_t();
        if (g_runnable()) {
            const int it = kItemG | gt;
            gt = kNoTicket;
            return it;
        }
        if (t_runnable()) {
            const int it = tt;
            tt = kNoTicket;
            return it;
        }
        return (gt == kExhausted && tt == kExhausted) ? kExhausted : kNoTicket;
    }
    // the next item to run: kind | index, or kNoTicket when both queues are exhausted (or the poll limit was hit)
    __device__ __forceinline__ int next(int *ctrl, unsigned limit, int kItemG)
    {
        unsigned spins = 0;
        int it = kNoTicket;
        for (;;) {
            draw_g();
            draw_t();
            if (g_runnable()) {
                it = kItemG | gt;
                gt = kNoTicket;
                break;
            }
            if (t_runnable()) {
                it = tt;
                tt = kNoTicket;
                break;
            }
            if (gt == kExhausted && tt == kExhausted) break;
            if (++spins > limit || ((spins & 255u) == 0 && ld_relaxed(ctrl + HS_CTRL_ERROR) != 0)) {
                atomicExch(ctrl + HS_CTRL_ERROR, 1);
                break;
            }
            __nanosleep(200);
        }
        if (spins) {
            atomicAdd(ctrl + HS_CTRL_STATS, 1);
            atomicAdd(ctrl + HS_CTRL_STATS + 1, (int)(spins > 0x7fffu ? 0x7fffu : spins));
        }
        return it;
    }
};

}  // namespace hssync
