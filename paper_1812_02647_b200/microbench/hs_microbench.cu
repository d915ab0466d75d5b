// hs_microbench.cu — the hardware rates DESIGN.md section 6 quotes as secondary roofs of the harmonic sum on B200:
// distributed-shared-memory (cluster) gather bandwidth, scattered-sector load rates through L1 and L2, and how much of
// a dirty, repeatedly rewritten buffer stays resident in L2 while a stream passes through.  Stand-alone program,
// built and run by `python -m paper_1812_02647_b200.microbench` (nvcc -gencode arch=compute_100a,code=sm_100a).
// SURVEY.md section 7.1 step 7 asks for the first measurement before deciding eq. 4's design (candidate (d): a cluster
// holding a whole 2^18-bin spectrum in distributed shared memory).
#include <cooperative_groups.h>
#include <cuda_runtime.h>

#include <cstdio>
#include <cstdlib>
#include <utility>
#include <vector>

namespace cg = cooperative_groups;

#define CK(x)                                                                                   \
    do {                                                                                        \
        cudaError_t e_ = (x);                                                                   \
        if (e_ != cudaSuccess) {                                                                \
            printf("CUDA error %s at %s:%d\n", cudaGetErrorString(e_), __FILE__, __LINE__);     \
            exit(1);                                                                            \
        }                                                                                       \
    } while (0)

__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ unsigned mapa(unsigned addr, unsigned rank)
{
    unsigned r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
    return r;
}
__device__ __forceinline__ float ld_dsmem(unsigned addr)
{
    float v;
    asm volatile("ld.shared::cluster.f32 %0, [%1];" : "=f"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ float4 ld_dsmem4(unsigned addr)
{
    float4 v;
    asm volatile("ld.shared::cluster.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
    return v;
}

// ---- DSMEM gather: every thread reads `iters` x UNROLL words (or float4) from the shared memory of the CTAs of its
// cluster.  MODE 0: random word anywhere in the cluster (a hashed index); MODE 1: lane-strided (stride 9 words) inside a
// randomly chosen CTA; MODE 2: the same addresses but always in the thread's OWN CTA (the local-shared-memory baseline).
template <int VEC, int MODE>
__global__ void dsmem_gather(float *out, int words_per_cta, int iters)
{
    extern __shared__ __align__(16) float sm[];
    cg::cluster_group cluster = cg::this_cluster();
    const unsigned csize = cluster.num_blocks(), crank = cluster.block_rank();
    for (int i = threadIdx.x; i < words_per_cta; i += blockDim.x) sm[i] = (float)(i & 255) * 1e-3f;
    cluster.sync();
    const unsigned base = smem_u32(sm);
    unsigned h = (blockIdx.x * blockDim.x + threadIdx.x) * 2654435761u + 12345u;
    const unsigned mask = (unsigned)words_per_cta - 1u;       // words_per_cta is a power of two
    float acc = 0.f;
    constexpr int UNROLL = 8;
    for (int it = 0; it < iters; it++) {
        unsigned addr[UNROLL];
#pragma unroll
        for (int u = 0; u < UNROLL; u++) {
            h = h * 1664525u + 1013904223u;
            unsigned w, rank;
            if (MODE == 0) {
                w = (h >> 8) & mask;
                rank = (h >> 4) % csize;
            } else {
                const unsigned warp_h = __shfl_sync(0xffffffffu, h, 0);
                w = (((warp_h >> 8) & mask) + 9u * (threadIdx.x & 31)) & mask;
                rank = MODE == 2 ? crank : (warp_h >> 4) % csize;
            }
            if (VEC == 4) w &= ~3u;
            addr[u] = mapa(base + 4u * w, rank);
        }
#pragma unroll
        for (int u = 0; u < UNROLL; u++) {
            if (VEC == 4) {
                const float4 v = ld_dsmem4(addr[u]);
                acc += v.x + v.y + v.z + v.w;
            } else {
                acc += ld_dsmem(addr[u]);
            }
        }
    }
    cluster.sync();                                           // no CTA may exit while its memory is still being read
    if (acc == 123.456f) out[0] = acc;
}

template <int VEC, int MODE>
void run_dsmem(int csize, int sms, float *d_out, const char *what)
{
    const int threads = 512, words = 32768;                   // 128 KiB of shared memory per CTA, 1 CTA per SM
    const int iters = 256;
    auto kern = dsmem_gather<VEC, MODE>;
    CK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, words * 4));
    if (csize > 8) CK(cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
    cudaLaunchConfig_t cfg = {};
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = csize;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.blockDim = dim3(threads);
    cfg.dynamicSmemBytes = words * 4;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    int nclusters = 0;
    cfg.gridDim = dim3(csize);
    if (cudaOccupancyMaxActiveClusters(&nclusters, kern, &cfg) != cudaSuccess || nclusters < 1) {
        (void)cudaGetLastError();
        printf("DSMEM %-44s cluster %2d: not launchable\n", what, csize);
        return;
    }
    const int grid = nclusters * csize;                       // one wave of co-resident clusters
    cfg.gridDim = dim3(grid);
    cudaEvent_t e0, e1;
    CK(cudaEventCreate(&e0));
    CK(cudaEventCreate(&e1));
    CK(cudaLaunchKernelEx(&cfg, kern, d_out, words, 8));
    CK(cudaDeviceSynchronize());
    CK(cudaEventRecord(e0));
    CK(cudaLaunchKernelEx(&cfg, kern, d_out, words, iters));
    CK(cudaEventRecord(e1));
    CK(cudaDeviceSynchronize());
    float ms = 0;
    CK(cudaEventElapsedTime(&ms, e0, e1));
    const double loads = (double)grid * threads * iters * 8;
    const double bytes = loads * 4 * VEC;
    printf("DSMEM %-44s cluster %2d: %3d clusters = %3d CTAs (of %d SMs)  %7.3f ms  %7.1f G loads/s  %8.1f GB/s  %6.1f B/clk/SM(@1.965 GHz, busy SMs)\n",
           what, csize, nclusters, grid, sms, ms, loads / ms * 1e-6, bytes / ms * 1e-6, bytes / (ms * 1e-3) / grid / 1.965e9);
}

// ---- scattered 4-byte loads from an L2-resident buffer: one word per 32-byte sector, through L1 (ld.global.nc) or
// L2 only (.cg); PAIR = 1 adds the right neighbour word (same sector 7 times in 8), as Greedy's l/r pair does.
template <int CG, int PAIR>
__global__ void scattered(const float *__restrict__ buf, unsigned mask, int iters, float *out)
{
    unsigned h = (blockIdx.x * blockDim.x + threadIdx.x) * 2654435761u + 777u;
    float acc = 0.f;
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int u = 0; u < 8; u++) {
            h = h * 1664525u + 1013904223u;
            const unsigned w = (h >> 6) & mask;
            float a, b = 0.f;
            if (CG) {
                asm volatile("ld.global.cg.f32 %0, [%1];" : "=f"(a) : "l"(buf + w));
                if (PAIR) asm volatile("ld.global.cg.f32 %0, [%1];" : "=f"(b) : "l"(buf + w + 1));
            } else {
                a = __ldg(buf + w);
                if (PAIR) b = __ldg(buf + w + 1);
            }
            acc += a + b;
        }
    }
    if (acc == 123.456f) out[0] = acc;
}

template <int CG, int PAIR>
void run_scattered(const float *d_buf, size_t words, int sms, float *d_out, const char *what)
{
    const int threads = 256, ctas = sms * 8, iters = 64;
    cudaEvent_t e0, e1;
    CK(cudaEventCreate(&e0));
    CK(cudaEventCreate(&e1));
    scattered<CG, PAIR><<<ctas, threads>>>(d_buf, (unsigned)words - 2, 4, d_out);
    CK(cudaDeviceSynchronize());
    CK(cudaEventRecord(e0));
    scattered<CG, PAIR><<<ctas, threads>>>(d_buf, (unsigned)words - 2, iters, d_out);
    CK(cudaEventRecord(e1));
    CK(cudaDeviceSynchronize());
    float ms = 0;
    CK(cudaEventElapsedTime(&ms, e0, e1));
    const double pos = (double)ctas * threads * iters * 8;
    printf("scattered %-34s %4zu MiB buffer: %7.3f ms  %7.1f G positions/s = %5.2f per clk per SM (@1.965 GHz)\n", what,
           words * 4 >> 20, ms, pos / ms * 1e-6, pos / (ms * 1e-3) / sms / 1.965e9);
}

// ---- dirty L2 residency: a ring of `ring_bytes` is rewritten and re-read over and over while a stream of
// `stream_ratio` x as many bytes is read (evict-first) and as many written (streaming stores) in between: the DRAM
// traffic the ring adds is what does not stay resident.  Measured by time only here (ncu gives the bytes).
__global__ void ring_and_stream(float4 *ring, size_t ring_v4, const float4 *src, float4 *dst, size_t stream_v4, int rounds)
{
    const size_t tid = (size_t)blockIdx.x * blockDim.x + threadIdx.x, nth = (size_t)gridDim.x * blockDim.x;
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int r = 0; r < rounds; r++) {
        for (size_t i = tid; i < ring_v4; i += nth) {
            float4 v = ring[i];
            v.x += 1.f;
            ring[i] = v;
        }
        const float4 *s = src + (size_t)r * stream_v4;
        float4 *d = dst + (size_t)r * stream_v4;
        for (size_t i = tid; i < stream_v4; i += nth) {
            float4 v;
            asm volatile("ld.global.cs.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(s + i));
            acc.x += v.x;
            asm volatile("st.global.cs.v4.f32 [%0], {%1,%2,%3,%4};" ::"l"(d + i), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
        }
    }
    if (acc.x == 123.456f) dst[0] = acc;
}

// ---- the two dies.  die_probe: one thread per SM times a chain of dependent L2 loads (.cg) on a few fixed 128-byte lines:
// an SM sees a line either in its own die's L2 partition or across the die link, so for every line the SMs fall into
// two latency classes -- that is the SM -> die map.  ring_by_die: the dirty-ring test above with the ring either shared by
// all CTAs or split into two halves that are each touched by the CTAs of ONE die only (does a die-private workspace stay
// resident better?).
__global__ void die_probe(unsigned *buf, int nlines, int stride_words, int iters, unsigned *out)
{
    extern __shared__ float die_pad[];
    unsigned smid;
    asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
    if (threadIdx.x != 0) return;
    for (int l = 0; l < nlines; l++) {
        unsigned *ptr = buf + (size_t)l * stride_words;
        unsigned v;
        asm volatile("ld.global.cg.u32 %0, [%1];" : "=r"(v) : "l"(ptr) : "memory");
        unsigned best = 0xffffffffu;
        for (int rep = 0; rep < 8; rep++) {
            unsigned idx = 0;
            const long long t0 = clock64();
            for (int i = 0; i < iters; i++) {
                asm volatile("ld.global.cg.u32 %0, [%1];" : "=r"(v) : "l"(ptr + idx) : "memory");
                idx = v;                                   // the buffer holds zeros: a dependent chain on one line
            }
            const unsigned dt = (unsigned)(clock64() - t0);
            if (dt < best) best = dt;
            if (idx == 12345u) out[0] = 1;
        }
        out[(size_t)smid * nlines + l] = best;
    }
}

__global__ void __launch_bounds__(512, 2)
ring_by_die(float4 *ring, size_t ring_v4, const float4 *src, float4 *dst, size_t stream_v4, int rounds, int split,
            const int *die, int *ticket, int ncta0, int ncta1)
{
    extern __shared__ float die_pad[];
    __shared__ int s_t, s_d;
    if (threadIdx.x == 0) {
        unsigned smid;
        asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
        s_d = die[smid];
        s_t = atomicAdd(ticket + s_d, 1);
    }
    __syncthreads();
    const size_t tid = (size_t)blockIdx.x * blockDim.x + threadIdx.x, nth = (size_t)gridDim.x * blockDim.x;
    size_t rt = tid, rn = nth, r0 = 0, rlen = ring_v4;
    if (split) {
        rt = (size_t)s_t * blockDim.x + threadIdx.x;
        rn = (size_t)(s_d ? ncta1 : ncta0) * blockDim.x;
        rlen = ring_v4 / 2;
        r0 = s_d ? rlen : 0;
    }
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int r = 0; r < rounds; r++) {
        for (size_t i = rt; i < rlen; i += rn) {
            float4 v = ring[r0 + i];
            v.x += 1.f;
            ring[r0 + i] = v;
        }
        const float4 *sp = src + (size_t)r * stream_v4;
        float4 *dp = dst + (size_t)r * stream_v4;
        for (size_t i = tid; i < stream_v4; i += nth) {
            float4 v;
            asm volatile("ld.global.cs.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(sp + i));
            acc.x += v.x;
            asm volatile("st.global.cs.v4.f32 [%0], {%1,%2,%3,%4};" ::"l"(dp + i), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
        }
    }
    if (acc.x == 123.456f) dst[0] = acc;
}

void run_die_tests(int sms)
{
    const int nlines = 8, stride_words = 4096 * 4 + 512, iters = 64;
    unsigned *buf, *out;
    CK(cudaMalloc(&buf, (size_t)nlines * stride_words * 4 + 4096));
    CK(cudaMemset(buf, 0, (size_t)nlines * stride_words * 4 + 4096));
    CK(cudaMalloc(&out, (size_t)sms * nlines * 4));
    CK(cudaFuncSetAttribute(die_probe, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));   // one CTA per SM
    for (int pass = 0; pass < 2; pass++) {
        die_probe<<<sms, 32, 200 * 1024>>>(buf, nlines, stride_words, iters, out);
        CK(cudaDeviceSynchronize());
    }
    std::vector<unsigned> h((size_t)sms * nlines);
    CK(cudaMemcpy(h.data(), out, h.size() * 4, cudaMemcpyDeviceToHost));
    std::vector<int> die(sms, 0);
    int n1 = 0;
    for (int l = 0; l < 2; l++) {                          // classes by the largest gap of the sorted latencies of a line
        std::vector<unsigned> v(sms);
        for (int s = 0; s < sms; s++) v[s] = h[(size_t)s * nlines + l];
        std::vector<unsigned> srt = v;
        for (int i = 1; i < sms; i++)
            for (int j = i; j > 0 && srt[j] < srt[j - 1]; j--) std::swap(srt[j], srt[j - 1]);
        int cut = sms / 4;
        unsigned gap = 0;
        for (int i = sms / 4; i < 3 * sms / 4; i++)
            if (srt[i] - srt[i - 1] > gap) gap = srt[i] - srt[i - 1], cut = i;
        const unsigned thr = (srt[cut] + srt[cut - 1]) / 2;
        int far = 0;
        for (int s = 0; s < sms; s++) far += v[s] > thr;
        printf("die probe, line %d: near class %5.1f .. %5.1f clk per load, far class %5.1f .. %5.1f; %d SMs near, %d far\n", l,
               srt[0] / (float)iters, srt[cut - 1] / (float)iters, srt[cut] / (float)iters, srt[sms - 1] / (float)iters, sms - far, far);
        if (l == 0) {
            for (int s = 0; s < sms; s++) die[s] = v[s] > thr, n1 += die[s];
        }
    }
    printf("SM -> die map from line 0 (smid order, 0 = near): ");
    for (int s = 0; s < sms; s++) printf("%d", die[s]);
    printf("\n");
    int *d_die, *d_ticket;
    CK(cudaMalloc(&d_die, sms * 4));
    CK(cudaMalloc(&d_ticket, 8));
    CK(cudaMemcpy(d_die, die.data(), sms * 4, cudaMemcpyHostToDevice));
    const int cps = 2, smem = 100 * 1024, rounds = 16;     // exactly two CTAs per SM
    CK(cudaFuncSetAttribute(ring_by_die, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    for (size_t ring_mib : {16, 32, 48, 64}) {
        const size_t ring_v4 = ring_mib << 16, stream_v4 = ring_v4;
        float4 *ring, *src, *dst;
        CK(cudaMalloc(&ring, ring_v4 * 16));
        CK(cudaMalloc(&src, stream_v4 * 16 * rounds));
        CK(cudaMalloc(&dst, stream_v4 * 16 * rounds));
        CK(cudaMemset(ring, 0, ring_v4 * 16));
        CK(cudaMemset(src, 0, stream_v4 * 16 * rounds));
        for (int split = 0; split < 2; split++) {
            cudaEvent_t e0, e1;
            CK(cudaEventCreate(&e0));
            CK(cudaEventCreate(&e1));
            CK(cudaMemset(d_ticket, 0, 8));
            ring_by_die<<<sms * cps, 512, smem>>>(ring, ring_v4, src, dst, stream_v4, 2, split, d_die, d_ticket, (sms - n1) * cps, n1 * cps);
            CK(cudaDeviceSynchronize());
            CK(cudaMemset(d_ticket, 0, 8));
            CK(cudaEventRecord(e0));
            ring_by_die<<<sms * cps, 512, smem>>>(ring, ring_v4, src, dst, stream_v4, rounds, split, d_die, d_ticket, (sms - n1) * cps, n1 * cps);
            CK(cudaEventRecord(e1));
            CK(cudaDeviceSynchronize());
            float ms = 0;
            CK(cudaEventElapsedTime(&ms, e0, e1));
            printf("L2 ring %2zu MiB %-28s rewritten between streams of its size: %7.3f ms; stream alone at 6.5 TB/s %6.3f ms\n", ring_mib,
                   split ? "as two die-private halves," : "shared by both dies,", ms, (double)stream_v4 * 16 * 2 * rounds / 6.5e9);
        }
        CK(cudaFree(ring));
        CK(cudaFree(src));
        CK(cudaFree(dst));
    }
    CK(cudaFree(buf));
    CK(cudaFree(out));
    CK(cudaFree(d_die));
    CK(cudaFree(d_ticket));
}

int main()
{
    cudaDeviceProp prop;
    CK(cudaGetDeviceProperties(&prop, 0));
    const int sms = prop.multiProcessorCount;
    printf("device %s SMs %d L2 %d MB persisting-L2 max %d MB\n", prop.name, sms, prop.l2CacheSize >> 20, prop.persistingL2CacheMaxSize >> 20);
    float *d_out;
    CK(cudaMalloc(&d_out, 256));

    for (int cs : {1, 2, 4, 8, 16}) {
        run_dsmem<1, 0>(cs, sms, d_out, "4 B, random word anywhere in the cluster");
        run_dsmem<4, 0>(cs, sms, d_out, "16 B, random float4 anywhere in the cluster");
        run_dsmem<1, 1>(cs, sms, d_out, "4 B, lane stride 9 words, random CTA per warp");
        if (cs == 1 || cs == 8) run_dsmem<1, 2>(cs, sms, d_out, "4 B, lane stride 9 words, OWN CTA (baseline)");
    }

    for (size_t mib : {8, 32}) {
        const size_t words = mib << 18;
        float *d_buf;
        CK(cudaMalloc(&d_buf, words * 4));
        CK(cudaMemset(d_buf, 0, words * 4));
        run_scattered<0, 0>(d_buf, words, sms, d_out, "1 word/sector, via L1 (ld.nc)");
        run_scattered<0, 1>(d_buf, words, sms, d_out, "word + right neighbour, via L1");
        run_scattered<1, 0>(d_buf, words, sms, d_out, "1 word/sector, L2 only (.cg)");
        run_scattered<1, 1>(d_buf, words, sms, d_out, "word + right neighbour, .cg");
        CK(cudaFree(d_buf));
    }

    {
        const int rounds = 16;
        for (size_t ring_mib : {8, 16, 24, 32, 48, 64}) {
            for (int ratio : {1, 3}) {
                const size_t ring_v4 = ring_mib << 16, stream_v4 = ring_v4 * ratio;
                float4 *ring, *src, *dst;
                CK(cudaMalloc(&ring, ring_v4 * 16));
                CK(cudaMalloc(&src, stream_v4 * 16 * rounds));
                CK(cudaMalloc(&dst, stream_v4 * 16 * rounds));
                CK(cudaMemset(ring, 0, ring_v4 * 16));
                CK(cudaMemset(src, 0, stream_v4 * 16 * rounds));
                cudaEvent_t e0, e1;
                CK(cudaEventCreate(&e0));
                CK(cudaEventCreate(&e1));
                ring_and_stream<<<sms * 4, 512>>>(ring, ring_v4, src, dst, stream_v4, 2);
                CK(cudaDeviceSynchronize());
                CK(cudaEventRecord(e0));
                ring_and_stream<<<sms * 4, 512>>>(ring, ring_v4, src, dst, stream_v4, rounds);
                CK(cudaEventRecord(e1));
                CK(cudaDeviceSynchronize());
                float ms = 0;
                CK(cudaEventElapsedTime(&ms, e0, e1));
                const double stream_bytes = (double)stream_v4 * 16 * 2 * rounds, ring_bytes = (double)ring_v4 * 16 * 2 * rounds;
                printf("L2 ring %2zu MiB rewritten between streams of %dx its size: %7.3f ms; stream alone at 6.5 TB/s would take %6.3f ms; "
                       "if the ring went through HBM too: %6.3f ms\n",
                       ring_mib, ratio, ms, stream_bytes / 6.5e9, (stream_bytes + ring_bytes) / 6.5e9);
                CK(cudaFree(ring));
                CK(cudaFree(src));
                CK(cudaFree(dst));
            }
        }
    }
    run_die_tests(sms);
    printf("done\n");
    return 0;
}
