// pack_stats.cu -- statistics pass for the packed warp-tier kernels: how much primitive work the
// grouping "Q consecutive quartets share a warp and loop to their largest K4" wastes on a given list.
// stat[0] = sum over groups of Q * max K4, stat[1] = sum of K4.  The class kernels read it on the
// device (emit_warp.py), so the choice costs no host synchronisation.
#include "rcg_internal.h"

__global__ void rcg_pack_stats_kernel(RcgBasisDev b, const int32_t *quartets, int64_t n, int p0, int p1, int p2, int p3,
                                      int Q, unsigned long long *stat)
{
    const int64_t ngroups = (n + Q - 1) / Q;
    unsigned long long padded = 0, real = 0;
    for (int64_t g = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; g < ngroups; g += (int64_t)gridDim.x * blockDim.x) {
        int kmax = 0;
        for (int j = 0; j < Q; ++j) {
            const int64_t q = g * Q + j < n ? g * Q + j : n - 1;
            const int s0 = quartets[4 * q + p0], s1 = quartets[4 * q + p1], s2 = quartets[4 * q + p2], s3 = quartets[4 * q + p3];
            const int k4 = (b.prim_off[s0 + 1] - b.prim_off[s0]) * (b.prim_off[s1 + 1] - b.prim_off[s1]) *
                           (b.prim_off[s2 + 1] - b.prim_off[s2]) * (b.prim_off[s3 + 1] - b.prim_off[s3]);
            kmax = k4 > kmax ? k4 : kmax;
            if (g * Q + j < n) real += k4;
        }
        padded += (unsigned long long)kmax * Q;
    }
    for (int o = 16; o > 0; o >>= 1) {
        padded += __shfl_down_sync(0xffffffffu, padded, o);
        real += __shfl_down_sync(0xffffffffu, real, o);
    }
    if ((threadIdx.x & 31) == 0) {
        atomicAdd(stat, padded);
        atomicAdd(stat + 1, real);
    }
}

cudaError_t rcg_pack_stats(const RcgLaunch &a, int Q, int which, const unsigned long long **stat)
{
    RcgStatHolder *h = a.stat_holder;
    if (!h) return cudaErrorInvalidValue;
    cudaError_t e;
    if (!h->words) {
        void *p = nullptr;
        if ((e = rcg_pool_alloc(&p, 4 * sizeof(unsigned long long), a.stream)) != cudaSuccess) return e;
        h->words = (unsigned long long *)p;
        h->stream = a.stream;
    }
    unsigned long long *s = h->words + 2 * (which ? 1 : 0);
    if ((e = cudaMemsetAsync(s, 0, 2 * sizeof(unsigned long long), a.stream)) != cudaSuccess) return e;
    int nsm = 0;
    if ((e = rcg_sm_count(&nsm)) != cudaSuccess) return e;
    const int64_t ngroups = (a.n + Q - 1) / Q;
    int blocks = (int)((ngroups + 255) / 256);
    if (blocks > 8 * nsm) blocks = 8 * nsm;
    rcg_pack_stats_kernel<<<blocks, 256, 0, a.stream>>>(a.basis, a.quartets, a.n, a.perm[0], a.perm[1], a.perm[2], a.perm[3], Q, s);
    *stat = s;
    return cudaGetLastError();
}

cudaError_t rcg_stat_release(RcgStatHolder &h)
{
    if (!h.words) return cudaSuccess;
    cudaError_t e = cudaFreeAsync(h.words, h.stream);      // stream-ordered: after every kernel of this call that reads it
    h.words = nullptr;
    return e;
}

// ---------------------------------------------------------------- per-device facts
static std::atomic<int> sm_count_of[64];

cudaError_t rcg_sm_count(int *nsm)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    int n = sm_count_of[dev & 63].load(std::memory_order_relaxed);
    if (n == 0) {
        if ((e = cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
        sm_count_of[dev & 63].store(n, std::memory_order_relaxed);
    }
    *nsm = n;
    return cudaSuccess;
}

cudaError_t rcg_prepare_kernel(RcgOnce &once, const void *func, size_t smem_bytes, int *nsm)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    const unsigned long long bit = 1ull << (dev & 63);
    if (!(once.done.load(std::memory_order_acquire) & bit)) {
        if (smem_bytes > 48 * 1024 &&
            (e = cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes)) != cudaSuccess) return e;
        once.done.fetch_or(bit, std::memory_order_release);
    }
    return nsm ? rcg_sm_count(nsm) : cudaSuccess;
}
