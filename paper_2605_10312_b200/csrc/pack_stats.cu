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

cudaError_t rcg_pack_stats(const RcgLaunch &a, int Q, const unsigned long long **stat)
{
    if (!a.stat_pool || !a.stat_next) return cudaErrorInvalidValue;
    const unsigned slot = (*a.stat_next)++ % (RCG_STAT_POOL / 2);
    unsigned long long *s = a.stat_pool + 2 * slot;
    cudaError_t e = cudaMemsetAsync(s, 0, 2 * sizeof(unsigned long long), a.stream);
    if (e != cudaSuccess) return e;
    const int64_t ngroups = (a.n + Q - 1) / Q;
    int blocks = (int)((ngroups + 255) / 256);
    if (blocks > 1184) blocks = 1184;
    rcg_pack_stats_kernel<<<blocks, 256, 0, a.stream>>>(a.basis, a.quartets, a.n, a.perm[0], a.perm[1], a.perm[2], a.perm[3], Q, s);
    *stat = s;
    return cudaGetLastError();
}
