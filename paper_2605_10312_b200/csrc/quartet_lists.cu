// quartet_lists.cu -- device-side helpers of the screened pass (BASELINE.json configs 3 and 5:
// "all unique quartets with Schwarz bound > 1e-10, batched by angular class"; reading R-SCHWARZ):
//   rcg_schwarz_from_blocks : Q_ab = sqrt(max_k |(ab|ab)[k][k]|) from the (ab|ab) blocks rcg_eri_batch wrote
//   rcg_quartets_from_pairs : the quartet list of a range of bra pairs against the surviving prefix of a
//                             Q-sorted ket pair list, written straight into the list rcg_eri_batch reads
// List logic only; the integrals come from the class kernels.
#include "../../include/rcg.h"
#include "rcg_internal.h"

__global__ void rcg_schwarz_kernel(const double *__restrict__ blocks, int64_t n, int dim, double *__restrict__ Q)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double *b = blocks + i * (int64_t)dim * dim;
    double m = 0.0;
    for (int k = 0; k < dim; ++k) m = fmax(m, fabs(b[(int64_t)k * dim + k]));
    Q[i] = sqrt(m);
}

extern "C" rcg_status rcg_schwarz_from_blocks(const double *blocks, int64_t n, int dim, double *Q, void *stream)
{
    if (n < 0 || dim <= 0) return RCG_ERR_INVALID_ARG;
    if (n == 0) return RCG_OK;
    if (!blocks || !Q) return RCG_ERR_INVALID_ARG;
    rcg_schwarz_kernel<<<(unsigned)((n + 127) / 128), 128, 0, (cudaStream_t)stream>>>(blocks, n, dim, Q);
    { const cudaError_t le = cudaGetLastError(); return le == cudaSuccess ? RCG_OK : rcg_cuda_fail(le); }
}

// one block per bra pair i: rows offs[i]-offs[i0] .. offs[i+1]-offs[i0] of the list
__global__ void rcg_quartets_kernel(const int2 *__restrict__ bra, const int2 *__restrict__ ket,
                                    const int64_t *__restrict__ offs, int64_t i0, int64_t i1, int4 *__restrict__ q)
{
    const int64_t base = offs[i0];
    for (int64_t i = i0 + blockIdx.x; i < i1; i += gridDim.x) {
        const int64_t o = offs[i] - base, cnt = offs[i + 1] - offs[i];
        const int2 ab = bra[i];
        for (int64_t j = threadIdx.x; j < cnt; j += blockDim.x) {
            const int2 cd = ket[j];
            q[o + j] = make_int4(ab.x, ab.y, cd.x, cd.y);
        }
    }
}

extern "C" rcg_status rcg_quartets_from_pairs(const int32_t *bra_pairs, const int32_t *ket_pairs, const int64_t *offs,
                                              int64_t i0, int64_t i1, int32_t *quartets, void *stream)
{
    if (i0 < 0 || i1 < i0) return RCG_ERR_INVALID_ARG;
    if (i1 == i0) return RCG_OK;
    if (!bra_pairs || !ket_pairs || !offs || !quartets || ((uintptr_t)quartets & 15) != 0 ||
        ((uintptr_t)bra_pairs & 7) != 0 || ((uintptr_t)ket_pairs & 7) != 0)
        return RCG_ERR_INVALID_ARG;
    int64_t blocks = i1 - i0;
    if (blocks > 65535 * 16) blocks = 65535 * 16;
    rcg_quartets_kernel<<<(unsigned)blocks, 128, 0, (cudaStream_t)stream>>>((const int2 *)bra_pairs, (const int2 *)ket_pairs,
                                                                          offs, i0, i1, (int4 *)quartets);
    { const cudaError_t le = cudaGetLastError(); return le == cudaSuccess ? RCG_OK : rcg_cuda_fail(le); }
}
