// jk_digest.cu -- SURVEY 8(f) NEXT-1: digestion of a batch of integrals into the Coulomb and exchange
// matrices, J_mn = sum_ls D_ls (mn|ls), K_mn = sum_ls D_ls (ml|ns)  ("J/K contraction",
// :291 "8-fold symmetry via scale factors", Alg. 2 line 10 at :283).  A separate kernel that reads the block
// rcg_eri_batch wrote (the paper's buffered "_jk_transform" form), not yet fused into the class
// kernels.  Each listed quartet (ab|cd) stands for its whole 8-fold orbit; with w = 1/2 for a == b, 1/2 for
// c == d, 1/2 for (a,b) == (c,d) (the scale factors) and a SYMMETRIC density,
//   Jt_ab += 2 w sum_cd D_cd I    Jt_cd += 2 w sum_ab D_ab I
//   Kt_ac += w sum_bd D_bd I      Kt_bc += w sum_ad D_ad I      Kt_ad += w sum_bc D_bc I      Kt_bd += w sum_ac D_ac I
// and J = Jt + Jt^T, K = Kt + Kt^T (rcg_jk_finish): the four permutations that swap bra and ket are the
// transposes of the four that do not.
#include "rcg_internal.h"

#define JK_WARPS 8

// one GROUP of G lanes per quartet (G = 4, 8, 16 or 32 by the size of the block, so that light classes do not
// leave most of a warp idle); the block of integrals and the six density blocks are staged in shared memory.  A
// group takes a CONTIGUOUS chunk of the list: consecutive quartets of a screened pass share the bra pair, so
// Jt_ab is accumulated in registers and written when the pair changes (otherwise every group would hammer the
// same entries).
// NA..ND > 0: block dimensions known at compile time (the 55 canonical classes with l <= 3: the index arithmetic
// of the generic version -- integer divisions by run-time dimensions -- was most of its instruction count);
// NA == 0: run-time dimensions (any other order or l = 4).
template <int NA, int NB, int NC, int ND>
__global__ void __launch_bounds__(JK_WARPS * 32) rcg_jk_digest_kernel(const int32_t *__restrict__ quartets,
                                                                      int64_t n, const double *__restrict__ I,
                                                                      const int32_t *__restrict__ bf_off,
                                                                      const double *__restrict__ D, double *Jt, double *Kt,
                                                                      int nbf, int rna, int rnb, int rnc, int rnd, int64_t chunk, int G, int dstride)
{
    const int na = NA ? NA : rna, nb = NA ? NB : rnb, nc = NA ? NC : rnc, nd = NA ? ND : rnd;
    extern __shared__ double sm[];
    const int lane = threadIdx.x % G, grp = threadIdx.x / G;          // lane within the group, group within the block
    const int nab = na * nb, ncd = nc * nd, nblk = nab * ncd;
    double *blk = sm + grp * (nblk + 6 * dstride);
    double *Dcd = blk + nblk, *Dab = Dcd + dstride, *Dbd = Dab + dstride, *Dad = Dbd + dstride, *Dbc = Dad + dstride, *Dac = Dbc + dstride;
    const int64_t gw = (int64_t)blockIdx.x * (blockDim.x / G) + grp;
    const int64_t q0 = gw * chunk, q1 = min(n, q0 + chunk);
    double jab[3] = {0.0, 0.0, 0.0};            // Jt_ab partial sums of this lane: elements lane, lane+G, lane+2G (nab <= 3G)
    int pa = -1, pb = -1, poa = 0, pob = 0;
    const unsigned gmask = G == 32 ? 0xffffffffu : (((1u << G) - 1u) << ((threadIdx.x & 31) / G * G));   // the group's lanes
    for (int64_t q = q0; q < q1; ++q) {
        const int sa = quartets[4 * q], sb = quartets[4 * q + 1], sc = quartets[4 * q + 2], sd = quartets[4 * q + 3];
        const int oa = bf_off[sa], ob = bf_off[sb], oc = bf_off[sc], od = bf_off[sd];
        if (sa != pa || sb != pb) {             // bra pair changed: flush Jt_ab
            if (pa >= 0)
            {
#pragma unroll
                for (int k = 0; k < 3; ++k) {
                    const int e = lane + G * k;
                    if (e < nab) atomicAdd(Jt + (int64_t)(poa + e / nb) * nbf + pob + e % nb, jab[k]);
                    jab[k] = 0.0;
                }
            }
            pa = sa; pb = sb; poa = oa; pob = ob;
        }
        double w = 1.0;
        if (sa == sb) w *= 0.5;
        if (sc == sd) w *= 0.5;
        if (sa == sc && sb == sd) w *= 0.5;
        __syncwarp(gmask);
        const double *Iq = I + q * (int64_t)nblk;
        for (int e = lane; e < nblk; e += G) blk[e] = Iq[e];
        for (int e = lane; e < ncd; e += G) Dcd[e] = D[(int64_t)(oc + e / nd) * nbf + od + e % nd];
        for (int e = lane; e < nab; e += G) Dab[e] = D[(int64_t)(oa + e / nb) * nbf + ob + e % nb];
        for (int e = lane; e < nb * nd; e += G) Dbd[e] = D[(int64_t)(ob + e / nd) * nbf + od + e % nd];
        for (int e = lane; e < na * nd; e += G) Dad[e] = D[(int64_t)(oa + e / nd) * nbf + od + e % nd];
        for (int e = lane; e < nb * nc; e += G) Dbc[e] = D[(int64_t)(ob + e / nc) * nbf + oc + e % nc];
        for (int e = lane; e < na * nc; e += G) Dac[e] = D[(int64_t)(oa + e / nc) * nbf + oc + e % nc];
        __syncwarp(gmask);
        // Jt_ab (kept in registers), Jt_cd
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const int e = lane + G * k;
            if (e < nab) {
                double s = 0.0;
                for (int t = 0; t < ncd; ++t) s = fma(Dcd[t], blk[e * ncd + t], s);
                jab[k] = fma(2.0 * w, s, jab[k]);
            }
        }
        for (int e = lane; e < ncd; e += G) {
            double s = 0.0;
            for (int t = 0; t < nab; ++t) s = fma(Dab[t], blk[t * ncd + e], s);
            atomicAdd(Jt + (int64_t)(oc + e / nd) * nbf + od + e % nd, 2.0 * w * s);
        }
        // Kt_ac, Kt_ad, Kt_bc, Kt_bd
        for (int e = lane; e < na * nc; e += G) {
            const int ia = e / nc, ic = e % nc;
            double s = 0.0;
            for (int ib = 0; ib < nb; ++ib)
                for (int id = 0; id < nd; ++id) s = fma(Dbd[ib * nd + id], blk[((ia * nb + ib) * nc + ic) * nd + id], s);
            atomicAdd(Kt + (int64_t)(oa + ia) * nbf + oc + ic, w * s);
        }
        for (int e = lane; e < na * nd; e += G) {
            const int ia = e / nd, id = e % nd;
            double s = 0.0;
            for (int ib = 0; ib < nb; ++ib)
                for (int ic = 0; ic < nc; ++ic) s = fma(Dbc[ib * nc + ic], blk[((ia * nb + ib) * nc + ic) * nd + id], s);
            atomicAdd(Kt + (int64_t)(oa + ia) * nbf + od + id, w * s);
        }
        for (int e = lane; e < nb * nc; e += G) {
            const int ib = e / nc, ic = e % nc;
            double s = 0.0;
            for (int ia = 0; ia < na; ++ia)
                for (int id = 0; id < nd; ++id) s = fma(Dad[ia * nd + id], blk[((ia * nb + ib) * nc + ic) * nd + id], s);
            atomicAdd(Kt + (int64_t)(ob + ib) * nbf + oc + ic, w * s);
        }
        for (int e = lane; e < nb * nd; e += G) {
            const int ib = e / nd, id = e % nd;
            double s = 0.0;
            for (int ia = 0; ia < na; ++ia)
                for (int ic = 0; ic < nc; ++ic) s = fma(Dac[ia * nc + ic], blk[((ia * nb + ib) * nc + ic) * nd + id], s);
            atomicAdd(Kt + (int64_t)(ob + ib) * nbf + od + id, w * s);
        }
    }
    if (pa >= 0) {
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const int e = lane + G * k;
            if (e < nab) atomicAdd(Jt + (int64_t)(poa + e / nb) * nbf + pob + e % nb, jab[k]);
        }
    }
}

extern "C" rcg_status rcg_jk_digest(int la, int lb, int lc, int ld, const int32_t *quartets,
                                    int64_t nquartet, const double *integrals, const int32_t *shell_bf_offset,
                                    const double *D, double *Jt, double *Kt, int nbf, void *stream)
{
    if (nquartet < 0 || nbf <= 0) return RCG_ERR_INVALID_ARG;
    if (la < 0 || lb < 0 || lc < 0 || ld < 0 || la > RCG_LMAX || lb > RCG_LMAX || lc > RCG_LMAX || ld > RCG_LMAX) return RCG_ERR_INVALID_ARG;
    if (nquartet == 0) return RCG_OK;
    if (!quartets || !integrals || !shell_bf_offset || !D || !Jt || !Kt) return RCG_ERR_INVALID_ARG;
    const int na = 2 * la + 1, nb = 2 * lb + 1, nc = 2 * lc + 1, nd = 2 * ld + 1;
    const int nblk = na * nb * nc * nd;
    int G = nblk > 64 ? 32 : (nblk > 27 ? 16 : (nblk > 9 ? 8 : 4));             // lanes per quartet ...
    while (3 * G < na * nb) G *= 2;                                               // ... at least nab / 3 (three Jt_ab registers per lane)
    int dstride = na * nb;                                                        // largest of the six density blocks
    { const int c[5] = {nc * nd, nb * nd, na * nd, nb * nc, na * nc}; for (int k = 0; k < 5; ++k) if (c[k] > dstride) dstride = c[k]; }
    // groups per block: JK_WARPS warps' worth, fewer where the staged blocks would not fit the 227 KB of an SM
    // ((gg|gg): 7,047 doubles per group -> 4 groups of 32 lanes)
    int groups = JK_WARPS * 32 / G;
    const size_t per_group = sizeof(double) * ((size_t)nblk + 6 * dstride);
    while (groups > 1 && groups * per_group > 220 * 1024) groups /= 2;
    if (per_group > 220 * 1024) return RCG_ERR_UNSUPPORTED_CLASS;
    const size_t smem = groups * per_group;
    int nsm = 0;
    cudaError_t e = rcg_sm_count(&nsm);
    if (e != cudaSuccess) return rcg_cuda_fail(e);
    // contiguous chunks: enough warps to fill the GPU several times over, chunks of at least 8 quartets
    int64_t ngroups = (int64_t)nsm * groups * 8;
    int64_t chunk = (nquartet + ngroups - 1) / ngroups;
    if (chunk < 8) chunk = 8;
    ngroups = (nquartet + chunk - 1) / chunk;
    const int64_t blocks = (ngroups + groups - 1) / groups;
#define JK_LAUNCH(A, B_, C, D_)                                                                                         \
    do {                                                                                                                \
        static RcgOnce once;                                                                                            \
        e = rcg_prepare_kernel(once, (const void *)rcg_jk_digest_kernel<A, B_, C, D_>, 220 * 1024, nullptr);            \
        if (e == cudaSuccess)                                                                                           \
            rcg_jk_digest_kernel<A, B_, C, D_><<<(unsigned)blocks, groups * G, smem, (cudaStream_t)stream>>>(           \
                quartets, nquartet, integrals, shell_bf_offset, D, Jt, Kt, nbf, na, nb, nc, nd, chunk, G, dstride);     \
    } while (0)
#define JK_CASE(LA, LB, LC, LD) case ((LA) * 64 + (LB) * 16 + (LC) * 4 + (LD)): JK_LAUNCH(2 * LA + 1, 2 * LB + 1, 2 * LC + 1, 2 * LD + 1); break;
    const bool canonical = la <= 3 && la >= lb && lc >= ld && (la > lc || (la == lc && lb >= ld));
    if (!canonical) JK_LAUNCH(0, 0, 0, 0);
    else switch (la * 64 + lb * 16 + lc * 4 + ld) {
        JK_CASE(0,0,0,0)
        JK_CASE(1,0,0,0) JK_CASE(1,0,1,0)
        JK_CASE(1,1,0,0) JK_CASE(1,1,1,0) JK_CASE(1,1,1,1)
        JK_CASE(2,0,0,0) JK_CASE(2,0,1,0) JK_CASE(2,0,1,1) JK_CASE(2,0,2,0)
        JK_CASE(2,1,0,0) JK_CASE(2,1,1,0) JK_CASE(2,1,1,1) JK_CASE(2,1,2,0) JK_CASE(2,1,2,1)
        JK_CASE(2,2,0,0) JK_CASE(2,2,1,0) JK_CASE(2,2,1,1) JK_CASE(2,2,2,0) JK_CASE(2,2,2,1) JK_CASE(2,2,2,2)
        JK_CASE(3,0,0,0) JK_CASE(3,0,1,0) JK_CASE(3,0,1,1) JK_CASE(3,0,2,0) JK_CASE(3,0,2,1) JK_CASE(3,0,2,2) JK_CASE(3,0,3,0)
        JK_CASE(3,1,0,0) JK_CASE(3,1,1,0) JK_CASE(3,1,1,1) JK_CASE(3,1,2,0) JK_CASE(3,1,2,1) JK_CASE(3,1,2,2) JK_CASE(3,1,3,0) JK_CASE(3,1,3,1)
        JK_CASE(3,2,0,0) JK_CASE(3,2,1,0) JK_CASE(3,2,1,1) JK_CASE(3,2,2,0) JK_CASE(3,2,2,1) JK_CASE(3,2,2,2) JK_CASE(3,2,3,0) JK_CASE(3,2,3,1) JK_CASE(3,2,3,2)
        JK_CASE(3,3,0,0) JK_CASE(3,3,1,0) JK_CASE(3,3,1,1) JK_CASE(3,3,2,0) JK_CASE(3,3,2,1) JK_CASE(3,3,2,2) JK_CASE(3,3,3,0) JK_CASE(3,3,3,1) JK_CASE(3,3,3,2) JK_CASE(3,3,3,3)
        default: JK_LAUNCH(0, 0, 0, 0);
    }
#undef JK_CASE
#undef JK_LAUNCH
    if (e == cudaSuccess) e = cudaGetLastError();
    return e == cudaSuccess ? RCG_OK : rcg_cuda_fail(e);
}

__global__ void rcg_jk_finish_kernel(double *M, int n)
{
    // M <- M + M^T, one thread per (i <= j)
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (int64_t)n * n) return;
    const int i = (int)(t / n), j = (int)(t % n);
    if (i > j) return;
    const double s = M[(int64_t)i * n + j] + M[(int64_t)j * n + i];
    M[(int64_t)i * n + j] = s;
    M[(int64_t)j * n + i] = s;
}

extern "C" rcg_status rcg_jk_finish(double *Jt, double *Kt, int nbf, void *stream)
{
    if (nbf <= 0 || !Jt || !Kt) return RCG_ERR_INVALID_ARG;
    const int64_t tot = (int64_t)nbf * nbf;
    rcg_jk_finish_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, (cudaStream_t)stream>>>(Jt, nbf);
    rcg_jk_finish_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, (cudaStream_t)stream>>>(Kt, nbf);
    const cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? RCG_OK : rcg_cuda_fail(e);
}
