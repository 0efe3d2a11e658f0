// rcg_phase2.cuh -- device tables of one class (GDev) and the table-driven Phase-2 node interpreter,
// shared by the global tier (tier_global.cu) and the generated block-tier kernels.
// Phase 2 = HRR of Eq. (3) with the stepwise Cartesian->spherical transform of
// Eqs. (11)-(16), as level-sorted node programs (gen/emit_global.py).
#ifndef RCG_PHASE2_CUH
#define RCG_PHASE2_CUH
#include "rcg_internal.h"

struct GDev {                 // device copies of one class's tables
    const uint32_t *vrr_fam; const int32_t *lvl_off; const int32_t *tslots; const int32_t *tindex; const int32_t *tgt_off;
    const uint32_t *bra_ops; const uint32_t *ket_ops;
    const uint16_t *bra_out; const uint16_t *ket_out;
    const double *consts;
    int n_fam, n_levels, n_targets, nA, nC, n_vslots;
    const int32_t *bra_noff, *bra_loff, *ket_noff, *ket_loff;
    int n_bra_levels, bra_nin, bra_nslots, bra_nout;
    int n_ket_levels, ket_nin, ket_nslots, ket_nout;
    int p2_slots, n_consts;       // shared-memory doubles per warp for Phase 2 (coefficients + vector)
    int L;
    int64_t slots_per_warp;
};

// Phase-2 node program executed by the whole warp on one vector held in shared memory `loc`:
// the nodes of a level (dst <- sum_k coef_k * src_k) are independent and are spread over the lanes.
__device__ __forceinline__ void run_nodes(const uint32_t *__restrict__ words, const int32_t *__restrict__ noff,
                                          const int32_t *__restrict__ loff, int nlev, const double *__restrict__ consts,
                                          double *loc, const double *__restrict__ cf, int lane)
{
    for (int lv = 0; lv < nlev; ++lv) {
        __syncwarp();
        const int ne = __ldg(loff + lv + 1);
        for (int n = __ldg(loff + lv) + lane; n < ne; n += 32) {
            const uint32_t *w = words + __ldg(noff + n);
            const uint32_t h = __ldg(w);
            const int dst = h & 0xffff, nt = h >> 16;
            double v = 0.0;
#pragma unroll 2
            for (int k = 1; k <= nt; ++k) {
                const uint32_t t = __ldg(w + k);
                v = fma(cf[t >> 16], loc[t & 0xffff], v);       // cf: 1, X_x, X_y, X_z, constants (shared memory)
            }
            loc[dst] = v;
        }
    }
    __syncwarp();
}


// Phase 2 of one quartet by a whole block (block tier): H [nA][nC] (contracted Cartesian targets) and the
// half-transformed Bh [bra_nout][nC] live in shared memory; each warp takes ket columns (bra side:
// HRR + Ta,Tb) and then spherical bra rows (ket side: HRR + Tc,Td) round-robin and runs the node programs
// on its own vector `loc`; results go to `out` in the caller's index order.  wbuf: per-warp p2_slots doubles.
__device__ __forceinline__ void rcg_phase2_block(const GDev &g, const RcgLaunch &a, int64_t q, const double *Hs,
                                                 double *Bh, double *wbuf, const double *AB, const double *CD,
                                                 int warp, int lane, int nwarps)
{
    double *cf = wbuf + warp * g.p2_slots;
    double *loc = cf + 4 + g.n_consts;
    for (int k = lane; k < g.n_consts; k += 32) cf[4 + k] = __ldg(g.consts + k);
    if (lane == 0) { cf[0] = 1.0; cf[1] = AB[0]; cf[2] = AB[1]; cf[3] = AB[2]; }
    for (int c = warp; c < g.nC; c += nwarps) {
        __syncwarp();
        for (int k = lane; k < g.nA; k += 32) loc[k] = Hs[k * g.nC + c];
        run_nodes(g.bra_ops, g.bra_noff, g.bra_loff, g.n_bra_levels, g.consts, loc, cf, lane);
        for (int o = lane; o < g.bra_nout; o += 32) Bh[o * g.nC + c] = loc[__ldg(g.bra_out + o)];
    }
    __syncthreads();
    if (lane == 0) { cf[1] = CD[0]; cf[2] = CD[1]; cf[3] = CD[2]; }
    double *out = a.out + q * a.out_stride;
    const int nsb = a.nsph[1], nsd = a.nsph[3];
    for (int o = warp; o < g.bra_nout; o += nwarps) {
        __syncwarp();
        for (int k = lane; k < g.nC; k += 32) loc[k] = Bh[o * g.nC + k];
        run_nodes(g.ket_ops, g.ket_noff, g.ket_loff, g.n_ket_levels, g.consts, loc, cf, lane);
        const int64_t obase = (int64_t)(o / nsb) * a.ostride[0] + (int64_t)(o % nsb) * a.ostride[1];
        for (int r = lane; r < g.ket_nout; r += 32)
            out[obase + (int64_t)(r / nsd) * a.ostride[2] + (int64_t)(r % nsd) * a.ostride[3]] = loc[__ldg(g.ket_out + r)];
    }
}

// tier_global.cu: device copies of a class's tables (uploaded on first use, cached per device)
cudaError_t rcg_global_tables(const RcgClassDesc &d, GDev *out);

#endif
