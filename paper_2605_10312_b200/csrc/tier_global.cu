// tier_global.cu -- RCG_TIER_GLOBAL: table-driven kernel, one WARP per shell quartet, every
// intermediate in a global scratch region owned by the warp (the paper's Tier 2 keeps its
// accumulators in a packed global buffer; here the whole recurrence graph lives
// there because it is executed from tables instead of unrolled code -- unrolled (gg|gg) does not
// compile).  Works for every generated class; it is the only tier for the heaviest
// ones ((fd|..), (ff|..), (gg|gg)) and the independent cross-check for the warp tier.
// Steps per quartet follow Alg. 2: H <- 0; for each primitive quartet
// {pair quantities, Boys, VRR level by level (the families of one level |a|+|c| are independent and
// are spread over the 32 lanes), H += V}; bra HRR + Ta,Tb (lane = ket column); ket HRR + Tc,Td
// (lane = spherical bra row); store.
#include <mutex>
#include <map>
#include "rcg_device.cuh"
#include "rcg_phase2.cuh"

#define GW 4   // warps per block
__global__ void __launch_bounds__(GW * 32, 8) rcg_eri_global_kernel(GDev g, RcgLaunch a)
{
    const int lane = threadIdx.x & 31;
    const int64_t nwarps = (int64_t)gridDim.x * GW;
    const int64_t gw = (int64_t)blockIdx.x * GW + (threadIdx.x >> 5);
    double *V = a.workspace + gw * g.slots_per_warp;              // VRR slots
    double *H = V + g.n_vslots;                                   // [nA][nC] contracted targets
    double *Bh = H + g.n_targets;                                 // [bra_nout][nC] half-transformed
    extern __shared__ double p2smem[];
    double *cf = p2smem + (threadIdx.x >> 5) * g.p2_slots;        // Phase-2 coefficient table of this warp
    double *loc = cf + 4 + g.n_consts;                            // Phase-2 vector of this warp
    for (int k = lane; k < g.n_consts; k += 32) cf[4 + k] = __ldg(g.consts + k);
    if (lane == 0) cf[0] = 1.0;
    const RcgBasisDev &b = a.basis;
    for (int64_t q = gw; q < a.n; q += nwarps) {
        int sh[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) sh[k] = a.quartets[4 * q + a.perm[k]];
        double R[4][3];
#pragma unroll
        for (int k = 0; k < 4; ++k)
#pragma unroll
            for (int t = 0; t < 3; ++t) R[k][t] = b.centers[3 * sh[k] + t];
        for (int t = lane; t < g.n_targets; t += 32) H[t] = 0.0;
        const int p0 = b.prim_off[sh[0]], p0e = b.prim_off[sh[0] + 1];
        const int p1 = b.prim_off[sh[1]], p1e = b.prim_off[sh[1] + 1];
        const int p2 = b.prim_off[sh[2]], p2e = b.prim_off[sh[2] + 1];
        const int p3 = b.prim_off[sh[3]], p3e = b.prim_off[sh[3] + 1];
        for (int i = p0; i < p0e; ++i)
        for (int j = p1; j < p1e; ++j)
        for (int k = p2; k < p2e; ++k)
        for (int l = p3; l < p3e; ++l) {
            RcgPrim p;                                           // every lane: same primitive quartet
            rcg_prim_setup(p, R[0], R[1], R[2], R[3], b.exps[i], b.exps[j], b.exps[k], b.exps[l],
                           b.coefs[i] * b.coefs[j] * b.coefs[k] * b.coefs[l]);
            double F[17];
            rcg_boys<-1>(g.L, p.T, p.pref, b.boys, F);
            __syncwarp();                                        // previous primitive's H += V reads are done
            if (lane == 0)
                for (int m = 0; m <= g.L; ++m) V[m] = F[m];
            __syncwarp();
            for (int t = __ldg(g.tgt_off) + lane; t < __ldg(g.tgt_off + 1); t += 32)      // level-0 target (ss|ss)
                H[__ldg(g.tindex + t)] += V[__ldg(g.tslots + t)];
            for (int lv = 0; lv < g.n_levels; ++lv) {
                __syncwarp();
                const int fe = __ldg(g.lvl_off + lv + 1);
                for (int f = __ldg(g.lvl_off + lv) + lane; f < fe; f += 32) {
                    const uint32_t *w = g.vrr_fam + 5 * f;
                    const int od = __ldg(w), o1 = __ldg(w + 1), o3 = __ldg(w + 2), o5 = __ldg(w + 3);
                    const uint32_t meta = __ldg(w + 4);
                    const int mlo = meta & 31, nm = (meta >> 5) & 31, ket = (meta >> 10) & 1, ax = (meta >> 11) & 3;
                    const int n2 = (meta >> 13) & 15, nx = (meta >> 17) & 15;
                    const double c1 = ket ? p.QC[ax] : p.PA[ax];
                    const double c2 = ket ? p.WQ[ax] : p.WP[ax];
                    const double k3 = (double)n2 * (ket ? p.he : p.hz);
                    const double r3 = ket ? p.re : p.rz;
                    const double k5 = (double)nx * p.hze;
                    // four Boys orders at a time: all parent loads first (independent, in flight together;
                    // p1/p2 and p3/p4 share values across m), then the arithmetic, then the stores
                    for (int m0 = mlo; m0 < mlo + nm; m0 += 4) {
                        const int cntm = min(4, mlo + nm - m0);
                        double a1[5], a3[5], a5[4];
#pragma unroll
                        for (int k = 0; k < 5; ++k) a1[k] = k <= cntm ? V[o1 + m0 + k] : 0.0;
                        if (n2) {
#pragma unroll
                            for (int k = 0; k < 5; ++k) a3[k] = k <= cntm ? V[o3 + m0 + k] : 0.0;
                        }
                        if (nx) {
#pragma unroll
                            for (int k = 0; k < 4; ++k) a5[k] = k < cntm ? V[o5 + m0 + k + 1] : 0.0;
                        }
#pragma unroll
                        for (int k = 0; k < 4; ++k) {
                            if (k < cntm) {
                                double v = c1 * a1[k];
                                v = fma(c2, a1[k + 1], v);
                                if (n2) v = fma(k3, fma(-r3, a3[k + 1], a3[k]), v);
                                if (nx) v = fma(k5, a5[k], v);
                                V[od + m0 + k] = v;
                            }
                        }
                    }
                }
                // contraction (Alg. 2 line 7) of the targets of this level, before its buffer is reused
                __syncwarp();
                for (int t = __ldg(g.tgt_off + lv + 1) + lane; t < __ldg(g.tgt_off + lv + 2); t += 32)
                    H[__ldg(g.tindex + t)] += V[__ldg(g.tslots + t)];
            }
        }
        __syncwarp();
        // Phase 2, bra side: one ket column at a time, the column's HRR + Ta,Tb nodes spread over the lanes
        const double AB0 = R[0][0] - R[1][0], AB1 = R[0][1] - R[1][1], AB2 = R[0][2] - R[1][2];
        const double CD0 = R[2][0] - R[3][0], CD1 = R[2][1] - R[3][1], CD2 = R[2][2] - R[3][2];
        if (lane == 0) { cf[1] = AB0; cf[2] = AB1; cf[3] = AB2; }
        for (int c = 0; c < g.nC; ++c) {
            for (int k = lane; k < g.nA; k += 32) loc[k] = H[k * g.nC + c];
            run_nodes(g.bra_ops, g.bra_noff, g.bra_loff, g.n_bra_levels, g.consts, loc, cf, lane);
            for (int o = lane; o < g.bra_nout; o += 32) Bh[o * g.nC + c] = loc[__ldg(g.bra_out + o)];
            __syncwarp();
        }
        // ket side: one spherical bra row o = ia*nsph(lb)+ib at a time
        double *out = a.out + q * a.out_stride;
        const int nsb = a.nsph[1], nsd = a.nsph[3];
        if (lane == 0) { cf[1] = CD0; cf[2] = CD1; cf[3] = CD2; }
        for (int o = 0; o < g.bra_nout; ++o) {
            for (int k = lane; k < g.nC; k += 32) loc[k] = Bh[o * g.nC + k];
            run_nodes(g.ket_ops, g.ket_noff, g.ket_loff, g.n_ket_levels, g.consts, loc, cf, lane);
            const int64_t obase = (int64_t)(o / nsb) * a.ostride[0] + (int64_t)(o % nsb) * a.ostride[1];
            for (int r = lane; r < g.ket_nout; r += 32)
                out[obase + (int64_t)(r / nsd) * a.ostride[2] + (int64_t)(r % nsd) * a.ostride[3]] = loc[__ldg(g.ket_out + r)];
            __syncwarp();
        }
        __syncwarp();
    }
}


// Block variant for the heaviest classes ((gg|gg): 32,814 VRR slots + 21,025 targets per quartet): one
// BLOCK of GBT threads per quartet instead of one warp.  With a warp per quartet the scratch of the warps in
// flight (0.5 MB each) is far larger than the L2 and every level is a round trip to HBM; with one block per
// SM the whole working set (148 x 0.5 MB) stays in the 126 MB L2 and each level is spread over 512 threads.
#define GBT 512
__global__ void __launch_bounds__(GBT, 1) rcg_eri_globalblock_kernel(GDev g, RcgLaunch a)
{
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    double *V = a.workspace + (int64_t)blockIdx.x * g.slots_per_warp;
    double *H = V + g.n_vslots;
    double *Bh = H + g.n_targets;
    extern __shared__ double p2smem[];
    const RcgBasisDev &b = a.basis;
    for (int64_t q = blockIdx.x; q < a.n; q += gridDim.x) {
        int sh[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) sh[k] = a.quartets[4 * q + a.perm[k]];
        double R[4][3];
#pragma unroll
        for (int k = 0; k < 4; ++k)
#pragma unroll
            for (int t = 0; t < 3; ++t) R[k][t] = b.centers[3 * sh[k] + t];
        for (int t = tid; t < g.n_targets; t += GBT) H[t] = 0.0;
        const int p0 = b.prim_off[sh[0]], p0e = b.prim_off[sh[0] + 1];
        const int p1 = b.prim_off[sh[1]], p1e = b.prim_off[sh[1] + 1];
        const int p2 = b.prim_off[sh[2]], p2e = b.prim_off[sh[2] + 1];
        const int p3 = b.prim_off[sh[3]], p3e = b.prim_off[sh[3] + 1];
        for (int i = p0; i < p0e; ++i)
        for (int j = p1; j < p1e; ++j)
        for (int k = p2; k < p2e; ++k)
        for (int l = p3; l < p3e; ++l) {
            RcgPrim p;
            rcg_prim_setup(p, R[0], R[1], R[2], R[3], b.exps[i], b.exps[j], b.exps[k], b.exps[l],
                           b.coefs[i] * b.coefs[j] * b.coefs[k] * b.coefs[l]);
            double F[17];
            rcg_boys<-1>(g.L, p.T, p.pref, b.boys, F);
            __syncthreads();                                     // previous primitive's H += V reads are done
            if (tid == 0)
                for (int m = 0; m <= g.L; ++m) V[m] = F[m];
            __syncthreads();
            for (int t = __ldg(g.tgt_off) + tid; t < __ldg(g.tgt_off + 1); t += GBT)
                H[__ldg(g.tindex + t)] += V[__ldg(g.tslots + t)];
            for (int lv = 0; lv < g.n_levels; ++lv) {
                __syncthreads();
                const int fe = __ldg(g.lvl_off + lv + 1);
                for (int f = __ldg(g.lvl_off + lv) + tid; f < fe; f += GBT) {
                    const uint32_t *w = g.vrr_fam + 5 * f;
                    const int od = __ldg(w), o1 = __ldg(w + 1), o3 = __ldg(w + 2), o5 = __ldg(w + 3);
                    const uint32_t meta = __ldg(w + 4);
                    const int mlo = meta & 31, nm = (meta >> 5) & 31, ket = (meta >> 10) & 1, ax = (meta >> 11) & 3;
                    const int n2 = (meta >> 13) & 15, nx = (meta >> 17) & 15;
                    const double c1 = ket ? p.QC[ax] : p.PA[ax];
                    const double c2 = ket ? p.WQ[ax] : p.WP[ax];
                    const double k3 = (double)n2 * (ket ? p.he : p.hz);
                    const double r3 = ket ? p.re : p.rz;
                    const double k5 = (double)nx * p.hze;
                    for (int m0 = mlo; m0 < mlo + nm; m0 += 4) {
                        const int cntm = min(4, mlo + nm - m0);
                        double a1[5], a3[5], a5[4];
#pragma unroll
                        for (int kk = 0; kk < 5; ++kk) a1[kk] = kk <= cntm ? V[o1 + m0 + kk] : 0.0;
                        if (n2) {
#pragma unroll
                            for (int kk = 0; kk < 5; ++kk) a3[kk] = kk <= cntm ? V[o3 + m0 + kk] : 0.0;
                        }
                        if (nx) {
#pragma unroll
                            for (int kk = 0; kk < 4; ++kk) a5[kk] = kk < cntm ? V[o5 + m0 + kk + 1] : 0.0;
                        }
#pragma unroll
                        for (int kk = 0; kk < 4; ++kk) {
                            if (kk < cntm) {
                                double v = c1 * a1[kk];
                                v = fma(c2, a1[kk + 1], v);
                                if (n2) v = fma(k3, fma(-r3, a3[kk + 1], a3[kk]), v);
                                if (nx) v = fma(k5, a5[kk], v);
                                V[od + m0 + kk] = v;
                            }
                        }
                    }
                }
                __syncthreads();
                for (int t = __ldg(g.tgt_off + lv + 1) + tid; t < __ldg(g.tgt_off + lv + 2); t += GBT)
                    H[__ldg(g.tindex + t)] += V[__ldg(g.tslots + t)];
            }
        }
        __syncthreads();
        double AB[3], CD[3];
#pragma unroll
        for (int t = 0; t < 3; ++t) { AB[t] = R[0][t] - R[1][t]; CD[t] = R[2][t] - R[3][t]; }
        rcg_phase2_block(g, a, q, H, Bh, p2smem, AB, CD, warp, lane, GBT / 32);
        __syncthreads();
    }
}

static bool use_block_variant(const RcgClassDesc &d) { return d.g.n_vslots >= 16384; }

// ---------------------------------------------------------------- host side
static size_t slots_per_warp(const RcgGlobalTables &t)
{
    return (size_t)t.n_vslots + (size_t)t.n_targets + (size_t)t.bra_nout * t.nC;
}

// warps of one launch: whole blocks of GW warps, at most 32 warps per SM, at most 8 GiB of scratch
static int64_t global_warps(const RcgClassDesc &d, int64_t n)
{
    int nsm = 148;
    rcg_sm_count(&nsm);                                           // cached per device
    if (use_block_variant(d)) return n < nsm ? n : nsm;          // units are blocks: one per SM, scratch stays in L2
    int64_t w = ((n + GW - 1) / GW) * GW;
    int64_t cap = (int64_t)nsm * 32;
    int64_t memcap = (int64_t)((8ull << 30) / (slots_per_warp(d.g) * 8)) / GW * GW;
    if (memcap < GW) memcap = GW;
    if (w > cap) w = cap;
    if (w > memcap) w = memcap;
    return w;
}

size_t rcg_global_workspace_bytes(const RcgClassDesc &d, int64_t n)
{
    if (n <= 0) return 0;
    return slots_per_warp(d.g) * 8 * (size_t)global_warps(d, n);
}

static std::mutex g_mu;
static std::map<std::pair<int, const RcgClassDesc *>, GDev> g_cache;

template <class T>
static cudaError_t upload(const T *h, size_t n, const T **d)
{
    void *p = nullptr;
    cudaError_t e = cudaMalloc(&p, (n ? n : 1) * sizeof(T));
    if (e != cudaSuccess) return e;
    e = cudaMemcpy(p, h, n * sizeof(T), cudaMemcpyHostToDevice);
    *d = (const T *)p;
    return e;
}

cudaError_t rcg_global_tables(const RcgClassDesc &d, GDev *out)
{
    int dev = 0;
    cudaGetDevice(&dev);
    std::lock_guard<std::mutex> lk(g_mu);
    auto key = std::make_pair(dev, &d);
    auto it = g_cache.find(key);
    if (it != g_cache.end()) { *out = it->second; return cudaSuccess; }
    const RcgGlobalTables &t = d.g;
    GDev g;
    cudaError_t e;
    if ((e = upload(t.vrr_fam, (size_t)t.n_fam * 5, &g.vrr_fam)) != cudaSuccess) return e;
    if ((e = upload(t.tslots, (size_t)t.n_targets, &g.tslots)) != cudaSuccess) return e;
    if ((e = upload(t.lvl_off, (size_t)t.n_levels + 1, &g.lvl_off)) != cudaSuccess) return e;
    if ((e = upload(t.tindex, (size_t)t.n_targets, &g.tindex)) != cudaSuccess) return e;
    if ((e = upload(t.tgt_off, (size_t)t.n_levels + 2, &g.tgt_off)) != cudaSuccess) return e;
    if ((e = upload(t.bra_ops, (size_t)t.n_bra_words, &g.bra_ops)) != cudaSuccess) return e;
    if ((e = upload(t.ket_ops, (size_t)t.n_ket_words, &g.ket_ops)) != cudaSuccess) return e;
    if ((e = upload(t.bra_noff, (size_t)t.n_bra_nodes, &g.bra_noff)) != cudaSuccess) return e;
    if ((e = upload(t.ket_noff, (size_t)t.n_ket_nodes, &g.ket_noff)) != cudaSuccess) return e;
    if ((e = upload(t.bra_loff, (size_t)t.n_bra_levels + 1, &g.bra_loff)) != cudaSuccess) return e;
    if ((e = upload(t.ket_loff, (size_t)t.n_ket_levels + 1, &g.ket_loff)) != cudaSuccess) return e;
    if ((e = upload(t.bra_out, (size_t)t.bra_nout, &g.bra_out)) != cudaSuccess) return e;
    if ((e = upload(t.ket_out, (size_t)t.ket_nout, &g.ket_out)) != cudaSuccess) return e;
    if ((e = upload(t.consts, (size_t)t.n_consts, &g.consts)) != cudaSuccess) return e;
    g.n_levels = t.n_levels; g.slots_per_warp = (int64_t)slots_per_warp(t);
    g.n_fam = t.n_fam; g.n_targets = t.n_targets; g.nA = t.nA; g.nC = t.nC; g.n_vslots = t.n_vslots;
    g.n_bra_levels = t.n_bra_levels; g.bra_nin = t.bra_nin; g.bra_nslots = t.bra_nslots; g.bra_nout = t.bra_nout;
    g.n_ket_levels = t.n_ket_levels; g.ket_nin = t.ket_nin; g.ket_nslots = t.ket_nslots; g.ket_nout = t.ket_nout;
    g.n_consts = t.n_consts;
    g.p2_slots = (t.bra_nslots > t.ket_nslots ? t.bra_nslots : t.ket_nslots) + 4 + t.n_consts;
    g.L = d.l[0] + d.l[1] + d.l[2] + d.l[3];
    g_cache[key] = g;
    *out = g;
    return cudaSuccess;
}

cudaError_t rcg_global_launch(const RcgClassDesc &d, const RcgLaunch &a)
{
    GDev g;
    cudaError_t e = rcg_global_tables(d, &g);
    if (e != cudaSuccess) return e;
    int64_t warps = global_warps(d, a.n);
    if (use_block_variant(d)) {
        const size_t smemb = sizeof(double) * (size_t)g.p2_slots * (GBT / 32);
        static RcgOnce onceb;        // the limit is raised once per device to the most any class needs
        if ((e = rcg_prepare_kernel(onceb, (const void *)rcg_eri_globalblock_kernel, 200 * 1024, nullptr)) != cudaSuccess) return e;
        if (smemb > 200 * 1024) return cudaErrorInvalidValue;
        rcg_eri_globalblock_kernel<<<(unsigned)warps, GBT, smemb, a.stream>>>(g, a);
        return cudaGetLastError();
    }
    const size_t smem = sizeof(double) * (size_t)g.p2_slots * GW;
    static RcgOnce once;
    if ((e = rcg_prepare_kernel(once, (const void *)rcg_eri_global_kernel, 200 * 1024, nullptr)) != cudaSuccess) return e;
    if (smem > 200 * 1024) return cudaErrorInvalidValue;
    rcg_eri_global_kernel<<<(unsigned)(warps / GW), GW * 32, smem, a.stream>>>(g, a);
    return cudaGetLastError();
}
