// eri_grad.cu -- first derivatives of contracted real-spherical ERIs with respect to the four shell centres
// (SURVEY 8(f) NEXT-4; PAPER.md:299 "first-derivative variants", :401; scheme of the HGP reference).
//
//   d/dA_i (ab|cd) = sum_prim c [ 2 alpha (a + 1_i, b|cd) - a_i (a - 1_i, b|cd) ]      (reading R-GRAD)
//
// and likewise for B (beta) and C (gamma); the D derivative is minus the sum of the other three (translational
// invariance).  One class-independent kernel, one thread block per shell quartet:
//   Phase 1, per primitive quartet: Gaussian-pair quantities and Boys values (csrc/rcg_device.cuh), the
//     vertical recurrence Eq. (2) level by level in shared memory -- bra levels [e0|00]^(m), e <= la+lb+1,
//     then ket levels [e0|f0]^(m), f <= lc+ld+1 -- and, fused with it (Alg. 2 line 7), the contraction of the
//     m = 0 values into FOUR accumulator sets that stay in shared memory: plain (for the lowered shells), and weighted by
//     2 alpha, 2 beta, 2 gamma (for the raised shell of the centre in question), each over the rectangle of targets its
//     horizontal recurrences need.
//   Phase 2, per centre: the horizontal recurrence Eq. (3) in closed form,
//     (a b| = sum_k binom(b, k) (A - B)^(b - k) [a + k, 0|, bra then ket, of the raised and of the lowered class; per axis the
//     combination above, the four dense Cartesian -> spherical steps Eq. (8)/(17) and the store.
// The integrals never leave the chip; out = [n][12][2la+1][2lb+1][2lc+1][2ld+1], derivative index 3 * centre + axis.
#define RCG_GRAD_QUAL __device__
#include "gen/grad_tables.h"
#include "rcg_device.cuh"

#define GRAD_MAX_THREADS 256
#define GRAD_SMEM_LIMIT 232448          // 227 KB per block on sm_100a
#define GRAD_TAB_DOUBLES 360            // component tables (880 + 1320 bytes) and the Phase-2 constants (72 doubles)

struct GradSet { int elo, ehi, flo, fhi, eoff, foff, nE, nF, base; };
struct GradPlan {
    int l[4];
    int E, F, M;                 // bra / ket levels of the vertical recurrence, top Boys order
    int nE, nElast;              // bra components of all levels <= E, and <= E - 1 (all the last ket level needs)
    GradSet set[4];              // plain, 2 alpha, 2 beta, 2 gamma
    int acc_doubles, bsize, lvlmax;
    int p2x, p2r, p2l, p2d;      // Phase-2 buffers: half-transformed, raised block, lowered block, Cartesian block
    int smem_doubles;
    int threads;
};

static inline int h_ncart(int l) { return (l + 1) * (l + 2) / 2; }
static inline int h_ncum(int l) { return l < 0 ? 0 : (l + 1) * (l + 2) * (l + 3) / 6; }   // components of levels 0..l

static void grad_plan(const int l[4], GradPlan &P)
{
    for (int k = 0; k < 4; ++k) P.l[k] = l[k];
    const int la = l[0], lb = l[1], lc = l[2], ld = l[3];
    P.E = la + lb + 1; P.F = lc + ld + 1; P.M = P.E + P.F;
    P.nE = h_ncum(P.E); P.nElast = h_ncum(P.E - 1);
    const int lo0 = la > 0 ? la - 1 : 0, fo0 = lc > 0 ? lc - 1 : 0;
    const int rect[4][4] = {{lo0, la + lb, fo0, lc + ld}, {la + 1, la + lb + 1, lc, lc + ld},
                            {la, la + lb + 1, lc, lc + ld}, {la, la + lb, lc + 1, lc + ld + 1}};
    int base = 0;
    for (int s = 0; s < 4; ++s) {
        GradSet &g = P.set[s];
        g.elo = rect[s][0]; g.ehi = rect[s][1]; g.flo = rect[s][2]; g.fhi = rect[s][3];
        g.eoff = h_ncum(g.elo - 1); g.foff = h_ncum(g.flo - 1);
        g.nE = h_ncum(g.ehi) - g.eoff; g.nF = h_ncum(g.fhi) - g.foff;
        g.base = base;
        base += g.nE * g.nF;
    }
    P.acc_doubles = base;
    P.bsize = (P.M + 1) * P.nE;
    P.lvlmax = 0;
    long long maxitems = 0;
    for (int f = 1; f <= P.F; ++f) {
        const int sz = P.nE * h_ncart(f) * (P.F - f + 1);
        if (sz > P.lvlmax) P.lvlmax = sz;
        if (sz > maxitems) maxitems = sz;
    }
    // Phase-2 buffers: the largest of the three raised / lowered classes
    P.p2x = P.p2r = P.p2l = 0;
    P.p2d = h_ncart(la) * h_ncart(lb) * h_ncart(lc) * h_ncart(ld);
    for (int p = 0; p < 3; ++p)
        for (int up = 0; up < 2; ++up) {
            int m[4] = {la, lb, lc, ld};
            m[p] += up ? 1 : -1;
            if (m[p] < 0) continue;
            const int nfr = h_ncum(m[2] + m[3]) - h_ncum(m[2] - 1);
            const int x = h_ncart(m[0]) * h_ncart(m[1]) * nfr;
            const int y = h_ncart(m[0]) * h_ncart(m[1]) * h_ncart(m[2]) * h_ncart(m[3]);
            if (x > P.p2x) P.p2x = x;
            if (up) { if (y > P.p2r) P.p2r = y; } else { if (y > P.p2l) P.p2l = y; }
        }
    if (P.p2x < P.p2d) P.p2x = P.p2d;         // doubles as the second buffer of the c2s steps
    const int vrr = P.bsize + 3 * P.lvlmax, p2 = P.p2x + P.p2r + P.p2l + P.p2d;
    P.smem_doubles = GRAD_TAB_DOUBLES + P.acc_doubles + (vrr > p2 ? vrr : p2);
    int nt = (int)((maxitems / 6 + 31) / 32) * 32;
    P.threads = nt < 32 ? 32 : (nt > GRAD_MAX_THREADS ? GRAD_MAX_THREADS : nt);
}

__device__ __forceinline__ double sel3(int i, double x, double y, double z) { return i == 0 ? x : (i == 1 ? y : z); }
__device__ __forceinline__ int seli(int i, int x, int y, int z) { return i == 0 ? x : (i == 1 ? y : z); }
__device__ __forceinline__ int d_ncart(int l) { return (l + 1) * (l + 2) / 2; }
__device__ __forceinline__ int d_ncum(int l) { return (l + 1) * (l + 2) * (l + 3) / 6; }      // l >= -1
// cumulative index of the component (i, j, lev - i - j)
__device__ __forceinline__ int d_cidx(int lev, int i, int j) { const int k = lev - i; return d_ncum(lev - 1) + k * (k + 1) / 2 + (k - j); }

// one side of Eq. (3) in closed form: dst[(row * n2 + i2) * ncol + col] = sum_k binom(b, k) X^(b - k) src[...(a + k)...], where the
// source is addressed as src[row_stride * row' + col_stride * col'] by the caller-supplied lambda
template <class Src>
__device__ __forceinline__ double hrr_sum(const uchar4 ca, const uchar4 cb, int l1, const double *bin, const double *pw, Src src)
{
    double s = 0.0;
    for (int kx = 0; kx <= cb.x; ++kx) {
        const double fx = bin[cb.x * 6 + kx] * pw[0 * 6 + cb.x - kx];
        for (int ky = 0; ky <= cb.y; ++ky) {
            const double fy = fx * bin[cb.y * 6 + ky] * pw[1 * 6 + cb.y - ky];
            for (int kz = 0; kz <= cb.z; ++kz) {
                const double f = fy * bin[cb.z * 6 + kz] * pw[2 * 6 + cb.z - kz];
                s = fma(f, src(d_cidx(l1 + kx + ky + kz, ca.x + kx, ca.y + ky)), s);
            }
        }
    }
    return s;
}

__global__ void __launch_bounds__(GRAD_MAX_THREADS)
rcg_eri_grad_kernel(const RcgBasisDev basis, const int32_t *__restrict__ quartets, double *__restrict__ out, const GradPlan P)
{
    extern __shared__ double smd[];
    uchar4 *comp = (uchar4 *)smd;                       // [220] (x, y, z, level)
    short *dec = (short *)(comp + RCG_GRAD_NCUM);       // [220][3] cumulative index of c - 1_i
    double *cst = smd + 288;                            // bin[6][6], pwAB[3][6], pwCD[3][6]
    double *acc = smd + GRAD_TAB_DOUBLES;
    double *work = acc + P.acc_doubles;
    const int tid = threadIdx.x, NT = blockDim.x;
    for (int t = tid; t < RCG_GRAD_NCUM; t += NT) {
        comp[t] = make_uchar4(rcg_grad_comp[t][0], rcg_grad_comp[t][1], rcg_grad_comp[t][2], rcg_grad_comp[t][3]);
        dec[3 * t] = rcg_grad_dec[t][0]; dec[3 * t + 1] = rcg_grad_dec[t][1]; dec[3 * t + 2] = rcg_grad_dec[t][2];
    }
    for (int t = tid; t < P.acc_doubles; t += NT) acc[t] = 0.0;
    const int64_t q = blockIdx.x;
    const int4 sh = *reinterpret_cast<const int4 *>(quartets + 4 * q);
    double A[3], B[3], C[3], D[3];
#pragma unroll
    for (int t = 0; t < 3; ++t) {
        A[t] = basis.centers[3 * sh.x + t]; B[t] = basis.centers[3 * sh.y + t];
        C[t] = basis.centers[3 * sh.z + t]; D[t] = basis.centers[3 * sh.w + t];
    }
    const int o0 = basis.prim_off[sh.x], o1 = basis.prim_off[sh.y], o2 = basis.prim_off[sh.z], o3 = basis.prim_off[sh.w];
    const int K0 = basis.prim_off[sh.x + 1] - o0, K1 = basis.prim_off[sh.y + 1] - o1;
    const int K2 = basis.prim_off[sh.z + 1] - o2, K3 = basis.prim_off[sh.w + 1] - o3;
    const int nE = P.nE, E = P.E, F = P.F, M = P.M;
    double *Bt = work;                                  // [m][nE]: [e0|00]^(m)
    double *lvl0 = work + P.bsize;
    __syncthreads();

    // ------------------------------------------------------------------ Phase 1
    for (int i0 = 0; i0 < K0; ++i0)
    for (int i1 = 0; i1 < K1; ++i1)
    for (int i2 = 0; i2 < K2; ++i2)
    for (int i3 = 0; i3 < K3; ++i3) {
        const double al = basis.exps[o0 + i0], be = basis.exps[o1 + i1], ga = basis.exps[o2 + i2], de = basis.exps[o3 + i3];
        const double cc4 = basis.coefs[o0 + i0] * basis.coefs[o1 + i1] * basis.coefs[o2 + i2] * basis.coefs[o3 + i3];
        RcgPrim pr;
        rcg_prim_setup(pr, A, B, C, D, al, be, ga, de, cc4);
        if (tid == 0) {
            double Fv[17];
            rcg_boys<-1>(M, pr.T, pr.pref, basis.boys, Fv);
            for (int m = 0; m <= M; ++m) Bt[m * nE] = Fv[m];
        }
        const double w1 = 2.0 * al, w2 = 2.0 * be, w3 = 2.0 * ga;
        __syncthreads();
        // bra levels: Eq. (2) with c = 0 on the first non-zero axis
        for (int n = 0; n < E; ++n) {
            const int nc = d_ncart(n + 1), rows = M - n, c0 = d_ncum(n);
            for (int t = tid; t < nc * rows; t += NT) {
                const int m = t / nc, c = c0 + (t - m * nc);
                const uchar4 cc = comp[c];
                const int i = cc.x ? 0 : (cc.y ? 1 : 2);
                const int c1 = dec[3 * c + i], n1 = seli(i, cc.x, cc.y, cc.z) - 1;
                const double *b0 = Bt + m * nE;
                double v = fma(sel3(i, pr.PA[0], pr.PA[1], pr.PA[2]), b0[c1], sel3(i, pr.WP[0], pr.WP[1], pr.WP[2]) * b0[nE + c1]);
                if (n1 > 0) {
                    const int c2 = dec[3 * c1 + i];
                    v = fma((double)n1 * pr.hz, fma(-pr.rz, b0[nE + c2], b0[c2]), v);
                }
                Bt[m * nE + c] = v;
            }
            __syncthreads();
        }
        // targets with f = 0
        for (int t = tid; t < nE; t += NT) {
            const double v = Bt[t];
            const int le = comp[t].w;
#pragma unroll
            for (int s = 0; s < 4; ++s) {
                const GradSet &g = P.set[s];
                if (g.flo == 0 && le >= g.elo && le <= g.ehi) {
                    const double w = s == 0 ? 1.0 : (s == 1 ? w1 : (s == 2 ? w2 : w3));
                    acc[g.base + (t - g.eoff)] = fma(w, v, acc[g.base + (t - g.eoff)]);
                }
            }
        }
        // ket levels: the mirror of Eq. (2) (R-KET) with the cross term e - 1_i
        const double *prev = Bt, *prev2 = Bt;
        int mcp = M + 1, mcp2 = M + 1;
        for (int f = 0; f < F; ++f) {
            double *cur = lvl0 + (f % 3) * P.lvlmax;
            const int mcn = F - f, ncf = d_ncart(f + 1), nEl = (f + 1 == F) ? P.nElast : nE;
            const int cf0 = d_ncum(f), cfm = d_ncum(f - 1), cfmm = f >= 2 ? d_ncum(f - 2) : 0;
            const int total = nEl * ncf * mcn;
            const float rnel = 1.0f / (float)nEl, rmcn = 1.0f / (float)mcn;
            for (int t = tid; t < total; t += NT) {
                int eidx, m;
                const int r = rcg_divmod(t, nEl, rnel, eidx);
                const int fc = rcg_divmod(r, mcn, rmcn, m);
                const int c = cf0 + fc;
                const uchar4 cc = comp[c];
                const int i = cc.x ? 0 : (cc.y ? 1 : 2);
                const int c1g = dec[3 * c + i], c1 = c1g - cfm, n1 = seli(i, cc.x, cc.y, cc.z) - 1;
                const double *p0 = prev + (c1 * mcp + m) * nE;
                double v = fma(sel3(i, pr.QC[0], pr.QC[1], pr.QC[2]), p0[eidx], sel3(i, pr.WQ[0], pr.WQ[1], pr.WQ[2]) * p0[nE + eidx]);
                if (n1 > 0) {
                    const int c2 = dec[3 * c1g + i] - cfmm;
                    const double *p2 = prev2 + (c2 * mcp2 + m) * nE;
                    v = fma((double)n1 * pr.he, fma(-pr.re, p2[nE + eidx], p2[eidx]), v);
                }
                const uchar4 ce = comp[eidx];
                const int ei = seli(i, ce.x, ce.y, ce.z);
                if (ei > 0) v = fma((double)ei * pr.hze, p0[nE + dec[3 * eidx + i]], v);
                cur[(fc * mcn + m) * nE + eidx] = v;
                if (m == 0) {
                    const int le = ce.w, lf = f + 1;
#pragma unroll
                    for (int s = 0; s < 4; ++s) {
                        const GradSet &g = P.set[s];
                        if (le >= g.elo && le <= g.ehi && lf >= g.flo && lf <= g.fhi) {
                            const double w = s == 0 ? 1.0 : (s == 1 ? w1 : (s == 2 ? w2 : w3));
                            double *a = acc + g.base + (c - g.foff) * g.nE + (eidx - g.eoff);
                            *a = fma(w, v, *a);
                        }
                    }
                }
            }
            __syncthreads();
            prev2 = prev; mcp2 = mcp; prev = cur; mcp = mcn;
        }
    }

    // ------------------------------------------------------------------ Phase 2
    double *bin = cst, *pwAB = cst + 36, *pwCD = cst + 54;
    if (tid < 36) {
        const int n = tid / 6, k = tid - 6 * n;
        double b = 0.0;
        if (k <= n) { b = 1.0; for (int j = 1; j <= k; ++j) b = b * (double)(n - k + j) / (double)j; }
        bin[tid] = b;
    }
    if (tid < 3) {
        const double ab = A[tid] - B[tid], cd = C[tid] - D[tid];
        double x = 1.0, y = 1.0;
        for (int k = 0; k < 6; ++k) { pwAB[tid * 6 + k] = x; pwCD[tid * 6 + k] = y; x *= ab; y *= cd; }
    }
    double *bufX = work, *bufR = bufX + P.p2x, *bufL = bufR + P.p2r, *bufD = bufL + P.p2l;
    const int la = P.l[0], lb = P.l[1], lc = P.l[2], ld = P.l[3];
    const int nsa = 2 * la + 1, nsb = 2 * lb + 1, nsc = 2 * lc + 1, nsd = 2 * ld + 1;
    const int nsph = nsa * nsb * nsc * nsd;
    double *outq = out + (size_t)q * 12 * nsph;
    __syncthreads();
    for (int p = 0; p < 3; ++p) {
        // horizontal recurrences of the raised (source: the weighted set p + 1) and the lowered class (the plain set)
        for (int up = 1; up >= 0; --up) {
            const int sh1 = up ? 1 : -1;
            const int l1 = la + (p == 0 ? sh1 : 0), l2 = lb + (p == 1 ? sh1 : 0), l3 = lc + (p == 2 ? sh1 : 0), l4 = ld;
            if (l1 < 0 || l2 < 0 || l3 < 0) continue;                  // uniform: no lowered class of an s shell
            const GradSet &g = P.set[up ? p + 1 : 0];
            const int n1 = d_ncart(l1), n2 = d_ncart(l2), n3 = d_ncart(l3), n4 = d_ncart(l4);
            const int f0 = d_ncum(l3 - 1), nfr = d_ncum(l3 + l4) - f0;
            const int c1o = d_ncum(l1 - 1), c2o = d_ncum(l2 - 1), c3o = f0, c4o = d_ncum(l4 - 1);
            double *Y = up ? bufR : bufL;
            for (int t = tid; t < n1 * n2 * nfr; t += NT) {
                const int fi = t % nfr, ab = t / nfr, ib = ab % n2, ia = ab / n2;
                const double *src = acc + g.base + (f0 + fi - g.foff) * g.nE - g.eoff;
                bufX[t] = hrr_sum(comp[c1o + ia], comp[c2o + ib], l1, bin, pwAB, [&](int e) { return src[e]; });
            }
            __syncthreads();
            for (int t = tid; t < n1 * n2 * n3 * n4; t += NT) {
                const int id = t % n4, r = t / n4, ic = r % n3, ab = r / n3;
                const double *src = bufX + ab * nfr - f0;
                Y[t] = hrr_sum(comp[c3o + ic], comp[c4o + id], l3, bin, pwCD, [&](int e) { return src[e]; });
            }
            __syncthreads();
        }
        const int lp = P.l[p];
        const int nca = d_ncart(la), ncb = d_ncart(lb), ncc = d_ncart(lc), ncd = d_ncart(ld);
        const int ncblk = nca * ncb * ncc * ncd;
        // strides of the raised / lowered blocks: position p has ncart(lp + 1) / ncart(lp - 1) components
        const int nup = d_ncart(lp + 1), ndn = lp > 0 ? d_ncart(lp - 1) : 1;
        const int dR1 = p == 1 ? nup : ncb, dR2 = p == 2 ? nup : ncc, dL1 = p == 1 ? ndn : ncb, dL2 = p == 2 ? ndn : ncc;
        const int cpo = d_ncum(lp - 1), cpu = d_ncum(lp), cpd = lp > 0 ? d_ncum(lp - 2) : 0;
        for (int ax = 0; ax < 3; ++ax) {
            for (int t = tid; t < ncblk; t += NT) {
                int r = t;
                const int i3 = r % ncd; r /= ncd;
                const int i2 = r % ncc; r /= ncc;
                const int i1 = r % ncb, i0 = r / ncb;
                const int cx = cpo + seli(p, i0, i1, i2);
                const uchar4 cc = comp[cx];
                const int upi = d_cidx(lp + 1, cc.x + (ax == 0), cc.y + (ax == 1)) - cpu;
                double v = bufR[(((p == 0 ? upi : i0) * dR1 + (p == 1 ? upi : i1)) * dR2 + (p == 2 ? upi : i2)) * ncd + i3];
                const int pw = seli(ax, cc.x, cc.y, cc.z);
                if (pw > 0) {
                    const int dn = dec[3 * cx + ax] - cpd;
                    v = fma(-(double)pw, bufL[(((p == 0 ? dn : i0) * dL1 + (p == 1 ? dn : i1)) * dL2 + (p == 2 ? dn : i2)) * ncd + i3], v);
                }
                bufD[t] = v;
            }
            __syncthreads();
            // four dense c2s steps, Eq. (17); the last one stores
            int dims[4] = {nca, ncb, ncc, ncd};
            double *src = bufD, *dst = bufX;
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const int lk = P.l[k], ns = 2 * lk + 1, ncx = dims[k];
                int inner = 1, outer = 1;
#pragma unroll
                for (int j = k + 1; j < 4; ++j) inner *= dims[j];
#pragma unroll
                for (int j = 0; j < k; ++j) outer *= dims[j];
                const double *T = rcg_grad_c2s + rcg_grad_c2s_off[lk];
                const int total = outer * ns * inner;
                for (int t = tid; t < total; t += NT) {
                    const int in = t % inner, r = t / inner, ms = r % ns, o = r / ns;
                    const double *s0 = src + (o * ncx) * inner + in;
                    double s = 0.0;
                    for (int c = 0; c < ncx; ++c) s = fma(T[ms * ncx + c], s0[c * inner], s);
                    if (k < 3) dst[t] = s;
                    else {
                        outq[(3 * p + ax) * nsph + t] = s;
                        double *od = outq + (9 + ax) * nsph + t;
                        *od = p == 0 ? -s : *od - s;
                    }
                }
                dims[k] = ns;
                __syncthreads();
                double *tmp = src; src = dst; dst = tmp;
            }
        }
    }
}

// ---------------------------------------------------------------- host side
bool rcg_grad_supported(const int l[4], size_t *smem_bytes)
{
    for (int k = 0; k < 4; ++k)
        if (l[k] < 0 || l[k] > RCG_LMAX) return false;
    GradPlan P;
    grad_plan(l, P);
    if (smem_bytes) *smem_bytes = sizeof(double) * (size_t)P.smem_doubles;
    return P.M <= 16 && P.E <= RCG_GRAD_LEVELS && P.F <= RCG_GRAD_LEVELS && sizeof(double) * (size_t)P.smem_doubles <= GRAD_SMEM_LIMIT;
}

cudaError_t rcg_grad_launch(const RcgGradLaunch &a)
{
    GradPlan P;
    grad_plan(a.l, P);
    static RcgOnce once;
    int nsm = 0;
    cudaError_t e = rcg_prepare_kernel(once, (const void *)rcg_eri_grad_kernel, GRAD_SMEM_LIMIT, &nsm);
    if (e != cudaSuccess) return e;
    const size_t smem = sizeof(double) * (size_t)P.smem_doubles;
    const int64_t maxgrid = 0x7fffffff;
    for (int64_t q0 = 0; q0 < a.n; q0 += maxgrid) {
        const int64_t qn = a.n - q0 < maxgrid ? a.n - q0 : maxgrid;
        const size_t nout = 12 * (size_t)(2 * a.l[0] + 1) * (2 * a.l[1] + 1) * (2 * a.l[2] + 1) * (2 * a.l[3] + 1);
        rcg_eri_grad_kernel<<<(unsigned)qn, P.threads, smem, a.stream>>>(a.basis, a.quartets + 4 * q0, a.out + nout * (size_t)q0, P);
        if ((e = cudaGetLastError()) != cudaSuccess) return e;
    }
    return cudaSuccess;
}
