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
// component tables (880 + 1320 bytes -> 288 doubles), Phase-2 constants (bin 36, powers 2 x 18), the c2s matrices (245)
#define GRAD_CST 288
#define GRAD_C2S (GRAD_CST + 72)
#define GRAD_TAB_DOUBLES (GRAD_C2S + RCG_GRAD_NC2S + 3)

struct GradSet { int elo, ehi, flo, fhi, eoff, foff, nE, nF, ldE, base; };   // ldE: odd row stride (a lane per ket target in Phase 2)
struct GradPlan {
    int l[4];
    int E, F, M;                 // bra / ket levels of the vertical recurrence, top Boys order
    int nE, nElast;              // bra components of all levels <= E, and <= E - 1 (all the last ket level needs)
    GradSet set[4];              // plain, 2 alpha, 2 beta, 2 gamma
    int acc_doubles, bsize, lvlmax;
    int p2x, p2r, p2l, p2d;      // Phase-2 buffers: half-transformed, raised block, lowered block, Cartesian block
    int nrows;                   // (ket component, m) rows of all ket levels: one 32-byte record each (built once per block)
    int tab_doubles;             // row records, per-bra-component records and cross-term tables
    int smem_doubles;
    int threads;                 // threads of one primitive group
    int groups;                  // mode 1: primitive groups (warps) per block, each with its own buffers
    int mode;                    // 0: a block per quartet; 1: a warp per primitive group of one quartet; 2: a sub-warp group of `sub` lanes per quartet;
                                 // 3: persistent blocks, accumulators and Phase-2 buffers in a global scratch
    int sub;                     // mode 2: lanes per quartet (4, 8, 16 or 32); 256 / sub quartets per block
    int scratch_doubles;         // mode 3: accumulator sets + Phase-2 buffers + constants of one block, in global memory
    int k4_lo, k4_hi;            // this launch evaluates the quartets with k4_lo <= K4 < k4_hi and leaves the others untouched (split lists)
    int vrr_doubles;             // bra table + three level buffers of one group
    int col[4];                  // kernel position k works on the caller's quartet column col[k] (the heavier shell of a pair first)
    int ostr[4];                 // stride of the kernel's spherical index k in the caller's output block
};

static inline int h_ncart(int l) { return (l + 1) * (l + 2) / 2; }
static inline int h_ncum(int l) { return l < 0 ? 0 : (l + 1) * (l + 2) * (l + 3) / 6; }   // components of levels 0..l

static void grad_plan(const int l[4], long long k4max, GradPlan &P)
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
        g.ldE = g.nE | 1;
        g.base = base;
        base += g.ldE * g.nF;
    }
    P.acc_doubles = base;
    P.bsize = (P.M + 1) * P.nE;
    P.lvlmax = 0;
    int maxunits = 1;
    P.nrows = 0;
    for (int f = 1; f <= P.F; ++f) {
        const int sz = P.nE * h_ncart(f) * (P.F - f + 1);
        if (sz > P.lvlmax) P.lvlmax = sz;
        const int units = h_ncart(f) * (P.F - f + 1) * ((P.nE + 31) / 32);
        if (units > maxunits) maxunits = units;
        P.nrows += h_ncart(f) * (P.F - f + 1);
    }
    // rows: 4 doubles each; bra records: 1 double per component; cross-term counts 3 nE doubles, cross-term indices 3 nE shorts
    P.tab_doubles = 4 * P.nrows + P.nE + 3 * P.nE + (3 * P.nE + 3) / 4 + 1;
    // Phase-2 buffers: the largest of the three raised / lowered classes
    P.p2x = P.p2r = P.p2l = 0;
    P.p2d = h_ncart(la) * h_ncart(lb) * h_ncart(lc) * h_ncart(ld);
    for (int p = 0; p < 3; ++p)
        for (int up = 0; up < 2; ++up) {
            int m[4] = {la, lb, lc, ld};
            m[p] += up ? 1 : -1;
            if (m[p] < 0) continue;
            const int nfr = h_ncum(m[2] + m[3]) - h_ncum(m[2] - 1);
            const int x = h_ncart(m[0]) * h_ncart(m[1]) * (nfr | 1);
            const int y = h_ncart(m[0]) * h_ncart(m[1]) * h_ncart(m[2]) * h_ncart(m[3]);
            if (x > P.p2x) P.p2x = x;
            if (up) { if (y > P.p2r) P.p2r = y; } else { if (y > P.p2l) P.p2l = y; }
        }
    if (P.p2x < P.p2d) P.p2x = P.p2d;         // doubles as the second buffer of the c2s steps
    const int p2 = P.p2x + P.p2r + P.p2l + P.p2d;
    P.vrr_doubles = P.bsize + 3 * P.lvlmax;
    const int warps = (maxunits + 5) / 6;     // about six (row, pass) units of the widest ket level per warp
    P.threads = 32 * (warps < 1 ? 1 : (warps > GRAD_MAX_THREADS / 32 ? GRAD_MAX_THREADS / 32 : warps));
    // light classes (at most three warps' worth of rows per level):
    //  * mode 1, ONE warp per primitive group and several groups per block, each with its own recurrence buffers and accumulator sets (summed
    //    before Phase 2), as many as fit 72 KB -- where the basis HAS deep contractions (K4 of 256 and more possible in this class): a deeply
    //    contracted quartet is not serial in one warp, the barriers of Phase 1 become __syncwarp, and Phase 2 has the whole block;
    //  * mode 2, a SUB-WARP GROUP of 4..32 lanes per quartet and 256 / lanes quartets per block, each with private buffers; the groups of a
    //    warp run one program in lockstep (full-warp __syncwarp), so a warp instruction serves 8 (ss|ss) quartets instead of one: the light
    //    classes are bound by the instruction count of the generic code.  K4 = 1 lists of 200,000 quartets: (ss|ss) 2.56 -> 0.36 ms,
    //    (ps|ss) 3.23 -> 0.85, (ds|ss) 4.28 -> 1.15, (pp|ps) 7.07 -> 4.03, (pp|pp) 14.6 -> 11.5.
    P.groups = 1; P.mode = 0; P.sub = 32;
    const int per_quartet = P.acc_doubles + (P.vrr_doubles > p2 ? P.vrr_doubles : p2) + 72;
    if (warps <= 3 && k4max >= 256) {
        P.threads = 32;
        for (int g = 8; g > 1; g >>= 1) {
            const int w = g * P.vrr_doubles, d = GRAD_TAB_DOUBLES + P.tab_doubles + g * P.acc_doubles + (w > p2 ? w : p2);
            if (d * 8 <= 72 * 1024) { P.groups = g; P.mode = 1; break; }
        }
    } else if (warps <= 3) {
        int sub = 4;          // the narrowest group whose 256 / sub quartets fit 110 KB (two blocks per SM; 72 and 220 KB measured slower)
        for (; sub <= 32; sub <<= 1)
            if ((GRAD_TAB_DOUBLES + P.tab_doubles + (GRAD_MAX_THREADS / sub) * per_quartet) * 8 <= 110 * 1024) { P.mode = 2; P.sub = sub; break; }
    }
    if (P.mode == 2) {
        P.smem_doubles = GRAD_TAB_DOUBLES + P.tab_doubles + (GRAD_MAX_THREADS / P.sub) * per_quartet;
        P.scratch_doubles = 0;
        P.k4_lo = 0; P.k4_hi = 0x7fffffff;
        return;
    }
    const int w = P.groups * P.vrr_doubles;
    P.smem_doubles = GRAD_TAB_DOUBLES + P.tab_doubles + P.groups * P.acc_doubles + (w > p2 ? w : p2);
    P.scratch_doubles = 0;
    P.k4_lo = 0; P.k4_hi = 0x7fffffff;
    // mode 3, heavy classes ((fd|fd), (ff|dd), (ff|fd), (ff|ff), ...): the accumulator sets and the Phase-2 buffers do not fit beside the
    // recurrence buffers -- they move to a per-block scratch in global memory (one persistent block per SM: 148 x 0.6 MB for (ff|ff) lives in
    // the L2), the tables and the level buffers of Phase 1 stay in shared memory
    if (P.mode == 0 && (size_t)P.smem_doubles * 8 > GRAD_SMEM_LIMIT && (size_t)(GRAD_TAB_DOUBLES + P.tab_doubles + P.vrr_doubles) * 8 <= GRAD_SMEM_LIMIT) {
        P.mode = 3;
        P.smem_doubles = GRAD_TAB_DOUBLES + P.tab_doubles + P.vrr_doubles;
        P.scratch_doubles = ((P.acc_doubles + p2 + 72) + 31) & ~31;
    }
}

__device__ __forceinline__ double sel3(int i, double x, double y, double z) { return i == 0 ? x : (i == 1 ? y : z); }
__device__ __forceinline__ int seli(int i, int x, int y, int z) { return i == 0 ? x : (i == 1 ? y : z); }
__device__ __forceinline__ int d_ncart(int l) { return (l + 1) * (l + 2) / 2; }
__device__ __forceinline__ int d_ncum(int l) { return (l + 1) * (l + 2) * (l + 3) / 6; }      // l >= -1
// cumulative index of the component (i, j, lev - i - j)
__device__ __forceinline__ int d_cidx(int lev, int i, int j) { const int k = lev - i; return d_ncum(lev - 1) + k * (k + 1) / 2 + (k - j); }

// one side of Eq. (3) in closed form for one (a, b) pair of components: sum_k binom(b, k) X^(b - k) src(a + k), the k loops and the
// coefficients warp-uniform, src(cumulative index of a + k) evaluated per lane
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

template <int NC>
__device__ __forceinline__ double c2s_dot(const double *__restrict__ T, const double *__restrict__ s0, int inner)
{
    double s = 0.0;
#pragma unroll
    for (int c = 0; c < NC; ++c) s = fma(T[c], s0[c * inner], s);
    return s;
}

template <int MODE>
__global__ void __launch_bounds__(GRAD_MAX_THREADS)
rcg_eri_grad_kernel(const RcgBasisDev basis, const int32_t *__restrict__ quartets, int64_t nq, double *__restrict__ out, double *scratch, const GradPlan P)
{
    extern __shared__ double smd[];
    uchar4 *comp = (uchar4 *)smd;                       // [220] (x, y, z, level)
    short *dec = (short *)(comp + RCG_GRAD_NCUM);       // [220][3] cumulative index of c - 1_i
    double *cst = smd + GRAD_CST;                       // bin[6][6], pwAB[3][6], pwCD[3][6]
    double *c2s = smd + GRAD_C2S;
    int4 *rowrec = (int4 *)(smd + GRAD_TAB_DOUBLES);            // [nrows][2]: {src0, src2, dst, axis | n1 << 8}, {acc offsets of the 4 sets}
    int2 *brarec = (int2 *)(smd + GRAD_TAB_DOUBLES + 4 * P.nrows);   // [nE]: {c1 | c2 << 16, axis | n1 << 8}
    double *ecn = smd + GRAD_TAB_DOUBLES + 4 * P.nrows + P.nE;       // [3][nE]: e_i as a double
    short *crs = (short *)(ecn + 3 * P.nE);                         // [3][nE]: cumulative index of e - 1_i (0 where e_i = 0)
    double *acc = smd + GRAD_TAB_DOUBLES + P.tab_doubles;
    if (MODE == 1 && P.k4_lo > 0) {                     // split list: a block whose quartet belongs to the other launch leaves before any set-up
        const int32_t *qq = quartets + 4 * (int64_t)blockIdx.x;
        long long k4 = 1;
        for (int k = 0; k < 4; ++k) k4 *= basis.prim_off[qq[k] + 1] - basis.prim_off[qq[k]];
        if (k4 < P.k4_lo) return;
    }
    constexpr bool GROUPED = MODE == 1;                 // a warp per primitive group of the block's quartet
    constexpr bool SUBQ = MODE == 2;                    // a sub-warp group of LS lanes per quartet
    constexpr bool HEAVY = MODE == 3;                   // persistent block; accumulators and Phase-2 buffers in the block's global scratch
    const int G = GROUPED ? P.groups : 1;
    const int tid = threadIdx.x, NT = blockDim.x, lane = tid & 31, warp = tid >> 5, NW = NT >> 5;
    // the unit that works on one row / one run of consecutive items: a warp (LS = 32 lanes, L0 = lane) or the quartet's sub-group
    const int LS = SUBQ ? P.sub : 32, L0 = SUBQ ? (tid & (P.sub - 1)) : lane;
    // mode 2: the sub-groups of a warp run in LOCKSTEP (one program, full-warp __syncwarp): a warp instruction serves 32 / LS quartets; every
    // group loops to the largest K4 of its warp (spent groups contribute zeros) and a group past the end of the list repeats the last quartet
    // without storing -- sub-group barriers with their own masks would split the warp into separately issued parts
    // Phase 1: group g = threads [g NTg, (g + 1) NTg) -- the whole block, one warp, or the sub-group; its barriers are its own
    const int NTg = SUBQ ? LS : (GROUPED ? 32 : NT), grp = GROUPED ? warp : 0, ltid = SUBQ ? L0 : (GROUPED ? lane : tid);
    const int lwarp = (GROUPED || SUBQ) ? 0 : warp, NWg = (GROUPED || SUBQ) ? 1 : NW;
    // Phase 2: the whole block (modes 0, 1) or the quartet's sub-group (mode 2)
    const int tid2 = SUBQ ? L0 : tid, NT2 = SUBQ ? LS : NT, warp2 = SUBQ ? 0 : warp, NW2 = SUBQ ? 1 : NW;
    const int p2doubles = P.p2x + P.p2r + P.p2l + P.p2d;
    const int per_quartet = P.acc_doubles + (P.vrr_doubles > p2doubles ? P.vrr_doubles : p2doubles) + 72;
    double *const smem_work = acc;                      // mode 3: the recurrence buffers take the place of the accumulators in shared memory
    if (HEAVY) acc = scratch + (size_t)blockIdx.x * P.scratch_doubles;
    double *accg = SUBQ ? acc + (tid / LS) * per_quartet : acc + grp * P.acc_doubles;
    double *work = SUBQ ? accg + P.acc_doubles : acc + G * P.acc_doubles;
    if (SUBQ) cst = work + (per_quartet - P.acc_doubles - 72);     // the group's own Phase-2 constants
    if (HEAVY) cst = acc + P.acc_doubles + p2doubles;
    for (int t = tid; t < RCG_GRAD_NCUM; t += NT) {
        comp[t] = make_uchar4(rcg_grad_comp[t][0], rcg_grad_comp[t][1], rcg_grad_comp[t][2], rcg_grad_comp[t][3]);
        dec[3 * t] = rcg_grad_dec[t][0]; dec[3 * t + 1] = rcg_grad_dec[t][1]; dec[3 * t + 2] = rcg_grad_dec[t][2];
    }
    for (int t = tid; t < RCG_GRAD_NC2S; t += NT) c2s[t] = rcg_grad_c2s[t];
    if (SUBQ) { for (int t = L0; t < P.acc_doubles; t += LS) accg[t] = 0.0; }
    else if (!HEAVY) { for (int t = tid; t < G * P.acc_doubles; t += NT) acc[t] = 0.0; }
    const int nE = P.nE, E = P.E, F = P.F, M = P.M;
    // the programs of Phase 1 do not depend on the primitive quartet: one record per (ket component, m) row and per bra component
    for (int t = tid; t < nE; t += NT) {
        const int cx = rcg_grad_comp[t][0], cy = rcg_grad_comp[t][1], cz = rcg_grad_comp[t][2];
        const int i = cx ? 0 : (cy ? 1 : 2);
        const int c1 = t ? rcg_grad_dec[t][i] : 0, n1 = t ? (i == 0 ? cx : (i == 1 ? cy : cz)) - 1 : 0;
        const int c2 = n1 > 0 ? rcg_grad_dec[c1][i] : 0;
        brarec[t] = make_int2(c1 | (c2 << 16), i | (n1 << 8));
        for (int a = 0; a < 3; ++a) {
            const int ea = rcg_grad_comp[t][a];
            ecn[a * nE + t] = (double)ea;
            crs[a * nE + t] = ea ? rcg_grad_dec[t][a] : 0;
        }
    }
    {
        int r0 = 0, mcp = M + 1, mcp2 = M + 1;
        for (int f = 0; f < F; ++f) {
            const int mcn = F - f, ncf = d_ncart(f + 1);
            const int cf0 = d_ncum(f), cfm = d_ncum(f - 1), cfmm = f >= 2 ? d_ncum(f - 2) : 0, lf = f + 1;
            for (int t = tid; t < ncf * mcn; t += NT) {
                const int fc = t / mcn, m = t - fc * mcn, c = cf0 + fc;
                const int cx = rcg_grad_comp[c][0], cy = rcg_grad_comp[c][1], cz = rcg_grad_comp[c][2];
                const int i = cx ? 0 : (cy ? 1 : 2);
                const int c1g = rcg_grad_dec[c][i], n1 = (i == 0 ? cx : (i == 1 ? cy : cz)) - 1;
                const int src0 = ((c1g - cfm) * mcp + m) * nE;
                const int src2 = n1 > 0 ? ((rcg_grad_dec[c1g][i] - cfmm) * mcp2 + m) * nE : -1;
                rowrec[2 * (r0 + t)] = make_int4(src0, src2, (fc * mcn + m) * nE, i | (n1 << 8));
                int ao[4];
#pragma unroll
                for (int s = 0; s < 4; ++s) {
                    const GradSet &g = P.set[s];
                    ao[s] = (m == 0 && lf >= g.flo && lf <= g.fhi) ? g.base + (c - g.foff) * g.ldE - g.eoff : (int)0x80000000;
                }
                rowrec[2 * (r0 + t) + 1] = make_int4(ao[0], ao[1], ao[2], ao[3]);
            }
            r0 += ncf * mcn;
            mcp2 = mcp; mcp = mcn;
        }
    }
    __syncthreads();
    for (int64_t qloop = blockIdx.x; qloop < (HEAVY ? nq : (int64_t)blockIdx.x + 1); qloop += gridDim.x) {      // mode 3: the block works through its share of the list
    const int64_t qraw = SUBQ ? (int64_t)blockIdx.x * (NT / LS) + tid / LS : qloop;
    if (SUBQ && (int64_t)blockIdx.x * (NT / LS) + (tid - lane) / LS >= nq) return;      // a whole warp past the end (no block-wide barrier beyond this point in mode 2)
    const bool valid = !SUBQ || qraw < nq;
    const int64_t q = valid ? qraw : nq - 1;
    if (HEAVY) {
        for (int t = tid; t < P.acc_doubles; t += NT) acc[t] = 0.0;
        __syncthreads();
    }
    const int4 shc = *reinterpret_cast<const int4 *>(quartets + 4 * q);      // the caller's columns
    int4 sh;            // pairs are only ever exchanged inside themselves: col[0], col[1] in {0, 1}, col[2], col[3] in {2, 3}
    sh.x = P.col[0] ? shc.y : shc.x; sh.y = P.col[1] ? shc.y : shc.x; sh.z = P.col[2] == 3 ? shc.w : shc.z; sh.w = P.col[3] == 3 ? shc.w : shc.z;
    double A[3], B[3], C[3], D[3];
#pragma unroll
    for (int t = 0; t < 3; ++t) {
        A[t] = basis.centers[3 * sh.x + t]; B[t] = basis.centers[3 * sh.y + t];
        C[t] = basis.centers[3 * sh.z + t]; D[t] = basis.centers[3 * sh.w + t];
    }
    const int o0 = basis.prim_off[sh.x], o1 = basis.prim_off[sh.y], o2 = basis.prim_off[sh.z], o3 = basis.prim_off[sh.w];
    const int K0 = basis.prim_off[sh.x + 1] - o0, K1 = basis.prim_off[sh.y + 1] - o1;
    const int K2 = basis.prim_off[sh.z + 1] - o2, K3 = basis.prim_off[sh.w + 1] - o3;
    double *Bt = HEAVY ? smem_work : (SUBQ ? work : work + grp * P.vrr_doubles);      // [m][nE]: [e0|00]^(m)
    double *lvl0 = Bt + P.bsize;
#define GRAD_GSYNC() do { if (SUBQ || GROUPED) __syncwarp(); else __syncthreads(); } while (0)

    // ------------------------------------------------------------------ Phase 1
    const int K4all = K0 * K1 * K2 * K3;
    const bool mine = !SUBQ || K4all < P.k4_hi;         // mode 2 on a split list: deeper quartets belong to the mode-1 launch
    const int K4 = mine ? K4all : 0;
    if (SUBQ && !__any_sync(0xffffffffu, mine)) return;      // a warp whose quartets all belong to the other launch
    const int K4w = SUBQ ? __reduce_max_sync(0xffffffffu, K4) : K4;
    for (int pq = GROUPED ? grp : 0; pq < K4w; pq += GROUPED ? G : 1) {
        int r4 = pq < K4 ? pq : (K4 > 0 ? K4 - 1 : 0);
        const int i3 = r4 % K3; r4 /= K3;
        const int i2 = r4 % K2; r4 /= K2;
        const int i1 = r4 % K1, i0 = r4 / K1;
        const double al = basis.exps[o0 + i0], be = basis.exps[o1 + i1], ga = basis.exps[o2 + i2], de = basis.exps[o3 + i3];
        const double cc4 = pq < K4 ? basis.coefs[o0 + i0] * basis.coefs[o1 + i1] * basis.coefs[o2 + i2] * basis.coefs[o3 + i3] : 0.0;
        RcgPrim pr;
        rcg_prim_setup(pr, A, B, C, D, al, be, ga, de, cc4);
        // Boys values [00|00]^(m) = pref F_m(T), m <= M (R-BOYS): below T = 36 every order by its own 9-term Taylor series about the
        // nearest grid point (a lane per order; the grid holds orders up to m + 8), above it F_0 = sqrt(pi / T) / 2 and the upward recursion
        if (lwarp == 0) {
            if (pr.T < RCG_BOYS_TS) {
                for (int mo = L0; mo <= M; mo += LS) {
                    const int row = (int)(pr.T * 8.0 + 0.5);
                    const double d = (double)row * 0.125 - pr.T;
                    const double *r = basis.boys + row * RCG_BOYS_NCOL + mo;
                    double f = __ldg(r + 8);
                    f = fma(f, d * (1.0 / 8.0), __ldg(r + 7));
                    f = fma(f, d * (1.0 / 7.0), __ldg(r + 6));
                    f = fma(f, d * (1.0 / 6.0), __ldg(r + 5));
                    f = fma(f, d * (1.0 / 5.0), __ldg(r + 4));
                    f = fma(f, d * (1.0 / 4.0), __ldg(r + 3));
                    f = fma(f, d * (1.0 / 3.0), __ldg(r + 2));
                    f = fma(f, d * (1.0 / 2.0), __ldg(r + 1));
                    f = fma(f, d, __ldg(r));
                    Bt[mo * nE] = f * pr.pref;
                }
            } else if (L0 == 0) {
                double f = 0.5 * sqrt(RCG_PI / pr.T) * pr.pref;
                const double r2 = 0.5 / pr.T, eTs = exp(-pr.T) * pr.pref;
                Bt[0] = f;
                for (int m = 0; m < M; ++m) {
                    f = ((double)(2 * m + 1) * f - eTs) * r2;
                    Bt[(m + 1) * nE] = f;
                }
            }
        }
        const double w1 = 2.0 * al, w2 = 2.0 * be, w3 = 2.0 * ga;
        GRAD_GSYNC();
        // bra levels: Eq. (2) with c = 0 on the first non-zero axis; a warp per row m, a lane per component
        for (int n = 0; n < E; ++n) {
            const int nc = d_ncart(n + 1), rows = M - n, c0 = d_ncum(n);
            for (int m = lwarp; m < rows; m += NWg) {
                double *b0 = Bt + m * nE;
                for (int j = L0; j < nc; j += LS) {
                    const int2 br = brarec[c0 + j];
                    const int c1 = br.x & 0xffff, c2 = br.x >> 16, i = br.y & 0xff, n1 = br.y >> 8;
                    double v = fma(sel3(i, pr.PA[0], pr.PA[1], pr.PA[2]), b0[c1], sel3(i, pr.WP[0], pr.WP[1], pr.WP[2]) * b0[nE + c1]);
                    v = fma((double)n1 * pr.hz, fma(-pr.rz, b0[nE + c2], b0[c2]), v);      // n1 = 0: c2 = 0, a finite value times zero
                    b0[c0 + j] = v;
                }
            }
            GRAD_GSYNC();
        }
        // targets with f = 0
        for (int t = ltid; t < nE; t += NTg) {
            const double v = Bt[t];
            const int le = comp[t].w;
#pragma unroll
            for (int s = 0; s < 4; ++s) {
                const GradSet &g = P.set[s];
                if (g.flo == 0 && le >= g.elo && le <= g.ehi) {
                    const double w = s == 0 ? 1.0 : (s == 1 ? w1 : (s == 2 ? w2 : w3));
                    accg[g.base + (t - g.eoff)] = fma(w, v, accg[g.base + (t - g.eoff)]);
                }
            }
        }
        // ket levels: the mirror of Eq. (2) (R-KET) with the cross term e - 1_i; a warp per row (ket component, m), a lane per
        // bra component; the row's axis, source and destination rows and accumulator rows come from its record
        const double *prev = Bt, *prev2 = Bt;
        int r0 = 0;
        for (int f = 0; f < F; ++f) {
            double *cur = lvl0 + (f % 3) * P.lvlmax;
            const int nrow = d_ncart(f + 1) * (F - f), nEl = (f + 1 == F) ? P.nElast : nE;
            for (int r = lwarp; r < nrow; r += NWg) {
                const int4 ra = rowrec[2 * (r0 + r)], rb = rowrec[2 * (r0 + r) + 1];
                const int i = ra.w & 0xff, n1 = ra.w >> 8;
                const double *p0 = prev + ra.x, *p2 = prev2 + (ra.y < 0 ? 0 : ra.y);
                double *dst = cur + ra.z;
                const double qc = sel3(i, pr.QC[0], pr.QC[1], pr.QC[2]), wq = sel3(i, pr.WQ[0], pr.WQ[1], pr.WQ[2]);
                const double k1 = (double)n1 * pr.he;
                const double *ec = ecn + i * nE;
                const short *cr = crs + i * nE;
                const int none = (int)0x80000000;        // an offset may be negative (it includes -eoff): the sentinel is INT_MIN
                const bool hasacc = rb.x != none || rb.y != none || rb.z != none || rb.w != none;
                // two bra components per lane and iteration: independent dependency chains
                for (int e0 = L0; e0 < nEl; e0 += 2 * LS) {
                    const int e1 = e0 + LS < nEl ? e0 + LS : e0;           // the tail repeats e0 (same value stored twice, no second update)
                    const bool two = e0 + LS < nEl;
                    double v0 = fma(qc, p0[e0], wq * p0[nE + e0]), v1 = fma(qc, p0[e1], wq * p0[nE + e1]);
                    if (n1 > 0) {
                        v0 = fma(k1, fma(-pr.re, p2[nE + e0], p2[e0]), v0);
                        v1 = fma(k1, fma(-pr.re, p2[nE + e1], p2[e1]), v1);
                    }
                    v0 = fma(ec[e0] * pr.hze, p0[nE + cr[e0]], v0);
                    v1 = fma(ec[e1] * pr.hze, p0[nE + cr[e1]], v1);
                    dst[e0] = v0;
                    dst[e1] = v1;
                    if (hasacc) {
#pragma unroll
                        for (int h = 0; h < 2; ++h) {
                            const int eidx = h ? e1 : e0;
                            const double v = h ? v1 : v0;
                            if (h && !two) break;
                            if (rb.x != none && (unsigned)(eidx - P.set[0].eoff) < (unsigned)P.set[0].nE) accg[rb.x + eidx] += v;
                            if (rb.y != none && (unsigned)(eidx - P.set[1].eoff) < (unsigned)P.set[1].nE) accg[rb.y + eidx] = fma(w1, v, accg[rb.y + eidx]);
                            if (rb.z != none && (unsigned)(eidx - P.set[2].eoff) < (unsigned)P.set[2].nE) accg[rb.z + eidx] = fma(w2, v, accg[rb.z + eidx]);
                            if (rb.w != none && (unsigned)(eidx - P.set[3].eoff) < (unsigned)P.set[3].nE) accg[rb.w + eidx] = fma(w3, v, accg[rb.w + eidx]);
                        }
                    }
                }
            }
            GRAD_GSYNC();
            r0 += nrow;
            prev2 = prev; prev = cur;
        }
    }

    // ------------------------------------------------------------------ Phase 2
    if (GROUPED) {                     // mode 1: sum the groups' accumulator sets into the first
        __syncthreads();
        for (int t = tid; t < P.acc_doubles; t += NT) {
            double v = acc[t];
            for (int g2 = 1; g2 < G; ++g2) v += acc[g2 * P.acc_doubles + t];
            acc[t] = v;
        }
    }
#define GRAD_P2SYNC() do { if (SUBQ) __syncwarp(); else __syncthreads(); } while (0)
    double *bin = cst, *pwAB = cst + 36, *pwCD = cst + 54;
    for (int t = tid2; t < 36; t += NT2) {
        const int n = t / 6, k = t - 6 * n;
        double b = 0.0;
        if (k <= n) { b = 1.0; for (int j = 1; j <= k; ++j) b = b * (double)(n - k + j) / (double)j; }
        bin[t] = b;
    }
    if (tid2 < 3) {
        const double ab = sel3(tid2, A[0], A[1], A[2]) - sel3(tid2, B[0], B[1], B[2]), cd = sel3(tid2, C[0], C[1], C[2]) - sel3(tid2, D[0], D[1], D[2]);
        double x = 1.0, y = 1.0;
        for (int k = 0; k < 6; ++k) { pwAB[tid2 * 6 + k] = x; pwCD[tid2 * 6 + k] = y; x *= ab; y *= cd; }
    }
    double *bufX = work, *bufR = bufX + P.p2x, *bufL = bufR + P.p2r, *bufD = bufL + P.p2l;
    const int la = P.l[0], lb = P.l[1], lc = P.l[2], ld = P.l[3];
    const int nsa = 2 * la + 1, nsb = 2 * lb + 1, nsc = 2 * lc + 1, nsd = 2 * ld + 1;
    const int nsph = nsa * nsb * nsc * nsd;
    double *outq = out + (size_t)q * 12 * nsph;
    GRAD_P2SYNC();
    for (int p = 0; p < 3; ++p) {
        // horizontal recurrences of the raised (source: the weighted set p + 1) and the lowered class (the plain set)
        for (int up = 1; up >= 0; --up) {
            const int sh1 = up ? 1 : -1;
            const int l1 = la + (p == 0 ? sh1 : 0), l2 = lb + (p == 1 ? sh1 : 0), l3 = lc + (p == 2 ? sh1 : 0), l4 = ld;
            if (l1 < 0 || l2 < 0 || l3 < 0) continue;                  // uniform: no lowered class of an s shell
            const GradSet &g = P.set[up ? p + 1 : 0];
            const int n1 = d_ncart(l1), n2 = d_ncart(l2), n3 = d_ncart(l3), n4 = d_ncart(l4);
            const int f0 = d_ncum(l3 - 1), nfr = d_ncum(l3 + l4) - f0, ldf = nfr | 1;
            const int c1o = d_ncum(l1 - 1), c2o = d_ncum(l2 - 1), c3o = f0, c4o = d_ncum(l4 - 1);
            double *Y = up ? bufR : bufL;
            {   // bra side: a warp per (a, b) pair, a lane per ket target
                const int np = (nfr + LS - 1) / LS;
                for (int u = warp2; u < n1 * n2 * np; u += NW2) {
                    const int ab = u / np, fi = (u - ab * np) * LS + L0;
                    const int ia = ab / n2, ib = ab - ia * n2;
                    const double *src = (SUBQ ? accg : acc) + g.base + (f0 + min(fi, nfr - 1) - g.foff) * g.ldE - g.eoff;
                    const double v = hrr_sum(comp[c1o + ia], comp[c2o + ib], l1, bin, pwAB, [&](int e) { return src[e]; });
                    if (fi < nfr) bufX[ab * ldf + fi] = v;
                }
            }
            GRAD_P2SYNC();
            {   // ket side: a warp per (c, d) pair, a lane per (a, b) pair
                const int nab = n1 * n2, np = (nab + LS - 1) / LS, n34 = n3 * n4;
                for (int u = warp2; u < n34 * np; u += NW2) {
                    const int cd = u / np, ab = (u - cd * np) * LS + L0;
                    const int ic = cd / n4, id = cd - ic * n4;
                    const double *src = bufX + min(ab, nab - 1) * ldf - f0;
                    const double v = hrr_sum(comp[c3o + ic], comp[c4o + id], l3, bin, pwCD, [&](int e) { return src[e]; });
                    if (ab < nab) Y[ab * n34 + cd] = v;
                }
            }
            GRAD_P2SYNC();
        }
        const int lp = P.l[p];
        const int nca = d_ncart(la), ncb = d_ncart(lb), ncc = d_ncart(lc), ncd = d_ncart(ld);
        const int ncblk = nca * ncb * ncc * ncd;
        // the raised / lowered blocks have ncart(lp + 1) / ncart(lp - 1) components at position p
        const int nup = d_ncart(lp + 1), ndn = lp > 0 ? d_ncart(lp - 1) : 1;
        const int dR1 = p == 1 ? nup : ncb, dR2 = p == 2 ? nup : ncc, dL1 = p == 1 ? ndn : ncb, dL2 = p == 2 ? ndn : ncc;
        const int cpo = d_ncum(lp - 1), cpu = d_ncum(lp), cpd = lp > 0 ? d_ncum(lp - 2) : 0;
        const float rcd = 1.0f / (float)ncd, rcc = 1.0f / (float)ncc, rcb = 1.0f / (float)ncb;
        for (int ax = 0; ax < 3; ++ax) {
            for (int t = tid2; t < ncblk; t += NT2) {
                int i3, i2, i1;
                int r = rcg_divmod(t, ncd, rcd, i3);
                r = rcg_divmod(r, ncc, rcc, i2);
                const int i0 = rcg_divmod(r, ncb, rcb, i1);
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
            GRAD_P2SYNC();
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
                const double *T = c2s + rcg_grad_c2s_off[lk];
                const int total = outer * ns * inner;
                const float rin = 1.0f / (float)inner, rns = 1.0f / (float)ns;
                for (int t = tid2; t < total; t += NT2) {
                    int in, ms;
                    const int r = rcg_divmod(t, inner, rin, in);
                    const int o = rcg_divmod(r, ns, rns, ms);
                    const double *s0 = src + (o * ncx) * inner + in;
                    const double *Tr = T + ms * ncx;
                    double s;
                    switch (lk) {
                    case 0: s = s0[0]; break;
                    case 1: s = c2s_dot<3>(Tr, s0, inner); break;
                    case 2: s = c2s_dot<6>(Tr, s0, inner); break;
                    case 3: s = c2s_dot<10>(Tr, s0, inner); break;
                    default: s = c2s_dot<15>(Tr, s0, inner); break;
                    }
                    if (k < 3) dst[t] = s;
                    else {          // t = ((ma nsb + mb) nsc + mc) nsd + md in the kernel's order: to the caller's layout and centre numbering
                        int mc2, mb2;
                        const int oab = rcg_divmod(o, nsc, 1.0f / (float)nsc, mc2);
                        const int ma2 = rcg_divmod(oab, nsb, 1.0f / (float)nsb, mb2);
                        const int ot = ma2 * P.ostr[0] + mb2 * P.ostr[1] + mc2 * P.ostr[2] + ms * P.ostr[3];
                        if (valid && mine) {
                            outq[(3 * P.col[p] + ax) * nsph + ot] = s;
                            double *od = outq + (3 * P.col[3] + ax) * nsph + ot;
                            *od = p == 0 ? -s : *od - s;
                        }
                    }
                }
                dims[k] = ns;
                GRAD_P2SYNC();
                double *tmp = src; src = dst; dst = tmp;
            }
        }
    }
    }          // quartets of the block (one, except in mode 3)
}

// ---------------------------------------------------------------- host side
// The kernel's horizontal recurrences move angular momentum from the first to the second shell of a pair: with the lighter shell first
// (an (sf| pair: three steps up from s with |AB|^3) their cancellation costs digits -- (sf|sg) derivatives measured 3.6e-6 of the quartet
// scale from the long-double value, the FP64 oracle in that order 6.5e-6.  So the heavier shell of each pair takes the first position
// (as the integral classes' canonical order does) and the result is written in the caller's layout and centre numbering.
static void grad_plan_for(const int l[4], long long k4max, GradPlan &P)
{
    const bool sb = l[0] < l[1], sk = l[2] < l[3];
    const int col[4] = {sb ? 1 : 0, sb ? 0 : 1, sk ? 3 : 2, sk ? 2 : 3};
    const int lk[4] = {l[col[0]], l[col[1]], l[col[2]], l[col[3]]};
    grad_plan(lk, k4max, P);
    int cstr[4];
    cstr[3] = 1; cstr[2] = 2 * l[3] + 1; cstr[1] = cstr[2] * (2 * l[2] + 1); cstr[0] = cstr[1] * (2 * l[1] + 1);
    for (int k = 0; k < 4; ++k) { P.col[k] = col[k]; P.ostr[k] = cstr[col[k]]; }
}

bool rcg_grad_supported(const int l[4], size_t *smem_bytes)
{
    for (int k = 0; k < 4; ++k)
        if (l[k] < 0 || l[k] > RCG_LMAX) return false;
    GradPlan P;
    grad_plan_for(l, 1, P);
    if (smem_bytes) *smem_bytes = sizeof(double) * (size_t)P.smem_doubles;
    return P.M <= 16 && P.E <= RCG_GRAD_LEVELS && P.F <= RCG_GRAD_LEVELS && sizeof(double) * (size_t)P.smem_doubles <= GRAD_SMEM_LIMIT;      // mode 3 included
}

cudaError_t rcg_grad_launch(const RcgGradLaunch &a)
{
    GradPlan P;
    grad_plan_for(a.l, a.k4max, P);
    static RcgOnce once;
    int nsm = 0;
    cudaError_t e = rcg_prepare_kernel(once, (const void *)rcg_eri_grad_kernel<0>, GRAD_SMEM_LIMIT, &nsm);
    if (e != cudaSuccess) return e;
    static RcgOnce once1, once2, once3;
    if ((e = rcg_prepare_kernel(once3, (const void *)rcg_eri_grad_kernel<3>, GRAD_SMEM_LIMIT, &nsm)) != cudaSuccess) return e;
    if ((e = rcg_prepare_kernel(once1, (const void *)rcg_eri_grad_kernel<1>, 72 * 1024, &nsm)) != cudaSuccess) return e;
    if ((e = rcg_prepare_kernel(once2, (const void *)rcg_eri_grad_kernel<2>, GRAD_SMEM_LIMIT, &nsm)) != cudaSuccess) return e;
    const size_t smem = sizeof(double) * (size_t)P.smem_doubles;
    const size_t nout = 12 * (size_t)(2 * a.l[0] + 1) * (2 * a.l[1] + 1) * (2 * a.l[2] + 1) * (2 * a.l[3] + 1);
    if (P.mode == 3) {          // one persistent block per SM, scratch from the library's stream-ordered pool (freed stream-ordered after the launch)
        const unsigned grid = (unsigned)(a.n < nsm ? a.n : nsm);
        void *scr = nullptr;
        if ((e = rcg_pool_alloc(&scr, sizeof(double) * (size_t)P.scratch_doubles * grid, a.stream)) != cudaSuccess) return e;
        rcg_eri_grad_kernel<3><<<grid, GRAD_MAX_THREADS, smem, a.stream>>>(a.basis, a.quartets, a.n, a.out, (double *)scr, P);
        e = cudaGetLastError();
        const cudaError_t e2 = cudaFreeAsync(scr, a.stream);
        return e != cudaSuccess ? e : e2;
    }
    // a light class of a basis WITH deep contractions, no K4 promise: the list may mix K4 = 1 and K4 = 10^4 quartets.  Two launches over
    // the same list: the sub-warp groups (mode 2) take the quartets below 256 primitive quartets, the primitive groups (mode 1) the others;
    // a quartet of the other kind costs a group a few loads, a block an early exit
    if (P.mode == 1 && !a.k4_promised) {
        GradPlan P2;
        grad_plan_for(a.l, 1, P2);
        if (P2.mode == 2) {
            P2.k4_hi = 256; P.k4_lo = 256;
            const int64_t pb = GRAD_MAX_THREADS / P2.sub;
            const size_t smem2 = sizeof(double) * (size_t)P2.smem_doubles;
            if (a.n > (int64_t)0x7fffffff) return cudaErrorInvalidValue;
            rcg_eri_grad_kernel<2><<<(unsigned)((a.n + pb - 1) / pb), GRAD_MAX_THREADS, smem2, a.stream>>>(a.basis, a.quartets, a.n, a.out, nullptr, P2);
            if ((e = cudaGetLastError()) != cudaSuccess) return e;
        }
    }
    const int64_t per_block = P.mode == 2 ? GRAD_MAX_THREADS / P.sub : 1;
    const int64_t maxq = (int64_t)(0x7fffffff / 64) * per_block;         // quartets per launch
    for (int64_t q0 = 0; q0 < a.n; q0 += maxq) {
        const int64_t qn = a.n - q0 < maxq ? a.n - q0 : maxq;
        const unsigned grid = (unsigned)((qn + per_block - 1) / per_block);
        const int32_t *ql = a.quartets + 4 * q0;
        double *ol = a.out + nout * (size_t)q0;
        if (P.mode == 2) rcg_eri_grad_kernel<2><<<grid, GRAD_MAX_THREADS, smem, a.stream>>>(a.basis, ql, qn, ol, nullptr, P);
        else if (P.mode == 1) rcg_eri_grad_kernel<1><<<grid, P.groups * 32, smem, a.stream>>>(a.basis, ql, qn, ol, nullptr, P);
        else rcg_eri_grad_kernel<0><<<grid, P.threads, smem, a.stream>>>(a.basis, ql, qn, ol, nullptr, P);
        if ((e = cudaGetLastError()) != cudaSuccess) return e;
    }
    return cudaSuccess;
}
