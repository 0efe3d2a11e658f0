/*
 * eri_grad_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, FP64 CPU oracle for the FIRST DERIVATIVES of contracted real-spherical electron repulsion
 * integrals (ab|cd) with respect to the four shell centres A, B, C, D (PAPER.md:299
 * "first-derivative variants", :401; the scheme is that of the Head-Gordon-Pople reference PAPER.md:409).
 *
 * Definition written out.  A primitive Cartesian Gaussian x_A^ax y_A^ay z_A^az exp(-alpha r_A^2) depends on its
 * centre only through r_A = r - A, so
 *     d/dA_i [a| = 2 alpha [a + 1_i| - a_i [a - 1_i|                                       (reading R-GRAD)
 * and the same for b (beta, B), c (gamma, C), d (delta, D).  The Cartesian-to-spherical matrices of Eq. (8)
 * do not depend on the centre, so the derivative of a spherical component is the transform of the
 * derivatives of the Cartesian ones.  Per primitive quartet the shifted Cartesian integrals come from the vertical
 * recurrence Eq. (2) and the horizontal recurrence Eq. (3) (:82-87) exactly as in eri_oracle.c's mode 1;
 * contraction (Eq. (1), :59-61) is last, then the dense transform Eq. (17) (:235).  ALL TWELVE components are computed
 * from the definition -- translational invariance (their sum over the centres vanishes) is a pin, not an input.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may call this file.  It shares no code, tables or
 * headers with the CUDA path.  orc_boys and orc_c2s_matrix are eri_oracle.c's (pinned there); the recursions are restated
 * here with the larger index ranges the shifted shells need.  Pins: tests/test_oracle_grad_pins.py (finite differences of
 * the pinned integral oracle, closed form of the (ss|ss) derivative, translational invariance, permutations).
 *
 * out: [n][12][2la+1][2lb+1][2lc+1][2ld+1], derivative index 3 * centre + axis (centre 0..3 = a, b, c, d of the
 * quartet's columns; axis 0..2 = x, y, z).
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <stdint.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define GLMAX 4                    /* max shell angular momentum */
#define GE (2 * GLMAX + 1)         /* max one-side VRR angular momentum (one shell raised) */
#define GM (4 * GLMAX + 1)         /* max Boys order */
#define GNC 220                    /* #Cartesian triples with |a| <= 9 : C(12,3) */

void orc_boys(int mmax, double T, double *F);
void orc_c2s_matrix(int l, double *T);

static const double G_PI = 3.14159265358979323846264338327950288;

static int g_ncart(int l) { return (l + 1) * (l + 2) / 2; }

/* component order of one level (R-SPH): for i=l..0: for j=l-i..0: x^i y^j z^(l-i-j) */
static void g_cart_list(int l, int (*c)[3])
{
    int n = 0;
    for (int i = l; i >= 0; --i)
        for (int j = l - i; j >= 0; --j) { c[n][0] = i; c[n][1] = j; c[n][2] = l - i - j; ++n; }
}

static int g_tri_index(const int *a)
{
    int l = a[0] + a[1] + a[2], k = l - a[0];
    return l * (l + 1) * (l + 2) / 6 + k * (k + 1) / 2 + (l - a[0] - a[1]);
}

typedef struct {
    double PA[3], WP[3], QC[3], WQ[3];
    double zeta, eta, rho;
    double F[GM + 1];              /* [00|00]^(m) = S F_m(T) (R-BASE) */
    double *val;
    int *stamp;
    int cur;
} g_vrr_ctx;

/* [a0|c0]^(m), Eq. (2) PAPER.md:71-78 on the first non-zero axis, bra before ket (R-EQ2, R-KET) */
static double g_vrr(g_vrr_ctx *x, int *a, int *c, int m)
{
    if (a[0] < 0 || a[1] < 0 || a[2] < 0 || c[0] < 0 || c[1] < 0 || c[2] < 0) return 0.0;
    int la = a[0] + a[1] + a[2], lc = c[0] + c[1] + c[2];
    if (la == 0 && lc == 0) return x->F[m];
    size_t key = ((size_t)g_tri_index(a) * GNC + g_tri_index(c)) * (GM + 1) + m;
    if (x->stamp[key] == x->cur) return x->val[key];
    double r;
    if (la > 0) {
        int i = a[0] > 0 ? 0 : (a[1] > 0 ? 1 : 2);
        a[i] -= 1;
        double ai = a[i], ci = c[i];
        r = x->PA[i] * g_vrr(x, a, c, m) + x->WP[i] * g_vrr(x, a, c, m + 1);
        if (a[i] > 0) {
            a[i] -= 1;
            r += ai / (2.0 * x->zeta) * (g_vrr(x, a, c, m) - x->rho / x->zeta * g_vrr(x, a, c, m + 1));
            a[i] += 1;
        }
        if (c[i] > 0) {
            c[i] -= 1;
            r += ci / (2.0 * (x->zeta + x->eta)) * g_vrr(x, a, c, m + 1);
            c[i] += 1;
        }
        a[i] += 1;
    } else {
        int i = c[0] > 0 ? 0 : (c[1] > 0 ? 1 : 2);
        c[i] -= 1;
        double ci = c[i];
        r = x->QC[i] * g_vrr(x, a, c, m) + x->WQ[i] * g_vrr(x, a, c, m + 1);
        if (c[i] > 0) {
            c[i] -= 1;
            r += ci / (2.0 * x->eta) * (g_vrr(x, a, c, m) - x->rho / x->eta * g_vrr(x, a, c, m + 1));
            c[i] += 1;
        }
        c[i] += 1;
    }
    x->val[key] = r;
    x->stamp[key] = x->cur;
    return r;
}

/* primitive Cartesian (ab|cd) by Eq. (3) PAPER.md:84 down to [a0|c0]; an index below zero gives 0 */
static double g_hrr(g_vrr_ctx *x, const double *AB, const double *CD, int *a, int *b, int *c, int *d)
{
    for (int i = 0; i < 3; ++i)
        if (a[i] < 0 || b[i] < 0 || c[i] < 0 || d[i] < 0) return 0.0;
    for (int i = 0; i < 3; ++i)
        if (b[i] > 0) {
            b[i] -= 1; a[i] += 1;
            double hi = g_hrr(x, AB, CD, a, b, c, d);
            a[i] -= 1;
            double lo = g_hrr(x, AB, CD, a, b, c, d);
            b[i] += 1;
            return hi + AB[i] * lo;
        }
    for (int i = 0; i < 3; ++i)
        if (d[i] > 0) {
            d[i] -= 1; c[i] += 1;
            double hi = g_hrr(x, AB, CD, a, b, c, d);
            c[i] -= 1;
            double lo = g_hrr(x, AB, CD, a, b, c, d);
            d[i] += 1;
            return hi + CD[i] * lo;
        }
    return g_vrr(x, a, c, 0);
}

static void grad_quartet(const int *l, const int *K, const double *const *ex, const double *const *co,
                         const double *const *R, double *out, double *val, int *stamp, int *gen,
                         double *cart, double *tmp)
{
    int nc4[4] = {g_ncart(l[0]), g_ncart(l[1]), g_ncart(l[2]), g_ncart(l[3])};
    int comps[4][15][3];
    for (int t = 0; t < 4; ++t) g_cart_list(l[t], comps[t]);
    size_t nblk = (size_t)nc4[0] * nc4[1] * nc4[2] * nc4[3];
    int L = l[0] + l[1] + l[2] + l[3] + 1;
    double AB[3], CD[3], AB2 = 0, CD2 = 0;
    for (int i = 0; i < 3; ++i) {
        AB[i] = R[0][i] - R[1][i]; CD[i] = R[2][i] - R[3][i];
        AB2 += AB[i] * AB[i]; CD2 += CD[i] * CD[i];
    }
    for (size_t k = 0; k < 12 * nblk; ++k) cart[k] = 0.0;
    g_vrr_ctx x;
    x.val = val; x.stamp = stamp;
    for (int i0 = 0; i0 < K[0]; ++i0)
    for (int i1 = 0; i1 < K[1]; ++i1)
    for (int i2 = 0; i2 < K[2]; ++i2)
    for (int i3 = 0; i3 < K[3]; ++i3) {
        double xp[4] = {ex[0][i0], ex[1][i1], ex[2][i2], ex[3][i3]};   /* alpha, beta, gamma, delta */
        double zeta = xp[0] + xp[1], eta = xp[2] + xp[3], rho = zeta * eta / (zeta + eta);
        double PQ2 = 0;
        for (int t = 0; t < 3; ++t) {                                   /* Gaussian-pair quantities (R-PAIR) */
            double P = (xp[0] * R[0][t] + xp[1] * R[1][t]) / zeta;
            double Q = (xp[2] * R[2][t] + xp[3] * R[3][t]) / eta;
            double W = (zeta * P + eta * Q) / (zeta + eta);
            PQ2 += (P - Q) * (P - Q);
            x.PA[t] = P - R[0][t]; x.WP[t] = W - P;
            x.QC[t] = Q - R[2][t]; x.WQ[t] = W - Q;
        }
        double S = 2.0 * pow(G_PI, 2.5) / (zeta * eta * sqrt(zeta + eta)) *
                   exp(-xp[0] * xp[1] * AB2 / zeta) * exp(-xp[2] * xp[3] * CD2 / eta);
        double cf = co[0][i0] * co[1][i1] * co[2][i2] * co[3][i3];
        x.zeta = zeta; x.eta = eta; x.rho = rho;
        orc_boys(L, rho * PQ2, x.F);
        for (int m = 0; m <= L; ++m) x.F[m] *= S;
        *gen += 1;
        if (*gen == 0x7fffffff) { memset(stamp, 0, sizeof(int) * (size_t)GNC * GNC * (GM + 1)); *gen = 1; }
        x.cur = *gen;
        size_t n = 0;
        for (int p = 0; p < nc4[0]; ++p) for (int q = 0; q < nc4[1]; ++q)
        for (int r = 0; r < nc4[2]; ++r) for (int s = 0; s < nc4[3]; ++s, ++n) {
            int idx[4][3];
            for (int i = 0; i < 3; ++i) {
                idx[0][i] = comps[0][p][i]; idx[1][i] = comps[1][q][i];
                idx[2][i] = comps[2][r][i]; idx[3][i] = comps[3][s][i];
            }
            for (int cen = 0; cen < 4; ++cen)
                for (int ax = 0; ax < 3; ++ax) {
                    int pw = idx[cen][ax];
                    idx[cen][ax] = pw + 1;
                    double up = g_hrr(&x, AB, CD, idx[0], idx[1], idx[2], idx[3]);
                    idx[cen][ax] = pw - 1;
                    double dn = pw > 0 ? g_hrr(&x, AB, CD, idx[0], idx[1], idx[2], idx[3]) : 0.0;
                    idx[cen][ax] = pw;
                    cart[(size_t)(3 * cen + ax) * nblk + n] += cf * (2.0 * xp[cen] * up - pw * dn);
                }
        }
    }
    /* dense c2s of every component block, one index at a time, Eq. (17) */
    size_t nsph_all = (size_t)(2 * l[0] + 1) * (2 * l[1] + 1) * (2 * l[2] + 1) * (2 * l[3] + 1);
    for (int g = 0; g < 12; ++g) {
        int dims[4] = {nc4[0], nc4[1], nc4[2], nc4[3]};
        double *src = cart + (size_t)g * nblk, *dst = tmp;
        double *bufs[2] = {tmp, tmp + nblk};
        int which = 0;
        for (int ax = 0; ax < 4; ++ax) {
            int lx = l[ax], nsph = 2 * lx + 1, ncx = dims[ax];
            double Tm[9 * 15];
            orc_c2s_matrix(lx, Tm);
            size_t outer = 1, inner = 1;
            for (int t = 0; t < ax; ++t) outer *= dims[t];
            for (int t = ax + 1; t < 4; ++t) inner *= dims[t];
            dst = bufs[which]; which ^= 1;
            for (size_t o = 0; o < outer; ++o)
                for (int ms = 0; ms < nsph; ++ms)
                    for (size_t in = 0; in < inner; ++in) {
                        double s = 0.0;
                        for (int k = 0; k < ncx; ++k) s += Tm[ms * ncx + k] * src[(o * ncx + k) * inner + in];
                        dst[(o * nsph + ms) * inner + in] = s;
                    }
            dims[ax] = nsph;
            src = dst;
        }
        memcpy(out + (size_t)g * nsph_all, src, nsph_all * sizeof(double));
    }
}

/* batch entry: every quartet of the list belongs to the angular class of quartet 0.  Returns 0, or -1 on a class
 * mismatch / l > 4. */
int orc_eri_grad_batch(int nshell, const int32_t *shell_l, const int32_t *prim_off, const double *exps,
                       const double *coefs, const double *centers, const int32_t *quartets, int64_t n,
                       int nthreads, double *out)
{
    if (n <= 0) return 0;
    int l[4];
    for (int t = 0; t < 4; ++t) {
        int s = quartets[t];
        if (s < 0 || s >= nshell) return -1;
        l[t] = shell_l[s];
        if (l[t] < 0 || l[t] > GLMAX) return -1;
    }
    for (int64_t q = 0; q < n; ++q)
        for (int t = 0; t < 4; ++t) {
            int s = quartets[4 * q + t];
            if (s < 0 || s >= nshell || shell_l[s] != l[t]) return -1;
        }
    size_t nout = 12 * (size_t)(2 * l[0] + 1) * (2 * l[1] + 1) * (2 * l[2] + 1) * (2 * l[3] + 1);
    size_t nblk = (size_t)g_ncart(l[0]) * g_ncart(l[1]) * g_ncart(l[2]) * g_ncart(l[3]);
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
    #pragma omp parallel
    {
        size_t nm = (size_t)GNC * GNC * (GM + 1);
        double *val = (double *)malloc(nm * sizeof(double));
        int *stamp = (int *)calloc(nm, sizeof(int));
        double *cart = (double *)malloc(12 * nblk * sizeof(double));
        double *tmp = (double *)malloc(2 * nblk * sizeof(double));
        int gen = 0;
        #pragma omp for schedule(dynamic, 1)
        for (int64_t q = 0; q < n; ++q) {
            int K[4];
            const double *ex[4], *co[4], *R[4];
            for (int t = 0; t < 4; ++t) {
                int s = quartets[4 * q + t];
                K[t] = prim_off[s + 1] - prim_off[s];
                ex[t] = exps + prim_off[s]; co[t] = coefs + prim_off[s]; R[t] = centers + 3 * s;
            }
            grad_quartet(l, K, ex, co, R, out + nout * q, val, stamp, &gen, cart, tmp);
        }
        free(val); free(stamp); free(cart); free(tmp);
    }
    return 0;
}
