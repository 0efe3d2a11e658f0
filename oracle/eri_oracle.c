/*
 * eri_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, FP64 CPU oracle for contracted real-spherical electron repulsion
 * integrals (ab|cd) by the Head-Gordon-Pople scheme as PAPER.md states it
 * (Eq. (1), VRR Eq. (2) :69-80, HRR Eq. (3) :82-87, c2s Eq. (8) :183-191,
 * conventional "materialise-then-transform" order Eq. (17) :235, Alg. 2 :269-283).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may call this file.  It shares no code, tables or headers with the CUDA path
 * (paper_2605_10312_b200/csrc) or with the kernel generator.
 *
 * Routes (all give the same numbers up to rounding):
 *   orc_eri_quartet(mode=0)  HGP: memoised recursive Obara-Saika VRR per primitive quartet,
 *                            contraction of [e0|f0], HRR on contracted integrals, dense c2s.
 *   orc_eri_quartet(mode=1)  "definitional": VRR + HRR per primitive quartet, contraction last.
 *   orc_eri_quartet_md       independent McMurchie-Davidson evaluation (tiny inputs).
 * Pins: see tests/test_oracle_*.py (Boys table, closed forms, golden ERIs, symmetries,
 * invariances, MD cross-check).  Readings of the paper (R-PAIR, R-BASE, R-EQ2, R-KET,
 * R-HRRK, R-SPH, R-PRIM, R-CONTR) are listed in DESIGN.md.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <stdint.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define LMAX 4                 /* max shell angular momentum */
#define EMAX (2 * LMAX)        /* max one-side VRR angular momentum */
#define MMAX (4 * LMAX)        /* max Boys order */
#define NC1 165                /* #Cartesian triples with |a| <= 8 : C(11,3) */

static const double PI = 3.14159265358979323846264338327950288;

static int ncart(int l) { return (l + 1) * (l + 2) / 2; }

/* ---------------------------------------------------------------- Boys function
 * F_m(T) = int_0^1 t^{2m} exp(-T t^2) dt   (PAPER.md:69 names it [00|00]^(m); R-BOYS).
 * T < 35 : F_m = e^{-T} sum_{i>=0} (2T)^i / ((2m+1)(2m+3)...(2m+2i+1)), each m separately.
 * T >= 35: F_0 = 1/2 sqrt(pi/T) erf(sqrt T), upward F_{m+1} = ((2m+1) F_m - e^{-T}) / (2T). */
void orc_boys(int mmax, double T, double *F)
{
    if (T < 35.0) {
        double eT = exp(-T);
        for (int m = 0; m <= mmax; ++m) {
            double term = 1.0 / (2 * m + 1), sum = term;
            for (int i = 1; i < 2000; ++i) {
                term *= 2.0 * T / (2 * m + 2 * i + 1);
                sum += term;
                if (term < 1e-18 * sum) break;
            }
            F[m] = eT * sum;
        }
    } else {
        double eT = exp(-T);
        F[0] = 0.5 * sqrt(PI / T) * erf(sqrt(T));
        for (int m = 0; m < mmax; ++m) F[m + 1] = ((2 * m + 1) * F[m] - eT) / (2.0 * T);
    }
}

/* ---------------------------------------------------------------- Cartesian components
 * order for one l (R-SPH): for i=l..0: for j=l-i..0: x^i y^j z^(l-i-j). */
static void cart_list(int l, int (*c)[3])
{
    int n = 0;
    for (int i = l; i >= 0; --i)
        for (int j = l - i; j >= 0; --j) { c[n][0] = i; c[n][1] = j; c[n][2] = l - i - j; ++n; }
}

/* rank of a triple among ALL triples with |a| <= 8 (levels in order, then cart_list order) */
static int tri_index(const int *a)
{
    int l = a[0] + a[1] + a[2];
    int off = l * (l + 1) * (l + 2) / 6;
    int i = a[0], j = a[1];
    /* position inside level: sum_{i'=l..i+1} (l-i'+1) + (l-i-j) */
    int k = l - i;
    return off + k * (k + 1) / 2 + (l - i - j);
}

/* ---------------------------------------------------------------- real solid harmonics
 * Racah-normalised S_lm, rows m=-l..l, closed form of R-SPH (SURVEY/DESIGN):
 * S_lm = N_lm sum_t sum_u sum_v C_tuv x^(2t+|m|-2(u+v)) y^(2(u+v)) z^(l-2t-|m|). */
static double binom(int n, int k)
{
    if (k < 0 || k > n) return 0.0;
    double r = 1.0;
    for (int i = 1; i <= k; ++i) r = r * (n - k + i) / i;
    return r;
}
static double fact(int n) { double r = 1.0; for (int i = 2; i <= n; ++i) r *= i; return r; }

/* T[(2l+1) x ncart(l)], row-major */
void orc_c2s_matrix(int l, double *T)
{
    int nc = ncart(l);
    int comps[45][3];
    cart_list(l, comps);
    memset(T, 0, sizeof(double) * (2 * l + 1) * nc);
    for (int m = -l; m <= l; ++m) {
        int am = m < 0 ? -m : m;
        double N = 1.0 / (pow(2.0, am) * fact(l)) *
                   sqrt(2.0 * fact(l + am) * fact(l - am) / (m == 0 ? 2.0 : 1.0));
        for (int t = 0; t <= (l - am) / 2; ++t)
            for (int u = 0; u <= t; ++u) {
                /* twov = 2v : even for m>=0 (v=0,1,..), odd for m<0 (v=1/2,3/2,..) */
                for (int twov = (m < 0 ? 1 : 0); twov <= am; twov += 2) {
                    int vint = (twov - (m < 0 ? 1 : 0)) / 2;          /* v - v_m */
                    double C = ((t + vint) % 2 ? -1.0 : 1.0) * pow(0.25, t) * binom(l, t) *
                               binom(l - t, am + t) * binom(t, u) * binom(am, twov);
                    int px = 2 * t + am - (2 * u + twov), py = 2 * u + twov, pz = l - 2 * t - am;
                    for (int k = 0; k < nc; ++k)
                        if (comps[k][0] == px && comps[k][1] == py && comps[k][2] == pz)
                            T[(m + l) * nc + k] += N * C;
                }
            }
    }
}

/* ---------------------------------------------------------------- primitive-quartet context */
typedef struct {
    double PA[3], WP[3], QC[3], WQ[3];
    double zeta, eta, rho;
    double F[MMAX + 1];          /* [00|00]^(m) = S * F_m(T)   (R-BASE) */
    double *val;                 /* memo [NC1][NC1][MMAX+1] */
    int *stamp;                  /* validity stamps */
    int cur;
} vrr_ctx;

/* [a0|c0]^(m) by memoised recursion; reduce FIRST non-zero axis, bra before ket.
 * bra step: Eq. (2) PAPER.md:71-78 (R-EQ2);  ket step: its mirror (R-KET). */
static double vrr(vrr_ctx *x, int *a, int *c, int m)
{
    if (a[0] < 0 || a[1] < 0 || a[2] < 0 || c[0] < 0 || c[1] < 0 || c[2] < 0) return 0.0;
    int la = a[0] + a[1] + a[2], lc = c[0] + c[1] + c[2];
    if (la == 0 && lc == 0) return x->F[m];
    size_t key = ((size_t)tri_index(a) * NC1 + tri_index(c)) * (MMAX + 1) + m;
    if (x->stamp[key] == x->cur) return x->val[key];
    double r;
    if (la > 0) {
        int i = a[0] > 0 ? 0 : (a[1] > 0 ? 1 : 2);
        a[i] -= 1;                                    /* a now is the lower index "a" of Eq. (2) */
        double ai = a[i], ci = c[i];
        r = x->PA[i] * vrr(x, a, c, m) + x->WP[i] * vrr(x, a, c, m + 1);
        if (a[i] > 0) {
            a[i] -= 1;
            r += ai / (2.0 * x->zeta) * (vrr(x, a, c, m) - x->rho / x->zeta * vrr(x, a, c, m + 1));
            a[i] += 1;
        }
        if (c[i] > 0) {
            c[i] -= 1;
            r += ci / (2.0 * (x->zeta + x->eta)) * vrr(x, a, c, m + 1);
            c[i] += 1;
        }
        a[i] += 1;
    } else {
        int i = c[0] > 0 ? 0 : (c[1] > 0 ? 1 : 2);
        c[i] -= 1;
        double ci = c[i];                              /* la == 0: no bra cross term */
        r = x->QC[i] * vrr(x, a, c, m) + x->WQ[i] * vrr(x, a, c, m + 1);
        if (c[i] > 0) {
            c[i] -= 1;
            r += ci / (2.0 * x->eta) * (vrr(x, a, c, m) - x->rho / x->eta * vrr(x, a, c, m + 1));
            c[i] += 1;
        }
        c[i] += 1;
    }
    x->val[key] = r;
    x->stamp[key] = x->cur;
    return r;
}

/* ---------------------------------------------------------------- HRR, Eq. (3)
 * (a,b+1i|c,d) = (a+1i,b|c,d) + (Ai-Bi)(a,b|c,d); ket analogue with C-D (R-HRRK).
 * Plain recursion down to base(a,c) = (a0|c0). */
typedef struct {
    const double *H;             /* [NC1][NC1] values (a0|c0) (only needed entries are filled) */
    double AB[3], CD[3];
} hrr_ctx;

static double hrr(const hrr_ctx *h, int *a, int *b, int *c, int *d)
{
    for (int i = 0; i < 3; ++i)
        if (b[i] > 0) {
            b[i] -= 1; a[i] += 1;
            double hi = hrr(h, a, b, c, d);
            a[i] -= 1;
            double lo = hrr(h, a, b, c, d);
            b[i] += 1;
            return hi + h->AB[i] * lo;
        }
    for (int i = 0; i < 3; ++i)
        if (d[i] > 0) {
            d[i] -= 1; c[i] += 1;
            double hi = hrr(h, a, b, c, d);
            c[i] -= 1;
            double lo = hrr(h, a, b, c, d);
            d[i] += 1;
            return hi + h->CD[i] * lo;
        }
    return h->H[(size_t)tri_index(a) * NC1 + tri_index(c)];
}

typedef struct { double *val; int *stamp; int gen; double *H; double *Hp; double *cart; double *tmp; } orc_work;

static orc_work *work_new(void)
{
    orc_work *w = (orc_work *)malloc(sizeof(orc_work));
    size_t n = (size_t)NC1 * NC1 * (MMAX + 1);
    w->val = (double *)malloc(n * sizeof(double));
    w->stamp = (int *)calloc(n, sizeof(int));
    w->gen = 0;
    w->H = (double *)malloc((size_t)NC1 * NC1 * sizeof(double));
    w->Hp = (double *)malloc((size_t)NC1 * NC1 * sizeof(double));
    w->cart = (double *)malloc((size_t)15 * 15 * 15 * 15 * sizeof(double));
    w->tmp = (double *)malloc((size_t)15 * 15 * 15 * 15 * sizeof(double));
    return w;
}
static void work_free(orc_work *w)
{
    free(w->val); free(w->stamp); free(w->H); free(w->Hp); free(w->cart); free(w->tmp); free(w);
}

/* triples for every level up to 8, in tri_index order; filled once by init_trip() */
static int trip[NC1][3];
static void init_trip(void)
{
    int n = 0;
    for (int lev = 0; lev <= EMAX; ++lev) { cart_list(lev, &trip[n]); n += ncart(lev); }
}

/* ---------------------------------------------------------------- one shell quartet
 * mode 0: Alg. 2 order: contract [e0|f0] over primitives, then HRR, then c2s.
 * mode 1: HRR applied per primitive quartet to full Cartesian (ab|cd), contraction last.
 * out: [nsph(la)][nsph(lb)][nsph(lc)][nsph(ld)], C order. */
static void eri_quartet(const int *l, const int *K, const double *const *ex, const double *const *co,
                        const double *const *R, int mode, double *out, orc_work *w)
{
    int la = l[0], lb = l[1], lc = l[2], ld = l[3];
    int L = la + lb + lc + ld;
    int na = ncart(la), nb = ncart(lb), nc = ncart(lc), nd = ncart(ld);
    int ca[15][3], cb[15][3], cc[15][3], cd[15][3];
    cart_list(la, ca); cart_list(lb, cb); cart_list(lc, cc); cart_list(ld, cd);
    size_t ncartall = (size_t)na * nb * nc * nd;
    const double *A = R[0], *B = R[1], *C = R[2], *D = R[3];
    hrr_ctx h;
    for (int i = 0; i < 3; ++i) { h.AB[i] = A[i] - B[i]; h.CD[i] = C[i] - D[i]; }
    double AB2 = 0, CD2 = 0;
    for (int i = 0; i < 3; ++i) { AB2 += h.AB[i] * h.AB[i]; CD2 += h.CD[i] * h.CD[i]; }

    /* index ranges of the VRR targets [e0|f0], e in [la,la+lb], f in [lc,lc+ld] */
    int e0 = la * (la + 1) * (la + 2) / 6, e1 = (la + lb + 1) * (la + lb + 2) * (la + lb + 3) / 6;
    int f0 = lc * (lc + 1) * (lc + 2) / 6, f1 = (lc + ld + 1) * (lc + ld + 2) * (lc + ld + 3) / 6;
    for (int ia = e0; ia < e1; ++ia)
        for (int ic = f0; ic < f1; ++ic) w->H[(size_t)ia * NC1 + ic] = 0.0;
    for (size_t k = 0; k < ncartall; ++k) w->cart[k] = 0.0;

    vrr_ctx x;
    x.val = w->val; x.stamp = w->stamp;
    for (int i = 0; i < K[0]; ++i)
    for (int j = 0; j < K[1]; ++j)
    for (int k = 0; k < K[2]; ++k)
    for (int m4 = 0; m4 < K[3]; ++m4) {
        /* Gaussian-pair quantities (R-PAIR) */
        double al = ex[0][i], be = ex[1][j], ga = ex[2][k], de = ex[3][m4];
        double zeta = al + be, eta = ga + de, rho = zeta * eta / (zeta + eta);
        double P[3], Q[3], W[3], PQ2 = 0;
        for (int t = 0; t < 3; ++t) {
            P[t] = (al * A[t] + be * B[t]) / zeta;
            Q[t] = (ga * C[t] + de * D[t]) / eta;
            W[t] = (zeta * P[t] + eta * Q[t]) / (zeta + eta);
            PQ2 += (P[t] - Q[t]) * (P[t] - Q[t]);
            x.PA[t] = P[t] - A[t]; x.WP[t] = W[t] - P[t];
            x.QC[t] = Q[t] - C[t]; x.WQ[t] = W[t] - Q[t];
        }
        double T = rho * PQ2;
        double S = 2.0 * pow(PI, 2.5) / (zeta * eta * sqrt(zeta + eta)) *
                   exp(-al * be * AB2 / zeta) * exp(-ga * de * CD2 / eta);
        double cf = co[0][i] * co[1][j] * co[2][k] * co[3][m4];
        x.zeta = zeta; x.eta = eta; x.rho = rho;
        orc_boys(L, T, x.F);
        for (int m = 0; m <= L; ++m) x.F[m] *= S;
        /* fresh memo generation for this primitive quartet */
        w->gen += 1;
        if (w->gen == 0x7fffffff) { memset(w->stamp, 0, sizeof(int) * (size_t)NC1 * NC1 * (MMAX + 1)); w->gen = 1; }
        x.cur = w->gen;
        double *Hdst = mode == 0 ? w->H : w->Hp;
        for (int ia = e0; ia < e1; ++ia)
            for (int ic = f0; ic < f1; ++ic) {
                int a[3] = {trip[ia][0], trip[ia][1], trip[ia][2]};
                int c[3] = {trip[ic][0], trip[ic][1], trip[ic][2]};
                double v = vrr(&x, a, c, 0);
                if (mode == 0) Hdst[(size_t)ia * NC1 + ic] += cf * v;       /* Alg. 2 line 7 */
                else           Hdst[(size_t)ia * NC1 + ic] = v;
            }
        if (mode == 1) {
            h.H = w->Hp;
            size_t n = 0;
            for (int p = 0; p < na; ++p) for (int q = 0; q < nb; ++q)
            for (int r = 0; r < nc; ++r) for (int s = 0; s < nd; ++s, ++n) {
                int a[3] = {ca[p][0], ca[p][1], ca[p][2]}, b[3] = {cb[q][0], cb[q][1], cb[q][2]};
                int c[3] = {cc[r][0], cc[r][1], cc[r][2]}, d[3] = {cd[s][0], cd[s][1], cd[s][2]};
                w->cart[n] += cf * hrr(&h, a, b, c, d);
            }
        }
    }
    if (mode == 0) {
        h.H = w->H;
        size_t n = 0;
        for (int p = 0; p < na; ++p) for (int q = 0; q < nb; ++q)
        for (int r = 0; r < nc; ++r) for (int s = 0; s < nd; ++s, ++n) {
            int a[3] = {ca[p][0], ca[p][1], ca[p][2]}, b[3] = {cb[q][0], cb[q][1], cb[q][2]};
            int c[3] = {cc[r][0], cc[r][1], cc[r][2]}, d[3] = {cd[s][0], cd[s][1], cd[s][2]};
            w->cart[n] = hrr(&h, a, b, c, d);
        }
    }
    /* dense c2s on each index in turn, Eq. (17) PAPER.md:235 / Eq. (8) :187 */
    int dims[4] = {na, nb, nc, nd};
    double *src = w->cart, *dst = w->tmp;
    for (int ax = 0; ax < 4; ++ax) {
        int lx = l[ax], nsph = 2 * lx + 1, ncx = dims[ax];
        double Tm[9 * 15];
        orc_c2s_matrix(lx, Tm);
        size_t outer = 1, inner = 1;
        for (int t = 0; t < ax; ++t) outer *= dims[t];
        for (int t = ax + 1; t < 4; ++t) inner *= dims[t];
        for (size_t o = 0; o < outer; ++o)
            for (int ms = 0; ms < nsph; ++ms)
                for (size_t in = 0; in < inner; ++in) {
                    double s = 0.0;
                    for (int k = 0; k < ncx; ++k) s += Tm[ms * ncx + k] * src[(o * ncx + k) * inner + in];
                    dst[(o * nsph + ms) * inner + in] = s;
                }
        dims[ax] = nsph;
        double *t2 = src; src = dst; dst = t2;
    }
    size_t nout = (size_t)dims[0] * dims[1] * dims[2] * dims[3];
    memcpy(out, src, nout * sizeof(double));
}

/* ---------------------------------------------------------------- independent route: McMurchie-Davidson
 * Own Boys routine (composite Gauss-Legendre quadrature of the defining integral), Hermite
 * expansion coefficients E_t^{ij}, Hermite Coulomb integrals R^n_{tuv}.  Tiny inputs only. */
static void gauss_legendre(int n, double *xs, double *ws)
{
    for (int i = 0; i < n; ++i) {
        double z = cos(PI * (i + 0.75) / (n + 0.5)), pp = 1.0;
        for (int it = 0; it < 100; ++it) {
            double p1 = 1.0, p2 = 0.0;
            for (int j = 1; j <= n; ++j) { double p3 = p2; p2 = p1; p1 = ((2.0 * j - 1.0) * z * p2 - (j - 1.0) * p3) / j; }
            pp = n * (z * p1 - p2) / (z * z - 1.0);
            double dz = p1 / pp;
            z -= dz;
            if (fabs(dz) < 1e-16) break;
        }
        xs[i] = z; ws[i] = 2.0 / ((1.0 - z * z) * pp * pp);
    }
}

/* F_m(T) = int_0^1 t^{2m} e^{-T t^2} dt by 64 panels x 20-point Gauss-Legendre */
void orc_boys_quadrature(int mmax, double T, double *F)
{
    enum { NP = 64, NG = 20 };
    double xs[NG], ws[NG];
    gauss_legendre(NG, xs, ws);
    for (int m = 0; m <= mmax; ++m) F[m] = 0.0;
    for (int p = 0; p < NP; ++p) {
        double lo = (double)p / NP, hw = 0.5 / NP;
        for (int g = 0; g < NG; ++g) {
            double t = lo + hw * (xs[g] + 1.0), t2 = t * t, e = exp(-T * t2) * ws[g] * hw, pw = 1.0;
            for (int m = 0; m <= mmax; ++m) { F[m] += pw * e; pw *= t2; }
        }
    }
}

/* 1-D Hermite coefficients E[i][j][t], i<=imax, j<=jmax; XAB = A-B */
static void hermite_E(int imax, int jmax, double al, double be, double XAB, double E[9][9][18])
{
    double p = al + be, mu = al * be / p, XPA = -be / p * XAB, XPB = al / p * XAB;
    memset(E, 0, sizeof(double) * 9 * 9 * 18);
    E[0][0][0] = exp(-mu * XAB * XAB);
    for (int i = 0; i <= imax; ++i)
        for (int j = 0; j <= jmax; ++j) {
            if (i == 0 && j == 0) continue;
            for (int t = 0; t <= i + j; ++t) {
                double v;
                if (j == 0) v = (t > 0 ? E[i - 1][j][t - 1] / (2 * p) : 0.0) + XPA * E[i - 1][j][t] + (t + 1) * E[i - 1][j][t + 1];
                else        v = (t > 0 ? E[i][j - 1][t - 1] / (2 * p) : 0.0) + XPB * E[i][j - 1][t] + (t + 1) * E[i][j - 1][t + 1];
                E[i][j][t] = v;
            }
        }
}

static void eri_quartet_md(const int *l, const int *K, const double *const *ex, const double *const *co,
                           const double *const *R, double *out, orc_work *w)
{
    int la = l[0], lb = l[1], lc = l[2], ld = l[3], L = la + lb + lc + ld;
    int na = ncart(la), nb = ncart(lb), nc = ncart(lc), nd = ncart(ld);
    int ca[15][3], cb[15][3], cc[15][3], cd[15][3];
    cart_list(la, ca); cart_list(lb, cb); cart_list(lc, cc); cart_list(ld, cd);
    size_t ncartall = (size_t)na * nb * nc * nd;
    for (size_t k = 0; k < ncartall; ++k) w->cart[k] = 0.0;
    int N = L + 1;
    /* Rt[n][t][u][v] */
    double *Rt = (double *)malloc(sizeof(double) * N * N * N * N);
    #define RT(n, t, u, v) Rt[(((size_t)(n) * N + (t)) * N + (u)) * N + (v)]
    static __thread double Eab[3][9][9][18], Ecd[3][9][9][18];
    for (int i = 0; i < K[0]; ++i) for (int j = 0; j < K[1]; ++j)
    for (int k = 0; k < K[2]; ++k) for (int m4 = 0; m4 < K[3]; ++m4) {
        double al = ex[0][i], be = ex[1][j], ga = ex[2][k], de = ex[3][m4];
        double p = al + be, q = ga + de, alpha = p * q / (p + q);
        double PQ[3], PQ2 = 0;
        for (int t = 0; t < 3; ++t) {
            double P = (al * R[0][t] + be * R[1][t]) / p, Q = (ga * R[2][t] + de * R[3][t]) / q;
            PQ[t] = P - Q; PQ2 += PQ[t] * PQ[t];
            hermite_E(la, lb, al, be, R[0][t] - R[1][t], Eab[t]);
            hermite_E(lc, ld, ga, de, R[2][t] - R[3][t], Ecd[t]);
        }
        double F[MMAX + 1];
        orc_boys_quadrature(L, alpha * PQ2, F);
        for (int n = 0; n <= L; ++n)
            for (int t = 0; t + n <= L; ++t) for (int u = 0; t + u + n <= L; ++u) for (int v = 0; t + u + v + n <= L; ++v)
                RT(n, t, u, v) = 0.0;
        for (int n = L; n >= 0; --n) {
            RT(n, 0, 0, 0) = pow(-2.0 * alpha, n) * F[n];
            for (int s = 1; s + n <= L; ++s)                 /* total order s = t+u+v */
                for (int t = 0; t <= s; ++t) for (int u = 0; t + u <= s; ++u) {
                    int v = s - t - u;
                    double r;
                    if (t > 0)      r = (t > 1 ? (t - 1) * RT(n + 1, t - 2, u, v) : 0.0) + PQ[0] * RT(n + 1, t - 1, u, v);
                    else if (u > 0) r = (u > 1 ? (u - 1) * RT(n + 1, t, u - 2, v) : 0.0) + PQ[1] * RT(n + 1, t, u - 1, v);
                    else            r = (v > 1 ? (v - 1) * RT(n + 1, t, u, v - 2) : 0.0) + PQ[2] * RT(n + 1, t, u, v - 1);
                    RT(n, t, u, v) = r;
                }
        }
        double pref = 2.0 * pow(PI, 2.5) / (p * q * sqrt(p + q)) * co[0][i] * co[1][j] * co[2][k] * co[3][m4];
        size_t n = 0;
        for (int pa = 0; pa < na; ++pa) for (int pb = 0; pb < nb; ++pb)
        for (int pc = 0; pc < nc; ++pc) for (int pd = 0; pd < nd; ++pd, ++n) {
            const int *a = ca[pa], *b = cb[pb], *c = cc[pc], *d = cd[pd];
            double s = 0.0;
            for (int t = 0; t <= a[0] + b[0]; ++t) for (int u = 0; u <= a[1] + b[1]; ++u) for (int v = 0; v <= a[2] + b[2]; ++v) {
                double eab = Eab[0][a[0]][b[0]][t] * Eab[1][a[1]][b[1]][u] * Eab[2][a[2]][b[2]][v];
                double s2 = 0.0;
                for (int tt = 0; tt <= c[0] + d[0]; ++tt) for (int uu = 0; uu <= c[1] + d[1]; ++uu) for (int vv = 0; vv <= c[2] + d[2]; ++vv) {
                    double ecd = Ecd[0][c[0]][d[0]][tt] * Ecd[1][c[1]][d[1]][uu] * Ecd[2][c[2]][d[2]][vv];
                    s2 += ((tt + uu + vv) % 2 ? -1.0 : 1.0) * ecd * RT(0, t + tt, u + uu, v + vv);
                }
                s += eab * s2;
            }
            w->cart[n] += pref * s;
        }
    }
    #undef RT
    free(Rt);
    int dims[4] = {na, nb, nc, nd};
    double *src = w->cart, *dst = w->tmp;
    for (int ax = 0; ax < 4; ++ax) {
        int lx = l[ax], nsph = 2 * lx + 1, ncx = dims[ax];
        double Tm[9 * 15];
        orc_c2s_matrix(lx, Tm);
        size_t outer = 1, inner = 1;
        for (int t = 0; t < ax; ++t) outer *= dims[t];
        for (int t = ax + 1; t < 4; ++t) inner *= dims[t];
        for (size_t o = 0; o < outer; ++o) for (int ms = 0; ms < nsph; ++ms) for (size_t in = 0; in < inner; ++in) {
            double s = 0.0;
            for (int k = 0; k < ncx; ++k) s += Tm[ms * ncx + k] * src[(o * ncx + k) * inner + in];
            dst[(o * nsph + ms) * inner + in] = s;
        }
        dims[ax] = nsph;
        double *t2 = src; src = dst; dst = t2;
    }
    memcpy(out, src, sizeof(double) * dims[0] * dims[1] * dims[2] * dims[3]);
}

/* ---------------------------------------------------------------- batch entry (C ABI for ctypes)
 * All quartets must belong to one angular class (la,lb,lc,ld) = class of quartet 0.
 * mode: 0 HGP (Alg. 2 order), 1 HRR-per-primitive, 2 McMurchie-Davidson.
 * out: [n][nsph(la)][nsph(lb)][nsph(lc)][nsph(ld)].  Returns 0, or -1 on class mismatch / l > 4. */
int orc_eri_batch(int nshell, const int32_t *shell_l, const int32_t *prim_off, const double *exps,
                  const double *coefs, const double *centers, const int32_t *quartets, int64_t n,
                  int mode, int nthreads, double *out)
{
    if (n <= 0) return 0;
    int l[4];
    for (int t = 0; t < 4; ++t) {
        int s = quartets[t];
        if (s < 0 || s >= nshell) return -1;
        l[t] = shell_l[s];
        if (l[t] < 0 || l[t] > LMAX) return -1;
    }
    for (int64_t q = 0; q < n; ++q)
        for (int t = 0; t < 4; ++t) {
            int s = quartets[4 * q + t];
            if (s < 0 || s >= nshell || shell_l[s] != l[t]) return -1;
        }
    size_t nout = (size_t)(2 * l[0] + 1) * (2 * l[1] + 1) * (2 * l[2] + 1) * (2 * l[3] + 1);
    init_trip();
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
    #pragma omp parallel
    {
        orc_work *w = work_new();
        #pragma omp for schedule(dynamic, 4)
        for (int64_t q = 0; q < n; ++q) {
            int K[4];
            const double *ex[4], *co[4], *R[4];
            for (int t = 0; t < 4; ++t) {
                int s = quartets[4 * q + t];
                K[t] = prim_off[s + 1] - prim_off[s];
                ex[t] = exps + prim_off[s]; co[t] = coefs + prim_off[s]; R[t] = centers + 3 * s;
            }
            if (mode == 2) eri_quartet_md(l, K, ex, co, R, out + nout * q, w);
            else           eri_quartet(l, K, ex, co, R, mode, out + nout * q, w);
        }
        work_free(w);
    }
    return 0;
}

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
