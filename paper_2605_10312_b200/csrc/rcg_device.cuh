// rcg_device.cuh -- device helpers shared by every tier: Boys function and primitive-quartet setup.
#ifndef RCG_DEVICE_CUH
#define RCG_DEVICE_CUH
#include "rcg_internal.h"

#define RCG_PI 3.14159265358979323846
#define RCG_TWO_PI_2_5 34.986836655249725693   /* 2 * pi^(5/2) */

// F_m(T) = int_0^1 t^{2m} exp(-T t^2) dt, m = 0..L  (PAPER.md:69 [00|00]^(m); Alg. 2 line 5 at :273).
// Scheme R-BOYS: T < 36: nearest grid point T0 = round(8T)/8, 9-term Taylor series in
// (T0 - T) for the TOP order L only (d/dT F_m = -F_{m+1}), then the downward recursion
// F_{m-1} = (2T F_m + e^{-T}) / (2m-1).  T >= 36: F_0 = sqrt(pi/T)/2 (erf(6) = 1 in FP64) and the
// upward recursion F_{m+1} = ((2m+1) F_m - e^{-T}) / (2T), stable for T >> m.
// `scale` multiplies every value (the primitive prefactor, R-BASE).
template <int LT>
__device__ __forceinline__ void rcg_boys(int Lrt, double T, double scale, const double *__restrict__ tab, double *F)
{
    const int L = LT >= 0 ? LT : Lrt;
    const double eT = exp(-T);
    if (T < RCG_BOYS_TS) {
        const int row = (int)(T * 8.0 + 0.5);
        const double d = (double)row * 0.125 - T;
        const double *r = tab + row * RCG_BOYS_NCOL + L;
        double f = __ldg(r + 8);
        f = fma(f, d * (1.0 / 8.0), __ldg(r + 7));
        f = fma(f, d * (1.0 / 7.0), __ldg(r + 6));
        f = fma(f, d * (1.0 / 6.0), __ldg(r + 5));
        f = fma(f, d * (1.0 / 5.0), __ldg(r + 4));
        f = fma(f, d * (1.0 / 4.0), __ldg(r + 3));
        f = fma(f, d * (1.0 / 3.0), __ldg(r + 2));
        f = fma(f, d * (1.0 / 2.0), __ldg(r + 1));
        f = fma(f, d, __ldg(r));
        const double t2 = 2.0 * T, eTs = eT * scale;     // the recursion is linear: run it on the scaled values
        f *= scale;
        F[L] = f;
#pragma unroll
        for (int m = (LT >= 0 ? LT : 16); m >= 1; --m) {
            if (m <= L) {
                f = fma(t2, f, eTs) * (1.0 / (double)(2 * m - 1));
                F[m - 1] = f;
            }
        }
    } else {
        double f = 0.5 * sqrt(RCG_PI / T) * scale;
        const double r2 = 0.5 / T, eTs = eT * scale;
        F[0] = f;
#pragma unroll
        for (int m = 0; m < (LT >= 0 ? LT : 16); ++m) {
            if (m < L) {
                f = ((double)(2 * m + 1) * f - eTs) * r2;
                F[m + 1] = f;
            }
        }
    }
}

// p / k and p % k for 0 <= p < 2^22 (RCG_KMAX^4), rk = 1.0f / k to 2 ulp: float quotient (off by at most one), exact
// integer fix-up.  Replaces two run-time integer divisions per index of the primitive-quartet decode.
__device__ __forceinline__ int rcg_divmod(int p, int k, float rk, int &rem)
{
    int t = (int)(((float)p + 0.5f) * rk);
    int r = p - t * k;
    if (r < 0) { r += k; --t; }
    if (r >= k) { r -= k; ++t; }
    rem = r;
    return t;
}

// Gaussian-pair / quartet quantities of one primitive quartet ("GAUSSIANPAIRS",
// Alg. 2 line 4 at :272; formulas: reading R-PAIR).
struct RcgPrim {
    double PA[3], WP[3], QC[3], WQ[3];
    double hz, he, hze;     // 1/(2 zeta), 1/(2 eta), 1/(2(zeta+eta))
    double rz, re;          // rho/zeta, rho/eta
    double T, pref;         // Boys argument; 2 pi^{5/2}/(zeta eta sqrt(zeta+eta)) K_AB K_CD ca cb cc cd
};

__device__ __forceinline__ void rcg_prim_setup(RcgPrim &p, const double *A, const double *B, const double *C,
                                               const double *D, double al, double be, double ga, double de,
                                               double cc4)
{
    const double zeta = al + be, eta = ga + de;
    const double ze = zeta + eta;
    const double inv = 1.0 / (zeta * eta * ze);           // one FP64 division for the three reciprocals
    const double iz = inv * (eta * ze), ie = inv * (zeta * ze), ize = inv * (zeta * eta);
    const double rho = zeta * eta * ize;
    double ab2 = 0.0, cd2 = 0.0, pq2 = 0.0;
#pragma unroll
    for (int t = 0; t < 3; ++t) {
        const double P = (al * A[t] + be * B[t]) * iz;
        const double Q = (ga * C[t] + de * D[t]) * ie;
        const double W = (zeta * P + eta * Q) * ize;
        p.PA[t] = P - A[t];
        p.WP[t] = W - P;
        p.QC[t] = Q - C[t];
        p.WQ[t] = W - Q;
        const double ab = A[t] - B[t], cd = C[t] - D[t], pq = P - Q;
        ab2 = fma(ab, ab, ab2);
        cd2 = fma(cd, cd, cd2);
        pq2 = fma(pq, pq, pq2);
    }
    p.hz = 0.5 * iz;
    p.he = 0.5 * ie;
    p.hze = 0.5 * ize;
    p.rz = rho * iz;
    p.re = rho * ie;
    p.T = rho * pq2;
    p.pref = RCG_TWO_PI_2_5 * iz * ie * sqrt(ize) * exp(-al * be * iz * ab2 - ga * de * ie * cd2) * cc4;
}

#endif
