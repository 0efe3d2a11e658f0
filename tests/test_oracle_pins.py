"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU).

Each test names the plausible mistake it would catch.
"""
import math

import numpy as np
import pytest
from scipy import special

import oracle
from golden_util import read_boys, read_eri_golden
from paper_2605_10312_b200 import workloads as wl


# ------------------------------------------------------------------ Boys function
def test_boys_reference_table():
    """F_m(T) against the 50-digit table (tests/golden/boys_reference.txt)."""
    for T, m, ref in read_boys():
        got = oracle.boys(16, T)[m]
        assert abs(got - ref) <= 4e-15 * abs(ref) + 1e-300, (T, m, got, ref)


def test_boys_closed_forms_and_quadrature():
    rng = np.random.default_rng(5)
    assert np.allclose(oracle.boys(16, 0.0), 1.0 / (2 * np.arange(17) + 1), rtol=0, atol=1e-16)
    for T in np.concatenate([10 ** rng.uniform(-6, 2.3, 200), [34.999, 35.0, 35.001]]):
        F = oracle.boys(16, T)
        # F_0 closed form and incomplete-gamma form (scipy is an independent library routine)
        assert abs(F[0] - 0.5 * math.sqrt(math.pi / T) * math.erf(math.sqrt(T))) < 4e-15 * F[0]
        for m in (3, 9, 16):
            g = special.gammainc(m + 0.5, T) * special.gamma(m + 0.5) / (2 * T ** (m + 0.5))
            assert abs(F[m] - g) < 2e-13 * g
        # recurrence identity (2m+1) F_m = 2T F_{m+1} + e^-T
        m = np.arange(16)
        assert np.allclose((2 * m + 1) * F[:-1], 2 * T * F[1:] + math.exp(-T), rtol=2e-13, atol=1e-300)
        # direct quadrature of the defining integral
        assert np.allclose(F, oracle.boys_quadrature(16, T), rtol=1e-12, atol=1e-300)


# ------------------------------------------------------------------ c2s (R-SPH)
def test_c2s_printed_rows():
    """Rows of T^(l) written out for l <= 4 (SURVEY 8(c) R-SPH; l = 4 below the function); Cartesian order xx,xy,xz,yy,yz,zz etc."""
    assert np.allclose(oracle.c2s_matrix(0), [[1.0]])
    # l=1: y, z, x  with components (x, y, z)
    assert np.allclose(oracle.c2s_matrix(1), [[0, 1, 0], [0, 0, 1], [1, 0, 0]])
    s3 = math.sqrt(3.0)
    assert np.allclose(oracle.c2s_matrix(2), [[0, s3, 0, 0, 0, 0], [0, 0, 0, 0, s3, 0],
                                              [-0.5, 0, 0, -0.5, 0, 1], [0, 0, s3, 0, 0, 0],
                                              [s3 / 2, 0, 0, -s3 / 2, 0, 0]])
    # l=3 components: xxx xxy xxz xyy xyz xzz yyy yyz yzz zzz
    a, b, c = math.sqrt(10) / 4, math.sqrt(15), math.sqrt(6) / 4
    ref = np.zeros((7, 10))
    ref[0, 1], ref[0, 6] = 3 * a, -a                      # (sqrt10/4)(3xxy - yyy)
    ref[1, 4] = b                                         # sqrt15 xyz
    ref[2, 8], ref[2, 1], ref[2, 6] = 4 * c, -c, -c       # (sqrt6/4)(4yzz - xxy - yyy)
    ref[3, 9], ref[3, 2], ref[3, 7] = 1.0, -1.5, -1.5     # zzz - 3/2(xxz + yyz)
    ref[4, 5], ref[4, 0], ref[4, 3] = 4 * c, -c, -c       # (sqrt6/4)(4xzz - xxx - xyy)
    ref[5, 2], ref[5, 7] = b / 2, -b / 2                  # (sqrt15/2)(xxz - yyz)
    ref[6, 0], ref[6, 3] = a, -3 * a                      # (sqrt10/4)(xxx - 3xyy)
    assert np.allclose(oracle.c2s_matrix(3), ref, atol=1e-15)
    # l=4: the nine rows written out monomial by monomial (keys are the exponents (i,j,k) of x^i y^j z^k); checked by hand
    # against the textbook table of Racah-normalised real solid harmonics, e.g. S_40 = z^4 - 3 z^2 (x^2+y^2) + 3/8 (x^2+y^2)^2,
    # S_44 = (sqrt35/8)(x^4 - 6 x^2 y^2 + y^4).  A negated row, two swapped rows or a wrong normalisation fails here.
    comps = _carts(4)
    T4 = oracle.c2s_matrix(4)
    assert T4.shape == (9, 15)
    for m, poly in L4_ROWS.items():
        want = np.zeros(15)
        for mono, coef in poly.items():
            want[comps.index(mono)] = coef
        assert np.allclose(T4[m + 4], want, atol=2e-15), (m, T4[m + 4], want)


_S35, _S70, _S5, _S10 = math.sqrt(35.0), math.sqrt(70.0), math.sqrt(5.0), math.sqrt(10.0)
L4_ROWS = {
    -4: {(3, 1, 0): _S35 / 2, (1, 3, 0): -_S35 / 2},                                        # (sqrt35/2)(x^3 y - x y^3)
    -3: {(2, 1, 1): 3 * _S70 / 4, (0, 3, 1): -_S70 / 4},                                    # (sqrt70/4)(3 x^2 y z - y^3 z)
    -2: {(1, 1, 2): 3 * _S5, (3, 1, 0): -_S5 / 2, (1, 3, 0): -_S5 / 2},                     # (sqrt5/2)(6 x y z^2 - x^3 y - x y^3)
    -1: {(0, 1, 3): _S10, (2, 1, 1): -3 * _S10 / 4, (0, 3, 1): -3 * _S10 / 4},              # (sqrt10/4)(4 y z^3 - 3 x^2 y z - 3 y^3 z)
    0: {(0, 0, 4): 1.0, (2, 0, 2): -3.0, (0, 2, 2): -3.0, (4, 0, 0): 0.375, (2, 2, 0): 0.75, (0, 4, 0): 0.375},
    1: {(1, 0, 3): _S10, (3, 0, 1): -3 * _S10 / 4, (1, 2, 1): -3 * _S10 / 4},               # (sqrt10/4)(4 x z^3 - 3 x^3 z - 3 x y^2 z)
    2: {(2, 0, 2): 3 * _S5 / 2, (0, 2, 2): -3 * _S5 / 2, (4, 0, 0): -_S5 / 4, (0, 4, 0): _S5 / 4},   # (sqrt5/4)(6 x^2 z^2 - 6 y^2 z^2 - x^4 + y^4)
    3: {(3, 0, 1): _S70 / 4, (1, 2, 1): -3 * _S70 / 4},                                     # (sqrt70/4)(x^3 z - 3 x y^2 z)
    4: {(4, 0, 0): _S35 / 8, (2, 2, 0): -6 * _S35 / 8, (0, 4, 0): _S35 / 8},                # (sqrt35/8)(x^4 - 6 x^2 y^2 + y^4)
}


def _dfact(n):
    return 1.0 if n <= 0 else n * _dfact(n - 2)


def _carts(l):
    return [(i, j, l - i - j) for i in range(l, -1, -1) for j in range(l - i, -1, -1)]


@pytest.mark.parametrize("l", [0, 1, 2, 3, 4])
def test_c2s_gram_matrix(l):
    """T M T^T = (2l-1)!!-proportional identity with Gaussian moments: rows orthogonal, equal norm."""
    comps = _carts(l)
    M = np.zeros((len(comps), len(comps)))
    for p, a in enumerate(comps):
        for q, b in enumerate(comps):
            s = [a[k] + b[k] for k in range(3)]
            if all(x % 2 == 0 for x in s):
                M[p, q] = _dfact(s[0] - 1) * _dfact(s[1] - 1) * _dfact(s[2] - 1)
    T = oracle.c2s_matrix(l)
    G = T @ M @ T.T
    assert np.allclose(G, G[0, 0] * np.eye(2 * l + 1), atol=1e-12 * G[0, 0])
    # harmonicity: Laplacian of every row vanishes
    low = {c: k for k, c in enumerate(_carts(l - 2))} if l >= 2 else {}
    for row in T:
        lap = np.zeros(len(low))
        for coef, c in zip(row, comps):
            for ax in range(3):
                if c[ax] >= 2:
                    d = list(c); d[ax] -= 2
                    lap[low[tuple(d)]] += coef * c[ax] * (c[ax] - 1)
        assert np.allclose(lap, 0, atol=1e-13)
    # leading term of S_l0 is z^l (Racah normalisation)
    assert abs(T[l, len(comps) - 1] - 1.0) < 1e-15


# ------------------------------------------------------------------ (ss|ss) closed forms
def _s_basis(alpha, centers):
    n = len(centers)
    c = wl.normalise_shell(0, [alpha], [1.0])
    return wl.make_basis([0] * n, [[alpha]] * n, [c] * n, centers)


def test_ssss_closed_forms():
    for alpha in (0.3, 1.0, 4.7):
        b = _s_basis(alpha, [[0.1, 0.2, 0.3]])
        v = oracle.eri_batch(b, [[0, 0, 0, 0]]).ravel()[0]
        assert abs(v - 2 * math.sqrt(alpha / math.pi)) < 1e-14 * v
        for Rd in (0.5, 2.0, 9.0):
            b = _s_basis(alpha, [[0, 0, 0], [0, 0, Rd]])
            v = oracle.eri_batch(b, [[0, 0, 1, 1]]).ravel()[0]
            assert abs(v - math.erf(math.sqrt(alpha) * Rd) / Rd) < 1e-14 * v


def test_primitive_ssss_formula():
    """S*F_0(T) written out for one unnormalised primitive quartet."""
    ex = [0.8, 1.3, 0.5, 2.1]
    cen = np.array([[0, 0, 0], [0.5, -0.3, 0.2], [1.0, 0.4, -0.7], [-0.2, 0.9, 0.3]], float)
    b = wl.make_basis([0] * 4, [[e] for e in ex], [[1.0]] * 4, cen)
    z, e = ex[0] + ex[1], ex[2] + ex[3]
    P = (ex[0] * cen[0] + ex[1] * cen[1]) / z
    Q = (ex[2] * cen[2] + ex[3] * cen[3]) / e
    T = z * e / (z + e) * np.sum((P - Q) ** 2)
    F0 = 0.5 * math.sqrt(math.pi / T) * math.erf(math.sqrt(T))
    ref = (2 * math.pi ** 2.5 / (z * e * math.sqrt(z + e)) * math.exp(-ex[0] * ex[1] / z * np.sum((cen[0] - cen[1]) ** 2))
           * math.exp(-ex[2] * ex[3] / e * np.sum((cen[2] - cen[3]) ** 2)) * F0)
    v = oracle.eri_batch(b, [[0, 1, 2, 3]]).ravel()[0]
    assert abs(v - ref) < 1e-14 * abs(ref)


# ------------------------------------------------------------------ golden ERIs
def test_golden_eris():
    basis, sums, comps = read_eri_golden()
    for mode in (0, 1, 2):
        for q, n, s, s2 in sums:
            v = oracle.eri_batch(basis, [q], mode=mode)
            assert v.size == n
            assert abs(v.sum() - s) < 2e-12 * abs(s) and abs((v ** 2).sum() - s2) < 2e-12 * s2, (mode, q)
        for q, idx, ref in comps:
            v = oracle.eri_batch(basis, [q], mode=mode)[0][idx]
            assert abs(v - ref) < 1e-12 * abs(ref) + 1e-15, (mode, q, idx, v, ref)
    # visible sanity of the table: (ps|ss) components are -(Ay, Az, Ax) ratios 0.2 : -0.5 : -0.3
    v = oracle.eri_batch(basis, [(1, 0, 0, 0)]).ravel()
    assert np.allclose(v / v[0], [1.0, -2.5, -1.5], rtol=1e-12)


# ------------------------------------------------------------------ g shells by Hobson differentiation (pins T^(4) inside an ERI)
def test_g_shell_by_hobson_differentiation():
    """An unnormalised solid-harmonic Gaussian is a derivative of an s Gaussian (Hobson's theorem):
    S_lm(r-A) exp(-a|r-A|^2) = (2a)^-l S_lm(d/dA) exp(-a|r-A|^2), so
    (g_m b|cd) = (2a)^-4 S_4m(d/dA) (s_A b|cd).  With the rows of L4_ROWS (written out above, never taken from the oracle)
    as differential operators applied to the closed form of the primitive (ss|ss) integral (mpmath's numerical
    central differences of step 1e-10 at 130 digits: O(h^2) truncation, 40 digits lost per nesting), this gives every component of (gs|ss), (gs|ps) and components of (gs|gs) with no
    recurrence, no Cartesian intermediate and no c2s matrix: row order, sign and normalisation of T^(4), the bra VRR up to
    l = 4 and the ket side are pinned together."""
    import mpmath as mp
    mp.mp.dps = 130
    al, be, ga, de = [mp.mpf(s) for s in ("0.9", "1.7", "0.6", "1.2")]
    Bc = [mp.mpf(s) for s in ("0.4", "-0.3", "0.5")]
    Dc = [mp.mpf(s) for s in ("0.8", "-0.5", "-0.2")]
    A0 = [mp.mpf(s) for s in ("0.1", "0.7", "-0.4")]
    C0 = [mp.mpf(s) for s in ("-0.6", "0.2", "0.9")]
    zeta, eta = al + be, ga + de

    def ssss(a0, a1, a2, c0, c1, c2):
        A, C = (a0, a1, a2), (c0, c1, c2)
        P = [(al * A[i] + be * Bc[i]) / zeta for i in range(3)]
        Q = [(ga * C[i] + de * Dc[i]) / eta for i in range(3)]
        T = zeta * eta / (zeta + eta) * sum((P[i] - Q[i]) ** 2 for i in range(3))
        F0 = mp.sqrt(mp.pi / T) * mp.erf(mp.sqrt(T)) / 2
        return (2 * mp.pi ** mp.mpf("2.5") / (zeta * eta * mp.sqrt(zeta + eta))
                * mp.exp(-al * be / zeta * sum((A[i] - Bc[i]) ** 2 for i in range(3)))
                * mp.exp(-ga * de / eta * sum((C[i] - Dc[i]) ** 2 for i in range(3))) * F0)

    def directional(poly):
        """p(grad) for a homogeneous polynomial p of degree l as a weighted sum of l-th DIRECTIONAL derivatives:
        (v.grad)^l = sum_alpha (l!/alpha!) v^alpha d^alpha, solved for the weights over ncart(l) integer directions."""
        l = sum(next(iter(poly)))
        monos = _carts(l)
        dirs = [tuple(mp.mpf(x + 1) for x in mno) for mno in monos]          # (i+1, j+1, k+1): a unisolvent set
        M = mp.matrix(len(monos), len(monos))
        for si, v in enumerate(dirs):
            for ai, (i, j, k) in enumerate(monos):
                M[ai, si] = mp.factorial(l) / (mp.factorial(i) * mp.factorial(j) * mp.factorial(k)) * v[0] ** i * v[1] ** j * v[2] ** k
        rhs = mp.matrix([mp.mpf(poly.get(mno, 0.0)) for mno in monos])
        w = mp.lu_solve(M, rhs)
        return l, dirs, [w[i] for i in range(len(monos))]

    H = mp.mpf(10) ** -10

    def dn(fun, n):
        """n-th derivative at 0 by the central difference of step H."""
        if n == 0:
            return fun(mp.mpf(0))
        return sum((-1) ** k * mp.binomial(n, k) * fun((mp.mpf(n) / 2 - k) * H) for k in range(n + 1)) / H ** n

    def op(bra_poly, ket_poly):
        la_, da, wa = directional(bra_poly)
        lc_, dc, wc = directional(ket_poly)

        def inner(c0, c1, c2):          # p(grad_A) f at fixed C
            tot = mp.mpf(0)
            for v, w in zip(da, wa):
                if w != 0:
                    tot += w * dn(lambda t: ssss(A0[0] + t * v[0], A0[1] + t * v[1], A0[2] + t * v[2], c0, c1, c2), la_)
            return tot

        tot = mp.mpf(0)
        for v, w in zip(dc, wc):
            if w != 0:
                tot += w * dn(lambda t: inner(C0[0] + t * v[0], C0[1] + t * v[1], C0[2] + t * v[2]), lc_)
        return tot

    ONE = {(0, 0, 0): 1.0}
    P_ROWS = {-1: {(0, 1, 0): 1.0}, 0: {(0, 0, 1): 1.0}, 1: {(1, 0, 0): 1.0}}        # l = 1: y, z, x
    cen = [[0.1, 0.7, -0.4], [0.4, -0.3, 0.5], [-0.6, 0.2, 0.9], [0.8, -0.5, -0.2]]
    ex = [0.9, 1.7, 0.6, 1.2]
    sa, sc = (2 * al) ** 4, 2 * ga
    # (gs|ss)
    b = wl.make_basis([4, 0, 0, 0], [[x] for x in ex], [[1.0]] * 4, cen)
    got = oracle.eri_batch(b, [[0, 1, 2, 3]])[0].ravel()
    ref = np.array([float(op(L4_ROWS[m], ONE) / sa) for m in range(-4, 5)])
    assert np.allclose(got, ref, rtol=2e-12, atol=1e-15 * np.abs(ref).max()), (got, ref)
    # (gs|ps): one more derivative on C
    b = wl.make_basis([4, 0, 1, 0], [[x] for x in ex], [[1.0]] * 4, cen)
    got = oracle.eri_batch(b, [[0, 1, 2, 3]])[0].reshape(9, 3)
    ref = np.array([[float(op(L4_ROWS[m], P_ROWS[mc]) / sa / sc) for mc in (-1, 0, 1)] for m in range(-4, 5)])
    assert np.allclose(got, ref, rtol=2e-12, atol=1e-15 * np.abs(ref).max()), (got, ref)
    # (gs|gs), five components (8th derivatives): the ket-side T^(4) and the ket VRR up to l = 4 as well
    b = wl.make_basis([4, 0, 4, 0], [[x] for x in ex], [[1.0]] * 4, cen)
    got = oracle.eri_batch(b, [[0, 1, 2, 3]])[0].reshape(9, 9)
    for m, mc in ((-4, 3), (0, 0), (2, -1), (4, 4), (-3, 1)):
        r = float(op(L4_ROWS[m], L4_ROWS[mc]) / sa / sc ** 4)
        assert abs(got[m + 4, mc + 4] - r) <= 2e-12 * abs(r) + 1e-15, (m, mc, got[m + 4, mc + 4], r)
