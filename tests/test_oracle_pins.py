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
    """Rows of T^(l) written out for l <= 3; Cartesian order xx,xy,xz,yy,yz,zz etc."""
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
