"""Pins of the first-derivative oracle (oracle/eri_grad_oracle.c), no GPU.

The derivative of an integral has a plain definition, so the pins are the ones the mathematics fixes:
  * five-point finite differences of the PINNED integral oracle (oracle.eri_batch, tests/test_oracle_pins.py) in every one
    of the twelve directions -- a dropped term, a wrong sign, exponent, centre, axis or component order fails it;
  * the closed form of d(ss|ss)/dA for primitives, typed out here from (ss|ss) = S F_0(T) with scipy's incomplete gamma
    function for F_0 and F_1;
  * translational invariance (the four centre derivatives sum to zero -- the oracle computes all twelve from the definition);
  * the permutations (ab|cd) = (ba|cd) = (ab|dc) = (cd|ab) carried over to the derivative index;
  * a shell on the same centre in two columns (A = B): the column derivatives add up to the derivative of the integral.
"""
import numpy as np
import pytest
from scipy import special

import oracle
from paper_2605_10312_b200 import workloads as wl


def _rand_basis(seed, ls, kmax=2, box=2.0):
    rng = np.random.default_rng(seed)
    exps = [np.exp(rng.uniform(np.log(0.3), np.log(3.0), rng.integers(1, kmax + 1))) for _ in ls]
    coefs = [wl.normalise_shell(l, e, rng.uniform(0.1, 1.0, len(e))) for l, e in zip(ls, exps)]
    return wl.make_basis(ls, exps, coefs, rng.uniform(0, box, (len(ls), 3)))


def _fd(basis, q, shell, axis, h=2e-3):
    """five-point central difference of oracle.eri_batch with respect to centers[shell][axis]"""
    def at(t):
        b = dict(basis)
        c = np.array(basis["centers"], float).copy()
        c[shell, axis] += t
        b["centers"] = c
        return oracle.eri_batch(b, q)[0]
    return (8.0 * (at(h) - at(-h)) - (at(2 * h) - at(-2 * h))) / (12.0 * h)


CLASSES = [(0, 0, 0, 0), (1, 0, 0, 0), (0, 1, 0, 0), (0, 0, 1, 0), (0, 0, 0, 1), (1, 1, 1, 1), (2, 1, 0, 1), (1, 2, 2, 0),
           (2, 2, 2, 2), (0, 2, 1, 2), (3, 1, 2, 0), (1, 0, 3, 2)]


@pytest.mark.parametrize("cls", CLASSES)
def test_grad_equals_finite_differences(cls):
    b = _rand_basis(1000 + sum(x * 5 ** i for i, x in enumerate(cls)), list(cls))
    q = [[0, 1, 2, 3]]
    g = oracle.eri_grad_batch(b, q)[0]
    ref = oracle.eri_batch(b, q)[0]
    assert g.shape == (12,) + ref.shape
    scale = max(np.abs(g).max(), np.abs(ref).max())
    for cen in range(4):
        for ax in range(3):
            fd = _fd(b, q, cen, ax)
            # truncation h^4 f^(5) / 30 and rounding 1e-16 / h: both far below 1e-8 of the scale
            assert np.abs(g[3 * cen + ax] - fd).max() < 1e-8 * scale, (cls, cen, ax)


def _boys01(T):
    if T < 1e-13:
        return 1.0, 1.0 / 3.0
    f = lambda m: special.gamma(m + 0.5) * special.gammainc(m + 0.5, T) / (2.0 * T ** (m + 0.5))   # noqa: E731
    return f(0), f(1)


def test_ssss_closed_form():
    """(ss|ss) = c S F_0(T), S = 2 pi^2.5 / (zeta eta sqrt(zeta + eta)) exp(-alpha beta |AB|^2 / zeta) exp(-gamma delta |CD|^2 / eta),
    T = rho |PQ|^2.  With dF_0/dT = -F_1, dP/dA = alpha / zeta:
    d/dA_i = c S [ -2 alpha beta / zeta (A_i - B_i) F_0 - 2 rho alpha / zeta (P_i - Q_i) F_1 ], and likewise for B, C, D."""
    rng = np.random.default_rng(5)
    for trial in range(6):
        ex = np.exp(rng.uniform(np.log(0.2), np.log(4.0), 4))
        co = rng.uniform(0.3, 1.2, 4)
        R = rng.uniform(0, 2.5 if trial < 5 else 0.0, (4, 3))
        b = wl.make_basis([0, 0, 0, 0], [[e] for e in ex], [[c] for c in co], R)
        g = oracle.eri_grad_batch(b, [[0, 1, 2, 3]])[0].reshape(4, 3)
        al, be, ga, de = ex
        zeta, eta = al + be, ga + de
        rho = zeta * eta / (zeta + eta)
        P = (al * R[0] + be * R[1]) / zeta
        Q = (ga * R[2] + de * R[3]) / eta
        S = 2 * np.pi ** 2.5 / (zeta * eta * np.sqrt(zeta + eta)) * np.exp(-al * be / zeta * ((R[0] - R[1]) ** 2).sum()
                                                                           - ga * de / eta * ((R[2] - R[3]) ** 2).sum())
        F0, F1 = _boys01(rho * ((P - Q) ** 2).sum())
        c = co.prod() * S
        want = np.array([c * (-2 * al * be / zeta * (R[0] - R[1]) * F0 - 2 * rho * al / zeta * (P - Q) * F1),
                         c * (+2 * al * be / zeta * (R[0] - R[1]) * F0 - 2 * rho * be / zeta * (P - Q) * F1),
                         c * (-2 * ga * de / eta * (R[2] - R[3]) * F0 + 2 * rho * ga / eta * (P - Q) * F1),
                         c * (+2 * ga * de / eta * (R[2] - R[3]) * F0 + 2 * rho * de / eta * (P - Q) * F1)])
        assert np.abs(g - want).max() < 1e-13 * max(abs(c), np.abs(want).max())


@pytest.mark.parametrize("cls", [(1, 1, 1, 1), (2, 0, 1, 2), (2, 2, 2, 2), (3, 2, 1, 0), (4, 1, 0, 0)])
def test_translational_invariance(cls):
    b = _rand_basis(77 + sum(cls), list(cls))
    g = oracle.eri_grad_batch(b, [[0, 1, 2, 3]])[0]
    tot = g.reshape((4, 3) + g.shape[1:]).sum(axis=0)
    assert np.abs(tot).max() < 2e-13 * np.abs(g).max()


def test_permutations():
    cls = (2, 1, 0, 2)
    b = _rand_basis(31, list(cls))
    g = oracle.eri_grad_batch(b, [[0, 1, 2, 3]])[0].reshape(4, 3, 5, 3, 1, 5)
    tol = 1e-13 * np.abs(g).max()
    for perm in ((1, 0, 2, 3), (0, 1, 3, 2), (2, 3, 0, 1), (3, 2, 1, 0)):
        h = oracle.eri_grad_batch(b, [list(perm)])[0]
        h = h.reshape((4, 3) + h.shape[1:])
        # column k of the permuted quartet is shell perm[k]: its derivative is centre perm[k] of the reference, and the
        # component axes are permuted the same way
        want = g[list(perm)].transpose((0, 1) + tuple(2 + p for p in perm))
        assert np.abs(h - want).max() < tol, perm


def test_coincident_columns_add_up():
    """quartet (s0 s0|s1 s2): moving shell s0 moves columns a AND b, so FD of the integral = column a + column b."""
    b = _rand_basis(41, [1, 2, 1])
    q = [[0, 0, 1, 2]]
    g = oracle.eri_grad_batch(b, q)[0]
    for ax in range(3):
        fd = _fd(b, q, 0, ax)
        assert np.abs(g[ax] + g[3 + ax] - fd).max() < 1e-8 * np.abs(g).max()


def test_contraction_is_linear():
    """the derivative of a contracted quartet is the coefficient-weighted sum of its primitive quartets' derivatives"""
    rng = np.random.default_rng(3)
    ls = [1, 2, 0, 1]
    exps = [np.exp(rng.uniform(np.log(0.3), np.log(3.0), 2)) for _ in ls]
    coefs = [rng.uniform(0.2, 1.0, 2) for _ in ls]
    R = rng.uniform(0, 2, (4, 3))
    g = oracle.eri_grad_batch(wl.make_basis(ls, exps, coefs, R), [[0, 1, 2, 3]])[0]
    s = np.zeros_like(g)
    for i in range(16):
        k = [(i >> t) & 1 for t in range(4)]
        bp = wl.make_basis(ls, [[exps[t][k[t]]] for t in range(4)], [[coefs[t][k[t]]] for t in range(4)], R)
        s += oracle.eri_grad_batch(bp, [[0, 1, 2, 3]])[0]
    assert np.abs(g - s).max() < 1e-13 * np.abs(g).max()
