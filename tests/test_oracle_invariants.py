"""Invariants that pin the oracle's VRR / HRR / contraction / c2s (no GPU).

8-fold symmetry (bra/ket roles, HRR direction), translation / scaling / reflection,
linearity in primitives, Schwarz inequality, and agreement of the three routes
(HGP, HRR-per-primitive, McMurchie-Davidson) on tiny random inputs.
"""
import itertools

import numpy as np
import pytest

import oracle
from paper_2605_10312_b200 import workloads as wl


def _rand_basis(seed, ls, kmax=2, box=2.0):
    rng = np.random.default_rng(seed)
    exps = [np.exp(rng.uniform(np.log(0.3), np.log(3.0), rng.integers(1, kmax + 1))) for _ in ls]
    coefs = [wl.normalise_shell(l, e, rng.uniform(0.1, 1.0, len(e))) for l, e in zip(ls, exps)]
    return wl.make_basis(ls, exps, coefs, rng.uniform(0, box, (len(ls), 3)))


CLASSES = [(0, 0, 0, 0), (1, 0, 0, 0), (1, 1, 0, 0), (1, 0, 1, 0), (1, 1, 1, 1), (2, 0, 1, 0), (2, 1, 1, 0),
           (2, 1, 2, 1), (2, 2, 1, 1), (2, 2, 2, 2), (3, 1, 2, 0), (3, 2, 1, 1), (3, 3, 0, 0), (4, 0, 1, 1),
           (0, 1, 0, 2), (0, 0, 3, 1), (1, 2, 0, 3)]


@pytest.mark.parametrize("cls", CLASSES)
def test_three_routes_agree(cls):
    b = _rand_basis(sum(x * 7 ** i for i, x in enumerate(cls)) + 1, list(cls))
    q = [[0, 1, 2, 3]]
    r0, r1, r2 = (oracle.eri_batch(b, q, mode=m) for m in (0, 1, 2))
    scale = np.abs(r0).max()
    assert np.abs(r0 - r1).max() < 1e-13 * scale
    assert np.abs(r0 - r2).max() < 2e-12 * scale


def test_md_agrees_high_l():
    b = _rand_basis(99, [3, 3, 3, 3, 4, 4, 4, 4], kmax=1)
    for q in ([0, 1, 2, 3], [4, 5, 6, 7], [4, 1, 6, 3]):
        r0, r2 = oracle.eri_batch(b, [q], mode=0), oracle.eri_batch(b, [q], mode=2)
        assert np.abs(r0 - r2).max() < 1e-11 * np.abs(r0).max()


@pytest.mark.parametrize("cls", [(1, 0, 2, 1), (2, 1, 1, 0), (2, 2, 1, 0), (3, 1, 2, 2)])
def test_eightfold_symmetry(cls):
    b = _rand_basis(11, list(cls))
    ref = oracle.eri_batch(b, [[0, 1, 2, 3]])[0]
    assert np.allclose(oracle.eri_batch(b, [[1, 0, 2, 3]])[0], ref.transpose(1, 0, 2, 3), rtol=0, atol=1e-13 * np.abs(ref).max())
    assert np.allclose(oracle.eri_batch(b, [[0, 1, 3, 2]])[0], ref.transpose(0, 1, 3, 2), rtol=0, atol=1e-13 * np.abs(ref).max())
    assert np.allclose(oracle.eri_batch(b, [[2, 3, 0, 1]])[0], ref.transpose(2, 3, 0, 1), rtol=0, atol=1e-13 * np.abs(ref).max())
    assert np.allclose(oracle.eri_batch(b, [[3, 2, 1, 0]])[0], ref.transpose(3, 2, 1, 0), rtol=0, atol=1e-13 * np.abs(ref).max())


def test_translation_scaling_reflection():
    ls = [2, 1, 3, 2]
    b = _rand_basis(21, ls)
    q = [[0, 1, 2, 3]]
    ref = oracle.eri_batch(b, q)[0]
    sc = np.abs(ref).max()
    # translation
    b2 = dict(b); b2["centers"] = b["centers"] + np.array([3.1, -2.2, 0.7])
    assert np.abs(oracle.eri_batch(b2, q)[0] - ref).max() < 1e-12 * sc
    # scaling r -> r/lam, alpha -> lam^2 alpha, renormalised shells: integrals x lam
    lam = 1.7
    exps = [b["exps"][b["prim_off"][i]:b["prim_off"][i + 1]] * lam ** 2 for i in range(4)]
    coefs = []
    for i, l in enumerate(ls):
        c = b["coefs"][b["prim_off"][i]:b["prim_off"][i + 1]]
        # normalised coefficients scale as alpha^((2l+3)/4) -> lam^(l+3/2)
        coefs.append(c * lam ** (l + 1.5))
    b3 = wl.make_basis(ls, exps, coefs, b["centers"] / lam)
    assert np.abs(oracle.eri_batch(b3, q)[0] - lam * ref).max() < 1e-12 * lam * sc
    # reflection x -> -x: S_lm parity in x is (-1)^(number of x factors); rows with odd x-power flip
    b4 = dict(b); b4["centers"] = b["centers"] * np.array([-1.0, 1.0, 1.0])
    got = oracle.eri_batch(b4, q)[0]
    sign = []
    for l in ls:
        T = oracle.c2s_matrix(l)
        comps = [(i, j, l - i - j) for i in range(l, -1, -1) for j in range(l - i, -1, -1)]
        s = []
        for row in T:
            k = np.nonzero(np.abs(row) > 1e-12)[0][0]
            s.append(-1.0 if comps[k][0] % 2 else 1.0)
        sign.append(np.array(s))
    full = sign[0][:, None, None, None] * sign[1][None, :, None, None] * sign[2][None, None, :, None] * sign[3][None, None, None, :]
    assert np.abs(got - full * ref).max() < 1e-12 * sc


def test_axis_permutation_p_shells():
    """Cyclic relabelling x->y->z->x of all centres permutes p components (order y,z,x)."""
    b = _rand_basis(31, [1, 1, 1, 1])
    q = [[0, 1, 2, 3]]
    ref = oracle.eri_batch(b, q)[0]
    b2 = dict(b); b2["centers"] = b["centers"][:, [2, 0, 1]]      # new (x,y,z) = old (z,x,y)
    got = oracle.eri_batch(b2, q)[0]
    # new component 'y' (row 0) is old 'x' (row 2); new 'z' (row 1) is old 'y' (row 0); new 'x' (row 2) is old 'z' (row 1)
    perm = [2, 0, 1]
    assert np.abs(got - ref[np.ix_(perm, perm, perm, perm)]).max() < 1e-13 * np.abs(ref).max()


def test_linearity_in_primitives():
    rng = np.random.default_rng(41)
    ls = [2, 1, 1, 2]
    b = _rand_basis(42, ls, kmax=3)
    ref = oracle.eri_batch(b, [[0, 1, 2, 3]])[0]
    acc = np.zeros_like(ref)
    off = b["prim_off"]
    for idx in itertools.product(*[range(off[i + 1] - off[i]) for i in range(4)]):
        exps = [[b["exps"][off[i] + idx[i]]] for i in range(4)]
        b1 = wl.make_basis(ls, exps, [[1.0]] * 4, b["centers"])
        cf = np.prod([b["coefs"][off[i] + idx[i]] for i in range(4)])
        acc += cf * oracle.eri_batch(b1, [[0, 1, 2, 3]])[0]
    assert np.abs(acc - ref).max() < 1e-13 * np.abs(ref).max()
    del rng


def test_schwarz_and_positive_diagonal():
    b = _rand_basis(51, [1, 2, 0, 3, 2, 1])
    for (a, bb), (c, d) in itertools.product([(0, 1), (3, 2), (4, 5)], repeat=2):
        abab = oracle.eri_batch(b, [[a, bb, a, bb]])[0]
        cdcd = oracle.eri_batch(b, [[c, d, c, d]])[0]
        abcd = oracle.eri_batch(b, [[a, bb, c, d]])[0]
        da = np.einsum("ijij->ij", abab)
        dc = np.einsum("ijij->ij", cdcd)
        assert (da > -1e-14).all() and (dc > -1e-14).all()
        bound = np.sqrt(np.abs(da))[:, :, None, None] * np.sqrt(np.abs(dc))[None, None, :, :]
        assert (np.abs(abcd) <= bound * (1 + 1e-10) + 1e-14).all()


def test_repeated_shells_and_coincident_centres():
    """T = 0 and A = B paths: compare HGP with MD on degenerate quartets."""
    b = _rand_basis(61, [2, 1, 2, 1])
    b["centers"][1] = b["centers"][0]
    for q in ([0, 0, 0, 0], [0, 1, 0, 1], [2, 2, 3, 3], [1, 1, 1, 1]):
        r0, r2 = oracle.eri_batch(b, [q], mode=0), oracle.eri_batch(b, [q], mode=2)
        assert np.abs(r0 - r2).max() < 2e-12 * np.abs(r0).max()


def test_class_mismatch_rejected():
    b = _rand_basis(71, [1, 1, 2, 2])
    with pytest.raises(ValueError):
        oracle.eri_batch(b, [[0, 1, 2, 3], [2, 1, 2, 3]])
