"""Pins of the oracle's J/K: the oracle contracts the DENSE tensor built from every ordered
shell quartet (no symmetry).  Pinned here by what the mathematics fixes: the 8-fold symmetry of the tensor it
builds, a closed form for one s function, a brute-force route over UNIQUE quartets with the paper's scale
factors written as explicit loops over the eight permutations, symmetry of J and K for a
symmetric density, and positivity of the Coulomb energy."""
import itertools

import numpy as np

import oracle
from paper_2605_10312_b200 import workloads


def _tiny_basis(seed=3):
    rng = np.random.default_rng(seed)
    ls = [0, 1, 2, 0, 1]
    exps, coefs, cen = [], [], []
    for l in ls:
        e = np.exp(rng.uniform(np.log(0.4), np.log(2.0), 2))
        exps.append(e)
        coefs.append(workloads.normalise_shell(l, e, rng.uniform(0.3, 1.0, 2)))
        cen.append(rng.uniform(0.0, 2.0, 3))
    return workloads.make_basis(ls, exps, coefs, np.array(cen))


def test_dense_tensor_symmetry_and_jk():
    basis = _tiny_basis()
    off, nbf = oracle.bf_offsets(basis)
    assert nbf == 1 + 3 + 5 + 1 + 3
    T = oracle.eri_tensor(basis)
    # (mn|ls) = (nm|ls) = (mn|sl) = (ls|mn): each ordered quartet was evaluated separately, so this tests the oracle
    scale = np.abs(T).max()
    for perm in ((1, 0, 2, 3), (0, 1, 3, 2), (2, 3, 0, 1)):
        assert np.abs(T - T.transpose(perm)).max() <= 1e-13 * scale
    rng = np.random.default_rng(0)
    D = rng.normal(size=(nbf, nbf))
    D = D + D.T
    J, K = oracle.jk_dense(basis, D)
    assert np.abs(J - J.T).max() <= 1e-12 * np.abs(J).max() and np.abs(K - K.T).max() <= 1e-12 * np.abs(K).max()
    # Coulomb energy of a density is positive: sum D_mn D_ls (mn|ls) > 0 (the tensor is a positive-definite kernel)
    assert np.einsum("mn,mn->", D, J) > 0
    # brute force over UNIQUE shell quartets, the eight permutations written out with weight w (scale factors)
    ns = len(basis["shell_l"])
    nf = 2 * np.asarray(basis["shell_l"]) + 1
    J2, K2 = np.zeros_like(J), np.zeros_like(K)
    pairs = [(a, b) for a in range(ns) for b in range(a + 1)]
    for i, (a, b) in enumerate(pairs):
        for (c, d) in pairs[: i + 1]:
            w = (0.5 if a == b else 1.0) * (0.5 if c == d else 1.0) * (0.5 if (a, b) == (c, d) else 1.0)
            blk = T[off[a]:off[a] + nf[a], off[b]:off[b] + nf[b], off[c]:off[c] + nf[c], off[d]:off[d] + nf[d]]
            for (p, axes) in (((a, b, c, d), (0, 1, 2, 3)), ((b, a, c, d), (1, 0, 2, 3)), ((a, b, d, c), (0, 1, 3, 2)),
                              ((b, a, d, c), (1, 0, 3, 2)), ((c, d, a, b), (2, 3, 0, 1)), ((d, c, a, b), (3, 2, 0, 1)),
                              ((c, d, b, a), (2, 3, 1, 0)), ((d, c, b, a), (3, 2, 1, 0))):
                I = blk.transpose(axes)           # I[p0,p1,p2,p3] = (p0 p1|p2 p3)
                sl = [slice(off[s], off[s] + nf[s]) for s in p]
                J2[sl[0], sl[1]] += w * np.einsum("mnls,ls->mn", I, D[sl[2], sl[3]])
                K2[sl[0], sl[2]] += w * np.einsum("mlns,ls->mn", I, D[sl[1], sl[3]])
    assert np.abs(J2 - J).max() <= 1e-12 * np.abs(J).max()
    assert np.abs(K2 - K).max() <= 1e-12 * np.abs(K).max()


def test_single_s_function_closed_form():
    # one normalised s primitive: J = K = D (ss|ss) with (ss|ss) = 2 sqrt(alpha/pi)
    alpha = 0.8
    basis = workloads.make_basis([0], [np.array([alpha])], [np.array([(2 * alpha / np.pi) ** 0.75])], np.zeros((1, 3)))
    J, K = oracle.jk_dense(basis, np.array([[1.7]]))
    ref = 1.7 * 2.0 * np.sqrt(alpha / np.pi)
    assert abs(J[0, 0] - ref) <= 1e-14 * ref and abs(K[0, 0] - ref) <= 1e-14 * ref
