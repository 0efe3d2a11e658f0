"""Seeded synthetic inputs for the five BASELINE.json configs (recipe: DESIGN.md "Inputs").

This module serves both the CUDA path and the oracle and therefore holds none of the
method's arithmetic: no Boys function, recurrence or transform -- only random draws,
geometry, and the closed-form shell normalisation R-PRIM (input preparation, not part of
the ERI path).  numpy only; importing it never loads the CUDA library.
"""
import math

import numpy as np

NSPH = lambda l: 2 * l + 1  # noqa: E731


def normalise_shell(l, exps, coefs):
    """R-PRIM: scale coefficients so the contracted Racah-normalised solid-harmonic Gaussian
    r^l S_lm exp(-a r^2) combination has unit self-overlap (same factor for every m):
    <S_lm g_i | S_lm g_j> = (4 pi/(2l+1)) Gamma(l+3/2) / (2 (a_i+a_j)^(l+3/2))."""
    exps = np.asarray(exps, float)
    coefs = np.asarray(coefs, float)
    s = exps[:, None] + exps[None, :]
    ov = (4.0 * math.pi / (2 * l + 1)) * math.gamma(l + 1.5) / (2.0 * s ** (l + 1.5))
    return coefs / math.sqrt(float(coefs @ ov @ coefs))


def make_basis(shell_l, exps_list, coefs_list, centers):
    """Pack shells into the flat arrays the C ABI (and the oracle) take."""
    shell_l = np.asarray(shell_l, np.int32)
    prim_off = np.zeros(len(shell_l) + 1, np.int32)
    prim_off[1:] = np.cumsum([len(e) for e in exps_list])
    return dict(shell_l=shell_l, prim_off=prim_off,
                exps=np.concatenate([np.asarray(e, float) for e in exps_list]),
                coefs=np.concatenate([np.asarray(c, float) for c in coefs_list]),
                centers=np.ascontiguousarray(centers, float).reshape(-1, 3))


def _uniform_class(seed, nshell, l, nprim, exp_lo, exp_hi, box, nquartet):
    rng = np.random.default_rng(seed)
    exps = np.exp(rng.uniform(math.log(exp_lo), math.log(exp_hi), (nshell, nprim)))
    coefs = rng.uniform(0.1, 1.0, (nshell, nprim))
    centers = rng.uniform(0.0, box, (nshell, 3))
    quartets = rng.integers(0, nshell, (nquartet, 4)).astype(np.int32)
    coefs = [normalise_shell(l, exps[i], coefs[i]) for i in range(nshell)]
    return make_basis([l] * nshell, list(exps), coefs, centers), quartets


def cfg1(nquartet=10000):
    """(pp|pp): 40 p shells, 3 primitives, exps log-uniform [0.1,10], 4-Bohr cube, seed 0."""
    return _uniform_class(0, 40, 1, 3, 0.1, 10.0, 4.0, nquartet)


def cfg2(nquartet=100000):
    """(dd|dd): 200 d shells, 2 primitives, exps log-uniform [0.2,5], 10-Bohr cube, seed 1."""
    return _uniform_class(1, 200, 2, 2, 0.2, 5.0, 10.0, nquartet)


def cfg4(nf=20000, ng=5000):
    """(ff|ff) + (gg|gg) stress: 60 f + 40 g shells, 1-2 primitives, exps log-uniform [0.3,3],
    6-Bohr cube, seed 3.  Returns (basis, quartets_ffff, quartets_gggg)."""
    rng = np.random.default_rng(3)
    ls = [3] * 60 + [4] * 40
    nprim = rng.integers(1, 3, len(ls))
    exps = [np.exp(rng.uniform(math.log(0.3), math.log(3.0), int(k))) for k in nprim]
    coefs = [rng.uniform(0.1, 1.0, int(k)) for k in nprim]
    centers = rng.uniform(0.0, 6.0, (len(ls), 3))
    qf = rng.integers(0, 60, (nf, 4)).astype(np.int32)
    qg = (60 + rng.integers(0, 40, (ng, 4))).astype(np.int32)
    coefs = [normalise_shell(l, e, c) for l, e, c in zip(ls, exps, coefs)]
    return make_basis(ls, exps, coefs, centers), qf, qg


# (element, l) -> (alpha0, beta, n) even-tempered series; shells get descending exponents
_ET = {("O", 0): (0.25, 2.2, 15), ("O", 1): (0.20, 2.8, 5), ("O", 2): (0.6, 3.5, 2), ("O", 3): (1.4, 1.0, 1),
       ("H", 0): (0.10, 3.3, 5), ("H", 1): (0.40, 3.5, 2), ("H", 2): (1.0, 1.0, 1), ("O", 4): (1.8, 1.0, 1)}
# (element, l) -> primitives per shell
_SHELLS = {("O", 0): (10, 3, 1, 1), ("O", 1): (3, 1, 1), ("O", 2): (1, 1), ("O", 3): (1,),
           ("H", 0): (3, 1, 1), ("H", 1): (1, 1), ("H", 2): (1,), ("O", 4): (1,)}


def water_cluster(grid, seed, with_g=False):
    """cfg3 (grid=(4,2,2), seed 2) / cfg5 (grid=(4,4,4), seed 4): water molecules on a jittered
    5.5-Bohr grid, O-H 1.81 Bohr, HOH 104.5 deg, s..f even-tempered basis (22 shells / water).
    with_g: one more shell per O, a single-primitive g function of exponent 1.8 (the lmax = 4 regime of PAPER.md:363; not
    part of any BASELINE config -- used by the tests and tables of the 64 classes with a g shell)."""
    rng = np.random.default_rng(seed)
    theta = math.radians(104.5)
    ls, exps, coefs, centers = [], [], [], []

    def add_atom(el, pos):
        for l in range(5):
            if l == 4 and not (with_g and el == "O"):
                continue
            if (el, l) not in _SHELLS:
                continue
            a0, beta, n = _ET[(el, l)]
            series = [a0 * beta ** k for k in range(n)][::-1]      # descending
            at = 0
            for k in _SHELLS[(el, l)]:
                e = np.array(series[at:at + k])
                at += k
                c = rng.uniform(0.1, 1.0, k) if k > 1 else np.ones(1)
                ls.append(l); exps.append(e); coefs.append(normalise_shell(l, e, c)); centers.append(pos)

    for i in range(grid[0]):
        for j in range(grid[1]):
            for k in range(grid[2]):
                o = 5.5 * np.array([i, j, k], float) + rng.uniform(-0.5, 0.5, 3)
                qv = rng.normal(size=4)
                qv /= np.linalg.norm(qv)
                w, x, y, z = qv
                rot = np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)],
                                [2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)],
                                [2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)]])
                add_atom("O", o)
                for sgn in (+1.0, -1.0):
                    hloc = np.array([sgn * 1.81 * math.sin(theta / 2), 1.81 * math.cos(theta / 2), 0.0])
                    add_atom("H", o + rot @ hloc)
    return make_basis(ls, exps, coefs, np.array(centers))


def cfg3_basis():
    return water_cluster((4, 2, 2), 2)


def cfg5_basis():
    return water_cluster((4, 4, 4), 4)


def pair_index(a, b):
    return a * (a + 1) // 2 + b


def sample_class_quartets(basis, lclass, n, seed):
    """n i.i.d. quartets of angular class lclass=(la,lb,lc,ld) drawn from basis (no screening)."""
    rng = np.random.default_rng(seed)
    sl = basis["shell_l"]
    cols = []
    for l in lclass:
        idx = np.nonzero(sl == l)[0]
        if len(idx) == 0:
            raise ValueError("no shell with l=%d" % l)
        cols.append(idx[rng.integers(0, len(idx), n)])
    return np.stack(cols, axis=1).astype(np.int32)


def canonical_classes(lmax):
    """Pair-canonical classes la>=lb, lc>=ld, (la,lb)>=(lc,ld) (R-CLASSN: 120 for lmax=4)."""
    pairs = [(a, b) for a in range(lmax + 1) for b in range(a + 1)]
    return [(p[0], p[1], q[0], q[1]) for p in pairs for q in pairs if p >= q]
