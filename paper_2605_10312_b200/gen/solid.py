"""Cartesian -> real-solid-harmonic coefficient matrices T^(l) for the kernel generator.

PAPER.md:183-191 (Eq. (8), (10)) only says I_sph = sum t^(l) I_cart and cites refs [5],[14];
reading R-SPH fixes rows m=-l..l of the Racah-normalised real solid harmonics.
Here they are built by the standard three-term recursion on polynomials in (x,y,z):

    S_00 = 1
    S_{l+1, l+1}  = sqrt(2^d (2l+1)/(2l+2)) (x S_{l,l} - (1-d) y S_{l,-l}),   d = delta_{l0}
    S_{l+1,-l-1}  = sqrt(2^d (2l+1)/(2l+2)) (y S_{l,l} + (1-d) x S_{l,-l})
    S_{l+1, m}    = ((2l+1) z S_{l,m} - sqrt((l+m)(l-m)) r^2 S_{l-1,m}) / sqrt((l+m+1)(l-m+1))

(the CPU oracle uses the closed-form triple sum instead; the two share no code).
"""
import math


def cart_comps(l):
    """Cartesian components of level l in the library's internal order (R-SPH):
    for i=l..0: for j=l-i..0: x^i y^j z^(l-i-j)."""
    return [(i, j, l - i - j) for i in range(l, -1, -1) for j in range(l - i, -1, -1)]


def ncart(l):
    return (l + 1) * (l + 2) // 2


def _mul(p, mono, s=1.0):
    return {(k[0] + mono[0], k[1] + mono[1], k[2] + mono[2]): v * s for k, v in p.items()}


def _add(*ps):
    out = {}
    for p in ps:
        for k, v in p.items():
            out[k] = out.get(k, 0.0) + v
    return {k: v for k, v in out.items() if abs(v) > 1e-300}


def _scale(p, s):
    return {k: v * s for k, v in p.items()}


def solid_harmonics(lmax):
    """dict (l,m) -> polynomial {(i,j,k): coef}."""
    S = {(0, 0): {(0, 0, 0): 1.0}}
    X, Y, Z = (1, 0, 0), (0, 1, 0), (0, 0, 1)
    for l in range(lmax):
        d = 1 if l == 0 else 0
        f = math.sqrt((2.0 ** d) * (2 * l + 1) / (2 * l + 2))
        if l == 0:
            S[(1, 1)] = _scale(_mul(S[(0, 0)], X), f)
            S[(1, -1)] = _scale(_mul(S[(0, 0)], Y), f)
        else:
            S[(l + 1, l + 1)] = _scale(_add(_mul(S[(l, l)], X), _mul(S[(l, -l)], Y, -1.0)), f)
            S[(l + 1, -l - 1)] = _scale(_add(_mul(S[(l, l)], Y), _mul(S[(l, -l)], X)), f)
        for m in range(-l, l + 1):
            t = _mul(S[(l, m)], Z, 2 * l + 1)
            if (l - 1, m) in S:
                g = -math.sqrt((l + m) * (l - m))
                lo = S[(l - 1, m)]
                t = _add(t, _mul(lo, (2, 0, 0), g), _mul(lo, (0, 2, 0), g), _mul(lo, (0, 0, 2), g))
            S[(l + 1, m)] = _scale(t, 1.0 / math.sqrt((l + m + 1) * (l - m + 1)))
    return S


_CACHE = {}


def c2s_rows(l):
    """T^(l) as a list of 2l+1 sparse rows [(cart_index, coef), ...], rows m=-l..l."""
    if l not in _CACHE:
        S = solid_harmonics(max(l, 1))
        comps = cart_comps(l)
        rows = []
        for m in range(-l, l + 1):
            p = S[(l, m)]
            row = [(comps.index(k), v) for k, v in sorted(p.items(), key=lambda kv: comps.index(kv[0]))]
            rows.append(row)
        _CACHE[l] = rows
    return _CACHE[l]
