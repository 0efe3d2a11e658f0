"""ctypes binding of oracle/eri_oracle.c (TEST INFRASTRUCTURE, not the product).

Every function here only marshals arguments; the arithmetic is in the C file, which cites
the PAPER.md passages it follows.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "eri_oracle.c")
_SO = os.path.join(_HERE, "liberi_oracle.so")
_lib = None


def build(force=False):
    """Compile eri_oracle.c with gcc (-O2, OpenMP).  Building the checker is not using it."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", _SO, _SRC, "-lm"])
    return _SO


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_SO)
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int32)
        lib.orc_boys.argtypes = [ctypes.c_int, ctypes.c_double, dp]
        lib.orc_boys_quadrature.argtypes = [ctypes.c_int, ctypes.c_double, dp]
        lib.orc_c2s_matrix.argtypes = [ctypes.c_int, dp]
        lib.orc_eri_batch.argtypes = [ctypes.c_int, ip, ip, dp, dp, dp, ip, ctypes.c_int64,
                                      ctypes.c_int, ctypes.c_int, dp]
        lib.orc_eri_batch.restype = ctypes.c_int
        lib.orc_num_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def _dp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _ip(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_int32))


def boys(mmax, T):
    """F_0..F_mmax(T) by the oracle's series / erf+upward routine."""
    F = np.zeros(mmax + 1)
    _load().orc_boys(int(mmax), float(T), _dp(F))
    return F


def boys_quadrature(mmax, T):
    """F_0..F_mmax(T) by direct Gauss-Legendre quadrature of the defining integral."""
    F = np.zeros(mmax + 1)
    _load().orc_boys_quadrature(int(mmax), float(T), _dp(F))
    return F


def c2s_matrix(l):
    """(2l+1) x ncart(l) Racah-normalised real solid harmonic coefficients (R-SPH)."""
    T = np.zeros((2 * l + 1, (l + 1) * (l + 2) // 2))
    _load().orc_c2s_matrix(int(l), _dp(T))
    return T


def num_threads():
    return int(_load().orc_num_threads())


def eri_batch(basis, quartets, mode=0, nthreads=0):
    """Spherical ERIs for a same-class quartet list.

    basis: dict with shell_l int32[ns], prim_off int32[ns+1], exps f64[np], coefs f64[np],
           centers f64[ns,3].  quartets: int32[n,4].  mode 0 HGP / 1 HRR-per-primitive / 2 MD.
    Returns f64[n, nsph(la), nsph(lb), nsph(lc), nsph(ld)].
    """
    q = np.ascontiguousarray(quartets, dtype=np.int32).reshape(-1, 4)
    sl = np.ascontiguousarray(basis["shell_l"], dtype=np.int32)
    po = np.ascontiguousarray(basis["prim_off"], dtype=np.int32)
    ex = np.ascontiguousarray(basis["exps"], dtype=np.float64)
    co = np.ascontiguousarray(basis["coefs"], dtype=np.float64)
    ce = np.ascontiguousarray(basis["centers"], dtype=np.float64)
    n = q.shape[0]
    if n == 0:
        return np.zeros((0,))
    ls = [int(sl[s]) for s in q[0]]
    out = np.zeros((n,) + tuple(2 * l + 1 for l in ls))
    rc = _load().orc_eri_batch(len(sl), _ip(sl), _ip(po), _dp(ex), _dp(co), _dp(ce), _ip(q), n,
                               int(mode), int(nthreads), _dp(out))
    if rc != 0:
        raise ValueError("oracle: quartet list is not of one angular class (or l > 4)")
    return out
