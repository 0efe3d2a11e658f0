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


_SO_LD = os.path.join(_HERE, "liberi_oracle_ld.so")
_lib_ld = None


def build_long_double(force=False):
    """Adjudicator for reading R-TOL: the SAME source compiled with every `double` replaced by
    `long double` (x87 80-bit) and libm calls by their l-variants; a thin wrapper converts the
    double I/O arrays.  No arithmetic differs from eri_oracle.c; only the rounding does."""
    import re
    if force or not os.path.exists(_SO_LD) or os.path.getmtime(_SO_LD) < os.path.getmtime(_SRC):
        src = open(_SRC).read()
        src = re.sub(r"\bdouble\b", "long double", src)
        for fn in ("exp", "sqrt", "erf", "pow", "cos", "fabs"):
            src = re.sub(r"\b%s\(" % fn, fn + "l(", src)
        src += """
int orc_ld_batch(int nshell, const int32_t *shell_l, const int32_t *prim_off, const DIO *exps, const DIO *coefs,
                 const DIO *centers, const int32_t *quartets, int64_t n, int mode, int nthreads, DIO *out, int64_t nout_per)
{
    int np = prim_off[nshell];
    long double *e = malloc(sizeof(long double) * np), *c = malloc(sizeof(long double) * np);
    long double *r = malloc(sizeof(long double) * 3 * nshell), *o = malloc(sizeof(long double) * n * nout_per);
    for (int i = 0; i < np; ++i) { e[i] = exps[i]; c[i] = coefs[i]; }
    for (int i = 0; i < 3 * nshell; ++i) r[i] = centers[i];
    int rc = orc_eri_batch(nshell, shell_l, prim_off, e, c, r, quartets, n, mode, nthreads, o);
    for (int64_t i = 0; i < n * nout_per; ++i) out[i] = (DIO)o[i];
    free(e); free(c); free(r); free(o);
    return rc;
}
""".replace("DIO", "double")
        tmp = os.path.join(_HERE, "_eri_oracle_ld.c")
        with open(tmp, "w") as f:
            f.write(src)
        try:
            subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-w", "-o", _SO_LD, tmp, "-lm"])
        finally:
            os.remove(tmp)
    return _SO_LD


def eri_batch_long_double(basis, quartets, mode=0, nthreads=0):
    """eri_batch evaluated in long double, rounded to FP64 on output (adjudication only)."""
    global _lib_ld
    if _lib_ld is None:
        build_long_double()
        _lib_ld = ctypes.CDLL(_SO_LD)
        _lib_ld.orc_ld_batch.restype = ctypes.c_int
    q = np.ascontiguousarray(quartets, dtype=np.int32).reshape(-1, 4)
    sl = np.ascontiguousarray(basis["shell_l"], dtype=np.int32)
    po = np.ascontiguousarray(basis["prim_off"], dtype=np.int32)
    ex = np.ascontiguousarray(basis["exps"], dtype=np.float64)
    co = np.ascontiguousarray(basis["coefs"], dtype=np.float64)
    ce = np.ascontiguousarray(basis["centers"], dtype=np.float64)
    ls = [int(sl[s]) for s in q[0]]
    out = np.zeros((len(q),) + tuple(2 * l + 1 for l in ls))
    vp = lambda a: ctypes.c_void_p(a.ctypes.data)   # noqa: E731
    rc = _lib_ld.orc_ld_batch(ctypes.c_int(len(sl)), vp(sl), vp(po), vp(ex), vp(co), vp(ce), vp(q),
                              ctypes.c_int64(len(q)), ctypes.c_int(mode), ctypes.c_int(nthreads), vp(out),
                              ctypes.c_int64(int(np.prod(out.shape[1:]))))
    if rc != 0:
        raise ValueError("oracle(long double): quartet list is not of one angular class")
    return out


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


# ----------------------------------------------------------------------------- J / K
def bf_offsets(basis):
    """first spherical basis function of each shell (functions m = -l..l of a shell are consecutive), and nbf."""
    n = 2 * np.asarray(basis["shell_l"], dtype=np.int64) + 1
    off = np.concatenate([[0], np.cumsum(n)])
    return off[:-1].astype(np.int32), int(off[-1])


def eri_tensor(basis, nthreads=0):
    """the DENSE tensor (mn|ls) over all spherical basis functions: every ORDERED shell quartet is evaluated on
    its own (no permutational symmetry is used), class by class.  Tiny bases only (nbf^4 doubles)."""
    sl = np.asarray(basis["shell_l"])
    off, nbf = bf_offsets(basis)
    T = np.zeros((nbf,) * 4)
    ns = len(sl)
    idx = np.array(np.meshgrid(*[np.arange(ns)] * 4, indexing="ij")).reshape(4, -1).T
    lq = sl[idx]
    for cls in sorted(set(map(tuple, lq.tolist()))):
        q = idx[(lq == np.array(cls)).all(axis=1)].astype(np.int32)
        blk = eri_batch(basis, q, nthreads=nthreads)
        for r, (a, b, c, d) in enumerate(q):
            T[off[a]:off[a] + 2 * cls[0] + 1, off[b]:off[b] + 2 * cls[1] + 1,
              off[c]:off[c] + 2 * cls[2] + 1, off[d]:off[d] + 2 * cls[3] + 1] = blk[r]
    return T


def jk_dense(basis, D, nthreads=0):
    """the definition (PAPER.md:291 'J_cd += sum_ab D_ab I[a,b,c,d]', K analogue):
    J_mn = sum_ls D_ls (mn|ls),  K_mn = sum_ls D_ls (ml|ns), from the dense tensor."""
    T = eri_tensor(basis, nthreads)
    J = np.einsum("mnls,ls->mn", T, D)
    K = np.einsum("mlns,ls->mn", T, D)
    return J, K


# ----------------------------------------------------------------------------- first derivatives
_SRC_GRAD = os.path.join(_HERE, "eri_grad_oracle.c")
_SO_GRAD = os.path.join(_HERE, "liberi_grad_oracle.so")
_lib_grad = None


def build_grad(force=False):
    """Compile eri_grad_oracle.c (with eri_oracle.c for orc_boys / orc_c2s_matrix) with gcc (-O2, OpenMP)."""
    newest = max(os.path.getmtime(_SRC), os.path.getmtime(_SRC_GRAD))
    if force or not os.path.exists(_SO_GRAD) or os.path.getmtime(_SO_GRAD) < newest:
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", _SO_GRAD, _SRC_GRAD, _SRC, "-lm"])
    return _SO_GRAD


def eri_grad_batch(basis, quartets, nthreads=0):
    """d(ab|cd)/dR for a same-class quartet list, from the definition (eri_grad_oracle.c).

    Returns f64[n, 12, nsph(la), nsph(lb), nsph(lc), nsph(ld)], derivative index 3 * centre + axis (centre = column of
    the quartet, axis = x, y, z).  A shell that stands in several columns is differentiated column by column."""
    global _lib_grad
    if _lib_grad is None:
        build_grad()
        _lib_grad = ctypes.CDLL(_SO_GRAD)
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int32)
        _lib_grad.orc_eri_grad_batch.argtypes = [ctypes.c_int, ip, ip, dp, dp, dp, ip, ctypes.c_int64, ctypes.c_int, dp]
        _lib_grad.orc_eri_grad_batch.restype = ctypes.c_int
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
    out = np.zeros((n, 12) + tuple(2 * l + 1 for l in ls))
    rc = _lib_grad.orc_eri_grad_batch(len(sl), _ip(sl), _ip(po), _dp(ex), _dp(co), _dp(ce), _ip(q), n, int(nthreads), _dp(out))
    if rc != 0:
        raise ValueError("gradient oracle: quartet list is not of one angular class (or l > 4)")
    return out


_SO_GRAD_LD = os.path.join(_HERE, "liberi_grad_oracle_ld.so")
_lib_grad_ld = None


def build_grad_long_double(force=False):
    """Adjudicator for the derivative gates: eri_oracle.c + eri_grad_oracle.c with every `double` replaced by `long double`
    (the same textual substitution as build_long_double) and a wrapper that converts the double I/O arrays."""
    import re
    newest = max(os.path.getmtime(_SRC), os.path.getmtime(_SRC_GRAD))
    if force or not os.path.exists(_SO_GRAD_LD) or os.path.getmtime(_SO_GRAD_LD) < newest:
        src = open(_SRC).read() + "\n" + open(_SRC_GRAD).read()
        src = re.sub(r"\bdouble\b", "long double", src)
        for fn in ("exp", "sqrt", "erf", "pow", "cos", "fabs"):
            src = re.sub(r"\b%s\(" % fn, fn + "l(", src)
        src += """
int orc_ld_grad_batch(int nshell, const int32_t *shell_l, const int32_t *prim_off, const DIO *exps, const DIO *coefs,
                      const DIO *centers, const int32_t *quartets, int64_t n, int nthreads, DIO *out, int64_t nout_per)
{
    int np = prim_off[nshell];
    long double *e = malloc(sizeof(long double) * np), *c = malloc(sizeof(long double) * np);
    long double *r = malloc(sizeof(long double) * 3 * nshell), *o = malloc(sizeof(long double) * n * nout_per);
    for (int i = 0; i < np; ++i) { e[i] = exps[i]; c[i] = coefs[i]; }
    for (int i = 0; i < 3 * nshell; ++i) r[i] = centers[i];
    int rc = orc_eri_grad_batch(nshell, shell_l, prim_off, e, c, r, quartets, n, nthreads, o);
    for (int64_t i = 0; i < n * nout_per; ++i) out[i] = (DIO)o[i];
    free(e); free(c); free(r); free(o);
    return rc;
}
""".replace("DIO", "double")
        tmp = os.path.join(_HERE, "_eri_grad_oracle_ld.c")
        with open(tmp, "w") as f:
            f.write(src)
        try:
            subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-w", "-o", _SO_GRAD_LD, tmp, "-lm"])
        finally:
            os.remove(tmp)
    return _SO_GRAD_LD


def eri_grad_batch_long_double(basis, quartets, nthreads=0):
    """eri_grad_batch evaluated in long double, rounded to FP64 on output (adjudication only)."""
    global _lib_grad_ld
    if _lib_grad_ld is None:
        build_grad_long_double()
        _lib_grad_ld = ctypes.CDLL(_SO_GRAD_LD)
        _lib_grad_ld.orc_ld_grad_batch.restype = ctypes.c_int
    q = np.ascontiguousarray(quartets, dtype=np.int32).reshape(-1, 4)
    sl = np.ascontiguousarray(basis["shell_l"], dtype=np.int32)
    po = np.ascontiguousarray(basis["prim_off"], dtype=np.int32)
    ex = np.ascontiguousarray(basis["exps"], dtype=np.float64)
    co = np.ascontiguousarray(basis["coefs"], dtype=np.float64)
    ce = np.ascontiguousarray(basis["centers"], dtype=np.float64)
    ls = [int(sl[s]) for s in q[0]]
    out = np.zeros((len(q), 12) + tuple(2 * l + 1 for l in ls))
    vp = lambda a: ctypes.c_void_p(a.ctypes.data)   # noqa: E731
    rc = _lib_grad_ld.orc_ld_grad_batch(ctypes.c_int(len(sl)), vp(sl), vp(po), vp(ex), vp(co), vp(ce), vp(q),
                                        ctypes.c_int64(len(q)), ctypes.c_int(nthreads), vp(out),
                                        ctypes.c_int64(int(np.prod(out.shape[1:]))))
    if rc != 0:
        raise ValueError("gradient oracle (long double): quartet list is not of one angular class")
    return out
