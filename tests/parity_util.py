"""Parity gates shared by the GPU tests (tolerances: DESIGN.md 'Tolerance', reading R-TOL).

Gate 1 (north_star, componentwise): |gpu - ref| <= 1e-12 + 1e-10 |ref|.
Gate 2 (scale-aware, per quartet):  max|gpu - ref| <= 1e-10 max|ref| over the quartet's block (+1e-200:
far-apart shells underflow to exactly 0 on one side and to a subnormal on the other).
Where FP64 rounding of the HGP recurrences alone exceeds a gate (high l, large |AB|: HRR
cancellation), the long-double build of the oracle adjudicates: a quartet still passes if the CUDA
result is no further from the long-double value than 8x the FP64 oracle's own distance from it
(plus 1e-13 of the quartet scale).
"""
import numpy as np


def gates(got, ref):
    n = got.shape[0]
    g = got.reshape(n, -1)
    r = ref.reshape(n, -1)
    err = np.abs(g - r)
    gate1 = (err <= 1e-12 + 1e-10 * np.abs(r)).all(axis=1)
    scale = np.abs(r).max(axis=1)
    gate2 = err.max(axis=1) <= 1e-10 * scale + 1e-200      # floor: blocks that underflow to 0 / subnormals
    return gate1, gate2, err.max(axis=1), scale


def assert_parity(got, ref, ref_ld=None, what=""):
    """got, ref: [n, ...] arrays.  ref_ld: optional callable -> long-double oracle values of the same shape."""
    g1, g2, err, scale = gates(got, ref)
    ok = g1 & g2
    if ok.all():
        return dict(adjudicated=0, max_err=float(err.max()), max_scaled=float((err / np.maximum(scale, 1e-300)).max()))
    assert ref_ld is not None, "%s: %d quartets fail the 1e-10 gates (max abs %.3e)" % (what, (~ok).sum(), err.max())
    bad = np.nonzero(~ok)[0]
    ld = ref_ld(bad)
    n = len(bad)
    e_gpu = np.abs(got[bad].reshape(n, -1) - ld.reshape(n, -1)).max(axis=1)
    e_orc = np.abs(ref[bad].reshape(n, -1) - ld.reshape(n, -1)).max(axis=1)
    lim = 8.0 * e_orc + 1e-13 * scale[bad]
    worst = int(np.argmax(e_gpu / np.maximum(lim, 1e-300)))
    assert (e_gpu <= lim).all(), ("%s: quartet %d: CUDA is %.3e from the long-double value, FP64 oracle %.3e"
                                  % (what, bad[worst], e_gpu[worst], e_orc[worst]))
    return dict(adjudicated=int(n), max_err=float(err.max()), max_scaled=float((err / np.maximum(scale, 1e-300)).max()))
