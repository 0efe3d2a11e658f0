"""Parity gates shared by the GPU tests and __graft_entry__.smoke() (tolerances: DESIGN.md section 6, reading R-TOL).

Gate 1 (north_star, componentwise): |gpu - ref| <= 1e-12 + 1e-10 |ref|.
Gate 2 (scale-aware, per quartet):  max|gpu - ref| <= 1e-10 max|ref| over the quartet's block (+1e-200:
far-apart shells underflow to exactly 0 on one side and to a subnormal on the other).

`ref` is the FP64 oracle.  A quartet that passes both gates against it is done.  For f and g shells FP64 rounding of
the HGP recurrences themselves exceeds the gates on some quartets (HRR cancellation at large |AB|; the FP64 oracle is up
to 4.6e-10 (ff|ff) / 3.9e-9 (gg|gg) of the quartet scale from its own long-double build), so a failing quartet is then
compared with the ACCURATE value (the long-double build of the oracle, 1e-13 from the independent MD route):
  * it passes outright if the CUDA result meets Gate 1 and Gate 2 against the accurate value;
  * otherwise it passes only if CUDA is no further from the accurate value than ADJ_FACTOR x the FP64 oracle's own
    distance (+1e-13 of the quartet scale, +1e-14 of the quartet's Schwarz bound Q_ab Q_cd when the caller supplies it): both
    sides then carry the rounding of the same FP64 algorithm.  The Schwarz term is the absolute floor of blocks that vanish by
    symmetry (a (gf| pair on one centre against distant s shells: true values 3e-19, intermediates of order Q_ab Q_cd ~ 1, and
    the FP64 oracle, its independent MD route and both CUDA tiers all sit 5e-18..1e-16 from the long-double value).
ADJ_FACTOR = 4 comes from the measured distribution of that ratio on the B200 (cfg4, first 500 (ff|ff) + 100 (gg|gg) quartets,
216 of them with the oracle beyond 1e-12 of the scale: median 0.9, 99th percentile 2.1, largest 2.64).
allow_adjudication = "direct" admits only the first rule (classes with sum l <= 8 at full config size, where 1 quartet in
100,000 sits at 1.007e-10 of its scale from the FP64 oracle).  Every call returns the counts:
adjudicated (quartets sent to the accurate value), over_accurate_gate (of those, outside 1e-10 of the scale from the
accurate value) and worst_ratio; tests of classes with sum l <= 8 assert adjudicated == 0.
"""
import numpy as np

ADJ_FACTOR = 4.0


def gates(got, ref):
    n = got.shape[0]
    g = got.reshape(n, -1)
    r = ref.reshape(n, -1)
    err = np.abs(g - r)
    gate1 = (err <= 1e-12 + 1e-10 * np.abs(r)).all(axis=1)
    scale = np.abs(r).max(axis=1)
    gate2 = err.max(axis=1) <= 1e-10 * scale + 1e-200      # floor: blocks that underflow to 0 / subnormals
    return gate1, gate2, err.max(axis=1), scale


def literal_metric(got, ref):
    """north_star's piecewise criterion as written: max relative error over |ref| >= 1e-8, max absolute error below."""
    g, r = got.ravel(), ref.ravel()
    big = np.abs(r) >= 1e-8
    rel = float((np.abs(g - r)[big] / np.abs(r)[big]).max()) if big.any() else 0.0
    ab = float(np.abs(g - r)[~big].max()) if (~big).any() else 0.0
    return rel, ab


def assert_parity(got, ref, ref_ld=None, what="", allow_adjudication=False, schwarz=None):
    """got, ref: [n, ...] arrays.  ref_ld: callable(indices) -> accurate (long-double oracle) values of those quartets;
    used only when allow_adjudication is set.  schwarz: optional callable(indices) -> Q_ab Q_cd of those quartets.
    Returns the counts described in the module docstring."""
    g1, g2, err, scale = gates(got, ref)
    ok = g1 & g2
    rel, ab = literal_metric(got, ref)
    res = dict(n=int(len(ok)), adjudicated=0, over_accurate_gate=0, worst_ratio=0.0, max_err=float(err.max()) if len(err) else 0.0,
               max_scaled=float((err / np.maximum(scale, 1e-300)).max()) if len(err) else 0.0, literal_rel=rel, literal_abs=ab)
    if ok.all():
        return res
    assert allow_adjudication and ref_ld is not None, \
        "%s: %d of %d quartets fail the 1e-10 gates against the FP64 oracle (max abs %.3e, max scaled %.3e)" % (
            what, (~ok).sum(), len(ok), err.max(), res["max_scaled"])
    bad = np.nonzero(~ok)[0]
    n = len(bad)
    ld = ref_ld(bad).reshape(n, -1)
    gb, rb = got[bad].reshape(n, -1), ref[bad].reshape(n, -1)
    e_gpu = np.abs(gb - ld).max(axis=1)
    e_orc = np.abs(rb - ld).max(axis=1)
    sc = np.abs(ld).max(axis=1)
    direct = (np.abs(gb - ld) <= 1e-12 + 1e-10 * np.abs(ld)).all(axis=1) & (e_gpu <= 1e-10 * sc + 1e-200)
    ratio = e_gpu / np.maximum(e_orc + 1e-13 * sc / ADJ_FACTOR, 1e-300)
    floor = 1e-13 * sc + (1e-14 * np.asarray(schwarz(bad)) if schwarz is not None else 0.0)
    passed = direct if allow_adjudication == "direct" else direct | (e_gpu <= ADJ_FACTOR * e_orc + floor)
    res.update(adjudicated=int(n), over_accurate_gate=int((e_gpu > 1e-10 * sc + 1e-200).sum()),
               worst_ratio=float(ratio[~direct].max()) if (~direct).any() else 0.0)
    worst = int(np.argmax(np.where(passed, 0.0, ratio)))
    assert passed.all(), ("%s: quartet %d: CUDA is %.3e from the accurate (long-double) value, the FP64 oracle %.3e, scale %.3e"
                          % (what, bad[worst], e_gpu[worst], e_orc[worst], sc[worst]))
    return res
