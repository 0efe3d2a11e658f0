"""Schwarz screening for the water-cluster configs (reading R-SCHWARZ):
Q_ab = sqrt(max over the spherical components of |(ab|ab)|), evaluated by the library itself on the
GPU; a unique quartet (a>=b, c>=d, pair(ab)>=pair(cd)) survives iff Q_ab * Q_cd > threshold.
Host-side list logic only -- the integrals come from rcg_eri_batch.  The full device-side quartet
pipeline for the ~1e9-quartet passes is SURVEY 8(f) NEXT-2; this module provides the bounds and seeded
class-stratified samples of the surviving quartets, which is what the parity tests need."""
import numpy as np

from . import rcg


def pair_lists(basis):
    """unique shell pairs a >= b grouped by pair type (lhi, llo); each row is (shell with lhi, shell with llo)."""
    sl = np.asarray(basis["shell_l"])
    n = len(sl)
    a, b = np.tril_indices(n)
    swap = sl[a] < sl[b]
    hi = np.where(swap, b, a).astype(np.int32)
    lo = np.where(swap, a, b).astype(np.int32)
    out = {}
    for lh in range(int(sl.max()) + 1):
        for ll in range(lh + 1):
            m = (sl[hi] == lh) & (sl[lo] == ll)
            if m.any():
                out[(lh, ll)] = np.stack([hi[m], lo[m]], axis=1)
    return out


def schwarz_bounds(B, basis, chunk=200000):
    """dict pair type -> (pairs int32[n,2], Q float64[n]) with Q from (ab|ab) blocks computed on the GPU."""
    import torch
    res = {}
    for (lh, ll), pairs in pair_lists(basis).items():
        qs = []
        for s in range(0, len(pairs), chunk):
            p = pairs[s:s + chunk]
            quart = np.concatenate([p, p], axis=1).astype(np.int32)
            out = rcg.eri_batch(B, (lh, ll, lh, ll), torch.tensor(quart, device="cuda"))
            na, nb = 2 * lh + 1, 2 * ll + 1
            diag = out.reshape(len(p), na * nb, na * nb).diagonal(dim1=1, dim2=2)
            qs.append(torch.sqrt(diag.abs().max(dim=1).values).cpu().numpy())
        res[(lh, ll)] = (pairs, np.concatenate(qs))
    return res


def sample_screened_quartets(bounds, cls, n, seed, threshold=1e-10, max_tries=50):
    """n surviving quartets of canonical class cls=(la,lb,lc,ld), seeded rejection sampling over the
    surviving pairs of types (la,lb) and (lc,ld).  Returns int32[m,4], m <= n."""
    la, lb, lc, ld = cls
    if (la, lb) not in bounds or (lc, ld) not in bounds:
        return np.zeros((0, 4), np.int32)
    rng = np.random.default_rng(seed)
    pb, qb = bounds[(la, lb)]
    pk, qk = bounds[(lc, ld)]
    out = []
    got = 0
    for _ in range(max_tries):
        i = rng.integers(0, len(pb), 4 * n)
        j = rng.integers(0, len(pk), 4 * n)
        keep = qb[i] * qk[j] > threshold
        if (la, lb) == (lc, ld):
            keep &= i >= j                      # pair(ab) >= pair(cd) inside one pair type
        sel = np.nonzero(keep)[0][: n - got]
        out.append(np.concatenate([pb[i[sel]], pk[j[sel]]], axis=1))
        got += len(sel)
        if got >= n:
            break
    return np.concatenate(out).astype(np.int32) if out else np.zeros((0, 4), np.int32)


def survivor_estimate(bounds, threshold=1e-10):
    """number of unique quartets with Q_ab Q_cd > threshold (exact count over sorted bounds)."""
    allq = np.sort(np.concatenate([q for (_, q) in bounds.values()]))
    # pairs (i<=j) with q_i q_j > t: for each i count j >= i with q_j > t / q_i
    with np.errstate(divide="ignore"):
        need = threshold / allq
    first = np.searchsorted(allq, need, side="right")
    idx = np.arange(len(allq))
    return int(np.sum(len(allq) - np.maximum(first, idx)))
