"""Schwarz screening for the water-cluster configs (reading R-SCHWARZ):
Q_ab = sqrt(max over the spherical components of |(ab|ab)|), evaluated by the library itself on the
GPU; a unique quartet (a>=b, c>=d, pair(ab)>=pair(cd)) survives iff Q_ab * Q_cd > threshold.
List logic only -- the integrals come from rcg_eri_batch.  `screened_pass` runs a whole config-3 /
config-5 pass in device batches per angular class: pair lists sorted by Q (and bucketed by the pair's
primitive count, so that every batch has one K4), surviving ket prefixes counted on the device, quartet
lists written by rcg_quartets_from_pairs, one rcg_eri_batch per batch into a reused output buffer.
`sample_screened_quartets` gives the seeded class-stratified samples the parity tests check against
the oracle."""
import numpy as np

from . import rcg, sharding


HBM_GBS = 6543.1      # measured copy bandwidth of this pool's B200s (MEASURED_PEAKS.json, driver-written), for the pass tables


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
            qs.append(rcg.schwarz_from_blocks(out, na * nb).cpu().numpy())
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


def screened_pass(B, basis, bounds=None, threshold=1e-10, out_bytes=1 << 31, classes=None, bucket_k=True,
                  digest=False, max_quartets=None, jk=None, fused=True, rank=0, world=1, grad=False):
    """Every unique quartet with Q_ab Q_cd > threshold, class by class, in device batches.
    Returns {class: dict(quartets, batches, ms, flops[, sum_abs])}; ms = CUDA-event time of list generation +
    rcg_eri_batch calls of the class (the Schwarz pass is `schwarz_bounds`, timed by the caller).
    max_quartets: stop a class after that many quartets (its stats then cover what was run).
    jk = (D, bf_off, Jt, Kt): every batch is digested into Jt, Kt (see fock_pass): by rcg_fock_batch (fused=True: no block buffer
    in HBM) or by rcg_eri_batch + rcg_jk_digest over the 2 GiB output buffer (fused=False).
    grad: rcg_eri_grad_batch (twelve derivative blocks per quartet) instead of rcg_eri_batch, for the classes it supports; the others are
    counted in stats[cls]["skipped"] and not run.
    rank, world: this process evaluates only its share of every unit (sharding.shard_rows: a contiguous range of bra pairs with about
    1/world of the unit's quartets); the stats then count this rank's quartets."""
    import torch
    if bounds is None:
        bounds = schwarz_bounds(B, basis)
    dev = "cuda"
    nprim = np.diff(np.asarray(basis["prim_off"]))
    # sub-lists: (pair type, K2 = Ka*Kb) -> pairs sorted by decreasing Q
    subs = []
    for typ in sorted(bounds):
        pairs, q = bounds[typ]
        keep = q > 0
        pairs, q = pairs[keep], q[keep]
        k2 = nprim[pairs[:, 0]] * nprim[pairs[:, 1]] if bucket_k else np.zeros(len(pairs), int)
        for kv in sorted(set(k2.tolist()), reverse=True):
            m = k2 == kv
            o = np.argsort(-q[m], kind="stable")
            subs.append(dict(typ=typ, k2=int(kv) if bucket_k else None,
                             pairs=torch.tensor(np.ascontiguousarray(pairs[m][o]), dtype=torch.int32, device=dev),
                             q=torch.tensor(q[m][o], device=dev)))
    stats = {}
    # both buffers are allocated once and reused by every batch (allocator calls stay out of the class times)
    list_rows_cap = (1 << 30) // 16
    out_buf = torch.empty(out_bytes // 8, dtype=torch.float64, device=dev)
    list_buf = torch.empty((min(list_rows_cap, out_bytes // 8), 4), dtype=torch.int32, device=dev)
    warmed = set()
    ws_buf = torch.empty(1, dtype=torch.float64, device=dev)          # scratch of the block-tier classes with side kernels: grown on demand, reused
    for xi, X in enumerate(subs):
        for yi in range(xi + 1):
            Y = subs[yi]
            cls = X["typ"] + Y["typ"]              # X's type >= Y's type: canonical class
            if classes is not None and cls not in classes:
                continue
            st = stats.setdefault(cls, dict(quartets=0, batches=0, ms=0.0, flops=0, sum_abs=0.0, skipped=0))
            if max_quartets is not None and st["quartets"] >= max_quartets:
                continue
            grad_ok = grad and rcg.eri_grad_supported(cls)[0]
            # surviving ket pairs of bra pair i: the prefix of the Q-sorted ket list with Q_j > threshold / Q_i
            need = threshold / X["q"]
            cnt = torch.searchsorted(-Y["q"], -need, right=False)      # number of j with Q_j > need (descending list)
            if xi == yi:
                cnt = torch.minimum(cnt, torch.arange(1, len(cnt) + 1, device=dev))     # unique: j <= i
            offs = torch.zeros(len(cnt) + 1, dtype=torch.int64, device=dev)
            torch.cumsum(cnt, 0, out=offs[1:])
            offs_h = offs.cpu().numpy()
            total = int(offs_h[-1])
            if total == 0:
                continue
            if grad and not grad_ok:
                st["skipped"] += total
                continue
            ncomp = int(np.prod([2 * l + 1 for l in cls])) * (12 if grad else 1)
            oshape = ((12,) if grad else ()) + tuple(2 * l + 1 for l in cls)
            max_rows = max(1, min(out_bytes // (8 * ncomp), list_rows_cap))
            if cls not in warmed:          # first call of a class: kernel attributes, table uploads -- not timed
                warmed.add(cls)
                w = torch.cat([X["pairs"][:1], Y["pairs"][:1]], dim=1).contiguous()
                if grad:
                    rcg.eri_grad_batch(B, cls, w, out=out_buf[:ncomp].view((1,) + oshape))
                else:
                    rcg.eri_batch(B, cls, w, out=out_buf[:ncomp].view((1,) + oshape))
                torch.cuda.synchronize()
            info = rcg.class_info(cls)
            k4 = (X["k2"] * Y["k2"]) if bucket_k else None
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            i0, n_i = (0, len(cnt)) if world == 1 else sharding.shard_rows(offs_h, rank, world)
            e0.record()
            while i0 < n_i:
                # largest i1 with offs[i1]-offs[i0] <= max_rows (at least one bra pair; a single bra pair never
                # exceeds max_rows unless the ket list is longer, then it still goes in one batch)
                i1 = int(np.searchsorted(offs_h, offs_h[i0] + max_rows, side="right")) - 1
                i1 = min(max(i1, i0 + 1), n_i)
                rows = int(offs_h[i1] - offs_h[i0])
                if rows:
                    if rows > list_buf.shape[0] or rows * ncomp > out_buf.numel():      # one bra pair against a very long ket list
                        list_buf = torch.empty((rows, 4), dtype=torch.int32, device=dev)
                        out_buf = torch.empty(max(out_buf.numel(), rows * ncomp), dtype=torch.float64, device=dev)
                    ql = rcg.quartets_from_pairs(X["pairs"], Y["pairs"], offs, i0, i1, rows, out=list_buf)
                    shaped = out_buf[: rows * ncomp].view((rows,) + oshape)
                    need = 0 if grad else rcg.eri_workspace_bytes(B, cls, rows)
                    if need > ws_buf.numel() * 8:
                        ws_buf = torch.empty((need + 7) // 8, dtype=torch.float64, device=dev)
                    if grad:
                        rcg.eri_grad_batch(B, cls, ql, out=shaped, k4=k4 or 0)      # bucketed pair lists: one K4 per batch
                    elif jk is not None and fused:       # integrals digested without leaving the chip (registers, or chunks that stay in the L2)
                        need = rcg.fock_workspace_bytes(B, cls, rows, uniform=bucket_k)
                        if need > ws_buf.numel() * 8:
                            ws_buf = torch.empty((need + 7) // 8, dtype=torch.float64, device=dev)
                        rcg.fock_batch(B, cls, ql, jk[1], jk[0], jk[2], jk[3], workspace=ws_buf, uniform=bucket_k)
                    else:
                        rcg.eri_batch(B, cls, ql, out=shaped, workspace=ws_buf, uniform=bucket_k)      # bucketed pair lists: one K4 per batch
                        if jk is not None:
                            rcg.jk_digest(cls, ql, shaped, jk[1], jk[0], jk[2], jk[3])
                    if digest:
                        st["sum_abs"] += float(shaped.abs().sum())
                    st["quartets"] += rows
                    st["batches"] += 1
                    if k4 is not None:
                        st["flops"] += rows * (info["flops_per_prim_quartet"] * k4 + info["flops_per_quartet"])
                i0 = i1
                if max_quartets is not None and st["quartets"] >= max_quartets:
                    break
            e1.record()
            torch.cuda.synchronize()
            st["ms"] += e0.elapsed_time(e1)
    return stats


def fock_pass(B, basis, D, bounds=None, threshold=1e-10, fused=True, rank=0, world=1, finish=True, **kw):
    """Coulomb and exchange matrices J_mn = sum_ls D_ls (mn|ls), K_mn = sum_ls D_ls (ml|ns) of a SYMMETRIC density
    (CUDA float64 [nbf, nbf]) from one screened pass: every batch of unique quartets is digested by rcg_jk_digest
    (scale factors for the 8-fold symmetry inside), rcg_jk_finish adds the transposes.  fused: rcg_fock_batch (the integrals never
    reach HBM) instead of rcg_eri_batch + rcg_jk_digest.  rank, world: multi-GPU build (one process per GPU, torch.distributed
    initialised by the caller): every rank digests its share of each unit, then one all-reduce of Jt and Kt.  Returns (J, K, stats)."""
    import torch
    nf = 2 * np.asarray(basis["shell_l"], dtype=np.int64) + 1
    off = np.concatenate([[0], np.cumsum(nf)])
    nbf = int(off[-1])
    assert tuple(D.shape) == (nbf, nbf)
    bf_off = torch.tensor(off[:-1].astype(np.int32), device="cuda")
    Jt = torch.zeros((nbf, nbf), dtype=torch.float64, device="cuda")
    Kt = torch.zeros((nbf, nbf), dtype=torch.float64, device="cuda")
    stats = screened_pass(B, basis, bounds, threshold, jk=(D.contiguous(), bf_off, Jt, Kt), fused=fused, rank=rank, world=world, **kw)
    if not finish:          # the caller sums the ranks' Jt, Kt itself (tests emulate the ranks one after the other on one GPU)
        return Jt, Kt, stats
    sharding.allreduce_sum_([Jt, Kt])          # the one collective of a multi-GPU Fock build
    rcg.jk_finish(Jt, Kt)
    return Jt, Kt, stats


def main(argv=None):
    """python -m paper_2605_10312_b200.screening cfg3|cfg5 [--md out.md] [--max-quartets N]
    Runs the whole screened pass of BASELINE.json config 3 (16 waters) or 5 (64 waters) and prints the
    per-class table: quartets, batches, device ms (CUDA events), quartets/s, algorithmic TFLOP/s."""
    import argparse
    import os
    import time
    os.environ.setdefault("CUDA_MODULE_LOADING", "EAGER")     # keep one-time kernel loading out of the class times
    import torch
    from . import workloads
    ap = argparse.ArgumentParser()
    ap.add_argument("config", choices=["cfg3", "cfg5"])
    ap.add_argument("--md", default="")
    ap.add_argument("--max-quartets", type=float, default=0)
    ap.add_argument("--grad", action="store_true", help="also run the pass through rcg_eri_grad_batch (first derivatives) for the classes it supports")
    ap.add_argument("--fock", action="store_true", help="also run the pass with J/K digestion (rcg_jk_digest) of a seeded symmetric density")
    args = ap.parse_args(argv)
    # one process per GPU under torchrun (RANK / LOCAL_RANK / WORLD_SIZE): every rank takes its share of each unit of the pass, J and K are
    # all-reduced once (NCCL); times are the maximum over the ranks, counts the sum; rank 0 reports
    world, rank, local = int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def merged(stats):      # per-class stats of all ranks: quartets, batches, flops summed; ms = the slowest rank
        if world == 1:
            return stats
        keys = sorted(set(k for lst in _gather(stats.keys()) for k in lst))
        t = torch.tensor([[stats.get(k, {}).get(f, 0.0) for f in ("quartets", "batches", "flops", "ms")] for k in keys], dtype=torch.float64, device="cuda")
        tsum, tmax = t.clone(), t.clone()
        dist.all_reduce(tsum, op=dist.ReduceOp.SUM)
        dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
        return {k: dict(quartets=int(tsum[i, 0]), batches=int(tsum[i, 1]), flops=int(tsum[i, 2]), ms=float(tmax[i, 3]), sum_abs=0.0) for i, k in enumerate(keys)}

    def _gather(obj):
        out = [None] * world
        dist.all_gather_object(out, list(obj))
        return out

    basis = workloads.cfg3_basis() if args.config == "cfg3" else workloads.cfg5_basis()
    B = rcg.Basis(basis)
    torch.cuda.synchronize()
    t = time.time()
    bounds = schwarz_bounds(B, basis)
    torch.cuda.synchronize()
    t_schwarz = time.time() - t
    nsurv = survivor_estimate(bounds)
    t = time.time()
    st = merged(screened_pass(B, basis, bounds, max_quartets=int(args.max_quartets) or None, rank=rank, world=world))
    wall = time.time() - t
    peak = rcg.fp64_peak_tflops()
    tq = sum(v["quartets"] for v in st.values())
    tms = sum(v["ms"] for v in st.values())
    tf = sum(v["flops"] for v in st.values())
    lines = ["# %s: full screened pass on one B200" % args.config, "",
             "Command (under gpurun): `python -m paper_2605_10312_b200.screening %s --md <this file>`" % args.config, "",
             "%d shells, %d shell pairs; Schwarz pass (all (ab|ab) blocks through rcg_eri_batch + rcg_schwarz_from_blocks): %.2f s wall; "
             "%d unique quartets with Q_ab Q_cd > 1e-10 (host count from the sorted bounds), %d evaluated."
             % (len(basis["shell_l"]), sum(len(p) for p, _ in bounds.values()), t_schwarz, nsurv, tq), "",
             "Whole pass: **%.1f ms** device time (sum of the per-class CUDA-event times: list generation + rcg_eri_batch), %.2f s wall "
             "including the host-side prefix sums; **%.3e quartets/s**, %.2f TFLOP/s algorithmic = %.1f%% of the measured FP64 peak (%.1f TFLOP/s)."
             % (tms, wall, tq / tms * 1e3, tf / tms * 1e-9, 100 * tf / tms * 1e-9 / peak, peak), "",
             "Pair lists are bucketed by the pair's primitive count, so every batch has one K4; output buffer 2 GiB, reused.", "",
             "| class | tier | quartets | batches | ms | quartets/s | TFLOP/s | frac of FP64 peak | HBM GB/s (16 B + output block per quartet) | frac of %.0f GB/s | bound |" % HBM_GBS,
             "|---|---|---|---|---|---|---|---|---|---|---|"]
    for cls in sorted(st):
        v = st[cls]
        if v["quartets"]:
            gbs = (16 + 8 * int(np.prod([2 * l + 1 for l in cls]))) * v["quartets"] / v["ms"] * 1e-6
            fa, fh = v["flops"] / v["ms"] * 1e-9 / peak, gbs / HBM_GBS
            lines.append("| (%d%d\\|%d%d) | %d | %d | %d | %.2f | %.3e | %.2f | %.3f | %.0f | %.3f | %s |"
                         % (cls + (rcg.class_info(cls)["tier"], v["quartets"], v["batches"], v["ms"], v["quartets"] / v["ms"] * 1e3,
                                   v["flops"] / v["ms"] * 1e-9, fa, gbs, fh, "hbm" if fh > fa else "alu")))
    if args.fock:
        nbf = int((2 * np.asarray(basis["shell_l"]) + 1).sum())
        Dh = np.random.default_rng(0).normal(size=(nbf, nbf))
        D = torch.tensor(Dh + Dh.T, device="cuda")
        res = {}
        for mode, fused in (("fused", True), ("buffered", False)):
            t = time.time()
            J, K, stf = fock_pass(B, basis, D, bounds, max_quartets=int(args.max_quartets) or None, fused=fused, rank=rank, world=world)
            torch.cuda.synchronize()
            stf = merged(stf)
            res[mode] = (J, K, stf, time.time() - t, sum(v["ms"] for v in stf.values()))
        Jf, Kf, stf, wallf, fms = res["fused"]
        Jb, Kb, stb, wallb, bms = res["buffered"]
        dj = float((Jf - Jb).abs().max() / Jb.abs().max())
        dk = float((Kf - Kb).abs().max() / Kb.abs().max())
        lines += ["", "## Fock pass: J/K digestion (`--fock`; SURVEY 8(f) NEXT-1)", "",
                  "Seeded symmetric density, %d basis functions.  **Fused** (`rcg_fock_batch`: digestion in the epilogue of the register- and warp-tier class kernels; "
                  "for the block-tier classes integral chunks of at most 1 GiB between the class kernel and `rcg_jk_digest`): **%.1f ms** device time, %.2f s wall "
                  "= %.2f x the integral-only pass (%.1f ms).  Buffered (round 1: `rcg_eri_batch` into the 2 GiB buffer, then `rcg_jk_digest`): %.1f ms, %.2f s wall.  "
                  "J and K of the two agree to %.1e / %.1e of their largest element; J and K symmetric to %.1e / %.1e."
                  % (nbf, fms, wallf, fms / tms, tms, bms, wallb, dj, dk, float((Jf - Jf.T).abs().max() / Jf.abs().max()), float((Kf - Kf.T).abs().max() / Kf.abs().max())), "",
                  "| class | ms fused | ms buffered | ms integrals only |", "|---|---|---|---|"]
        for cls in sorted(stf):
            if stf[cls]["quartets"]:
                lines.append("| (%d%d\\|%d%d) | %.2f | %.2f | %.2f |" % (cls + (stf[cls]["ms"], stb[cls]["ms"], st[cls]["ms"])))
    if args.grad and world == 1:
        t = time.time()
        sg = screened_pass(B, basis, bounds, max_quartets=int(args.max_quartets) or None, grad=True)
        torch.cuda.synchronize()
        wallg = time.time() - t
        gq = sum(v["quartets"] for v in sg.values())
        gms = sum(v["ms"] for v in sg.values())
        sk = sum(v["skipped"] for v in sg.values())
        ims = sum(st[c]["ms"] for c in sg if sg[c]["quartets"])
        lines += ["", "## First-derivative pass (`--grad`; SURVEY 8(f) NEXT-4)", "",
                  "The same screened lists through `rcg_eri_grad_batch` (twelve derivative blocks per quartet into the 2 GiB buffer, overwritten batch after batch): "
                  "%d quartets of the %d classes the entry point supports in **%.1f ms** device time (%.2f s wall) = %.3e quartets/s, %.1f x the integral-only time of the "
                  "same classes (%.1f ms); %d quartets of %d classes whose block does not fit the shared memory are not run."
                  % (gq, sum(1 for v in sg.values() if v["quartets"]), gms, wallg, gq / max(gms, 1e-9) * 1e3, gms / max(ims, 1e-9), ims, sk, sum(1 for v in sg.values() if v["skipped"])), "",
                  "| class | quartets | ms | quartets/s | output GB/s | ms integrals only |", "|---|---|---|---|---|---|"]
        for cls in sorted(sg):
            v = sg[cls]
            if v["quartets"]:
                gbs = (16 + 96 * int(np.prod([2 * l + 1 for l in cls]))) * v["quartets"] / v["ms"] * 1e-6
                lines.append("| (%d%d\\|%d%d) | %d | %.2f | %.3e | %.0f | %.2f |" % (cls + (v["quartets"], v["ms"], v["quartets"] / v["ms"] * 1e3, gbs, st[cls]["ms"])))
            elif v["skipped"]:
                lines.append("| (%d%d\\|%d%d) | %d not run (unsupported) | | | | %.2f |" % (cls + (v["skipped"], st[cls]["ms"])))
    text = "\n".join(lines) + "\n"
    if world > 1:
        text = text.replace("on one B200", "on %d B200s (one process per GPU; times are the slowest rank's, one NCCL all-reduce of J and K per Fock pass)" % world, 1)
        dist.barrier()
        dist.destroy_process_group()
        if rank != 0:
            return
    print(text)
    if args.md:
        with open(args.md, "w") as f:
            f.write(text)


if __name__ == "__main__":
    main()
