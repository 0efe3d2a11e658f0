"""Per-class throughput table: quartets/s, GFLOP/s and fraction of the measured FP64 peak for every
generated class, on seeded quartets drawn from the cfg3 water basis (contraction depths 1..10) or,
for (gg|gg), the cfg4 basis.  `--tier 3` forces the table-driven global tier.

    python -m paper_2605_10312_b200.class_bench [--n 20000] [--tier 0|3] [--md out.md]
"""
import argparse
import sys

import numpy as np


def main(argv=None):
    import torch
    from . import rcg, workloads
    ap = argparse.ArgumentParser()
    ap.add_argument("--n", type=int, default=20000)
    ap.add_argument("--tier", type=int, default=0)
    ap.add_argument("--md", default="")
    ap.add_argument("--both", action="store_true", help="time the class's own tier and the global tier")
    ap.add_argument("--sort-k4", action="store_true", help="order each list by decreasing K4 (lets the packed kernels engage)")
    ap.add_argument("--only", default="", help="comma-separated class tags, e.g. 3333,2222")
    ap.add_argument("--headline", action="store_true", help="also time cfg1, cfg2 and cfg4 at full size")
    args = ap.parse_args(argv)
    b3 = workloads.cfg3_basis()
    b4, _, _ = workloads.cfg4(1, 1)
    bg = workloads.water_cluster((4, 2, 2), 2, with_g=True)      # the cfg3 cluster with one g shell per O: classes with a g shell
    B3, B4, Bg = rcg.Basis(b3), rcg.Basis(b4), rcg.Basis(bg)
    peak = rcg.fp64_peak_tflops()
    rows = []
    only = {tuple(int(ch) for ch in t) for t in args.only.split(",") if t}
    for ci, cls in enumerate(rcg.classes()):
        if only and cls not in only:
            continue
        basis, B = (b4, B4) if cls == (4, 4, 4, 4) else ((bg, Bg) if max(cls) == 4 else (b3, B3))
        L = sum(cls)
        n = args.n if L <= 8 else max(500, args.n // (4 ** (L - 8)))
        q = workloads.sample_class_quartets(basis, cls, n, seed=5000 + ci)
        k4q = np.prod(np.diff(basis["prim_off"])[q], axis=1)
        if args.sort_k4:
            q = np.ascontiguousarray(q[np.argsort(-k4q, kind="stable")])
        k4 = int(k4q.sum())
        info = rcg.class_info(cls)
        flops = info["flops_per_prim_quartet"] * k4 + info["flops_per_quartet"] * n
        qd = torch.tensor(q, device="cuda")
        res = {}
        for tier in ([0, 3] if args.both else [args.tier]):
            if tier == 3 and info["tier"] == 3 and args.both:
                res[tier] = res[0]
                continue
            out = rcg.eri_batch(B, cls, qd, tier=tier)
            ws_bytes = rcg.eri_workspace_bytes(B, cls, n, tier)
            ws = torch.empty(max(1, ws_bytes // 8), dtype=torch.float64, device="cuda")
            for _ in range(2):
                rcg.eri_batch(B, cls, qd, out=out, workspace=ws, tier=tier)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            reps = 5
            e0.record()
            for _ in range(reps):
                rcg.eri_batch(B, cls, qd, out=out, workspace=ws, tier=tier)
            e1.record()
            torch.cuda.synchronize()
            res[tier] = e0.elapsed_time(e1) / reps * 1e-3
        t = res[0] if 0 in res else res[args.tier]
        rows.append((cls, info["tier"], n, k4 / n, n / t, flops / t * 1e-9, flops / t * 1e-12 / peak,
                     (n / res[3]) if 3 in res else float("nan")))
    hdr = "| class | tier | quartets | mean K4 | quartets/s | GFLOP/s | frac of measured FP64 peak (%.1f TF) | global tier quartets/s |" % peak
    lines = [hdr, "|---|---|---|---|---|---|---|---|"]
    for (cls, tier, n, k4, qps, gf, fr, gq) in rows:
        lines.append("| (%d%d\\|%d%d) | %d | %d | %.1f | %.3e | %.1f | %.3f | %.3e |" % (*cls, tier, n, k4, qps, gf, fr, gq))
    if args.headline:
        lines += ["", "Headline configs at full size (one call, CUDA events, after 2 warm-up calls; best of 5):", "",
                  "| config | class | tier | quartets | ms | quartets/s | GFLOP/s | frac of peak |", "|---|---|---|---|---|---|---|---|"]
        b1, q1 = workloads.cfg1()
        b2, q2 = workloads.cfg2()
        b4f, qf, qg = workloads.cfg4()
        for name, basis, q, cls in (("cfg1", b1, q1, (1, 1, 1, 1)), ("cfg2", b2, q2, (2, 2, 2, 2)),
                                    ("cfg4", b4f, qf, (3, 3, 3, 3)), ("cfg4", b4f, qg, (4, 4, 4, 4))):
            if only and cls not in only:
                continue
            Bx = rcg.Basis(basis)
            qd = torch.tensor(q, device="cuda")
            n = len(q)
            ws = torch.empty(max(1, rcg.eri_workspace_bytes(Bx, cls, n) // 8), dtype=torch.float64, device="cuda")
            out = rcg.eri_batch(Bx, cls, qd, workspace=ws)
            rcg.eri_batch(Bx, cls, qd, out=out, workspace=ws)
            best = 1e30
            for _ in range(5):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                rcg.eri_batch(Bx, cls, qd, out=out, workspace=ws)
                e1.record()
                torch.cuda.synchronize()
                best = min(best, e0.elapsed_time(e1) * 1e-3)
            info = rcg.class_info(cls)
            k4 = int(np.prod(np.diff(basis["prim_off"])[q], axis=1).sum())
            fl = info["flops_per_prim_quartet"] * k4 + info["flops_per_quartet"] * n
            lines.append("| %s | (%d%d\\|%d%d) | %d | %d | %.3f | %.3e | %.1f | %.3f |"
                         % ((name,) + cls + (info["tier"], n, best * 1e3, n / best, fl / best * 1e-9, fl / best * 1e-12 / peak)))
            del out, ws
    txt = "\n".join(lines)
    print(txt)
    if args.md:
        with open(args.md, "w") as f:
            f.write(txt + "\n")
    return 0


if __name__ == "__main__":
    sys.exit(main())
