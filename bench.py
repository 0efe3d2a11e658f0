#!/usr/bin/env python
"""bench.py -- one JSON line for the headline workload: config[1] of BASELINE.json, 100,000 (dd|dd)
shell quartets (200 d shells, 2 primitives each, K4 = 16) through rcg_eri_batch on one B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--workload cfg2|cfg1] [--class-table out.md]

A step = one pass of the whole hot path (pair quantities, Boys, VRR + contraction, HRR + stepwise
c2s, store) over the batch.  `value` = quartets/s with inputs resident in HBM; `e2e` = the same
through rcg_eri_batch_host with pinned HOST buffers (H2D of the list, D2H of the integrals inside
the timed region).  N > 1: every rank runs the same batch on its own GPU (the path shards over
independent quartets; no collective), value = N * quartets / max-over-ranks time ("weak").
--impl reference times the CPU oracle (oracle/) on a bounded sample on the host cores.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "contracted shell quartets/s per (la lb|lc ld) class; % of B200 FP64 peak"


def hbm_peak():
    """measured copy bandwidth of this pool's B200s (driver-written MEASURED_PEAKS.json), else the profiling guide's fallback."""
    try:
        return float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"
# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the class kernel: NOT measured by this run (ncu cannot run inside
# a timed bench) but taken from the committed ncu --set full capture of the same command, profiles/r2_ncu_eri_warp_2222.md
# (algorithmic bytes: 501.6 MB, almost all output; the tail of the output is still dirty in the 126 MB L2 when the kernel ends)
TRAFFIC = {"cfg2": 444.08e6}
TRAFFIC_SOURCE = "profiles/r2_ncu_eri_warp_2222.md (ncu --set full of this command; not measured in this run)"
UNIT = "quartets/s"


def load_workload(name):
    from paper_2605_10312_b200 import workloads
    if name == "cfg1":
        basis, q = workloads.cfg1()
        return basis, q, (1, 1, 1, 1), "cfg1: 10,000 (pp|pp) quartets, 40 p shells x 3 primitives, seed 0"
    basis, q = workloads.cfg2()
    return basis, q, (2, 2, 2, 2), "cfg2: 100,000 (dd|dd) quartets, 200 d shells x 2 primitives, seed 1"


def prim_quartets(basis, q):
    k = np.diff(basis["prim_off"])[q]
    return int(np.prod(k, axis=1).sum())


class ClockSampler(threading.Thread):
    """nvidia-smi clocks + throttle reasons during the timed region (B200_PROFILING.md recipe)."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index = index
        self.stop = threading.Event()
        self.rows = []

    def run(self):
        q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
        while not self.stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + q,
                                      "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5).stdout
                parts = [p.strip() for p in out.strip().split(",")]
                if len(parts) >= 6:
                    self.rows.append(parts)
            except Exception:
                pass
            self.stop.wait(0.02)

    def summary(self):
        if not self.rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        sm = sorted(float(r[0]) for r in self.rows)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for k, n in enumerate(names) if any(r[2 + k].lower().startswith("active") for r in self.rows)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(self.rows[0][1]), "reasons": reasons,
                "samples": len(self.rows)}


def time_oracle(basis, q, target_s=12.0):
    """oracle (as it stands) on a bounded prefix of the batch, all host cores."""
    import oracle
    oracle.build()
    n = min(len(q), 2000)
    oracle.eri_batch(basis, q[:64])            # thread pool / page-in warm-up, untimed
    t0 = time.time()
    oracle.eri_batch(basis, q[:n])
    dt = max(time.time() - t0, 1e-4)
    n2 = int(min(len(q), max(256, n * target_s / dt)))
    t0 = time.time()
    oracle.eri_batch(basis, q[:n2])
    dt = time.time() - t0
    return n2 / dt, n2, dt, oracle.num_threads()


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    basis, q, cls, wname = load_workload(args.workload)
    vals = []
    for _ in range(args.warmup + args.steps):
        v, n2, dt, cores = time_oracle(basis, q, target_s=max(2.0, 40.0 / max(1, args.steps + args.warmup)))
        vals.append((v, n2, dt))
    vals = vals[args.warmup:]
    value = float(np.mean([v for v, _, _ in vals]))
    sample = "first %d quartets of the batch per step (%.1f s of CPU work per step)" % (vals[-1][1], vals[-1][2])
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * float(np.mean([d for _, _, d in vals])),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": wname, "class": list(cls)},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))
    return 0


def run_class_table(path):
    """quartets/s, GFLOP/s and fraction of the FP64 peak PER CLASS with the oracle's quartets/s on the
    host cores beside it (the cpu_baseline leg, per class): K4-sorted seeded lists from the cfg3 water basis
    (cfg4 basis for (gg|gg)), the oracle on a bounded prefix (about 0.3 s per class), and the largest difference
    between the two on that prefix, scaled by the largest integral of the quartet."""
    import torch
    import oracle
    from paper_2605_10312_b200 import rcg, workloads
    oracle.build()
    b3 = workloads.cfg3_basis()
    b4, _, _ = workloads.cfg4(1, 1)
    bg = workloads.water_cluster((4, 2, 2), 2, with_g=True)      # the cfg3 cluster with one g shell per O: classes with a g shell
    B3, B4, Bg = rcg.Basis(b3), rcg.Basis(b4), rcg.Basis(bg)
    peak = rcg.fp64_peak_tflops()
    lines = ["# Per-class table with the oracle beside it (SURVEY 8(d))", "",
             "Command (under gpurun, one B200): `python bench.py --class-table <this file>`", "",
             "K4-sorted seeded lists of 200,000 quartets per class from the cfg3 water basis (fewer for the heaviest classes; the same cluster with one g shell "
             "per O for the classes with a g shell, cfg4 basis for (gg|gg)); 5 timed calls between CUDA events after 2 warm-up calls.  Oracle: `oracle.eri_batch` as it stands on %d host "
             "threads over an evenly spaced sample of the same list, sized from a 64-quartet probe (0.01 to 0.5 s of wall time); last columns: largest |CUDA - oracle| on that "
             "sample and the number of its quartets with a component outside north_star's criterion |CUDA - oracle| <= 1e-12 + 1e-10 |oracle| "
             "(the tests add a scale-aware gate per quartet and, for f and g shells, the long-double oracle; DESIGN.md section 6).  "
             "Measured FP64 peak %.1f TFLOP/s." % (oracle.num_threads(), peak), "",
             "Bytes per quartet are the algorithmic ones (16-byte index record + the output block; shell data stay in the L2); HBM peak %.0f GB/s, %s.  "
             "`bound` names the roofline the class sits closer to on this list (SURVEY 8(d)): alu = FP64 pipe, hbm = the output store." % hbm_peak(), "",
             "| class | tier | quartets | mean K4 | quartets/s | GFLOP/s | frac of FP64 peak | B/quartet | HBM GB/s | frac of HBM peak | bound | oracle quartets/s | oracle sample | GPU / oracle | max abs diff | quartets outside 1e-12 + 1e-10 rel |",
             "|---|---|---|---|---|---|---|---|---|---|---|---|---|---|---|---|"]
    for ci, cls in enumerate(rcg.classes()):
        basis, B = (b4, B4) if cls == (4, 4, 4, 4) else ((bg, Bg) if max(cls) == 4 else (b3, B3))
        L = sum(cls)
        n = 200000 if L <= 8 else max(500, 200000 // (4 ** (L - 8)))
        q = workloads.sample_class_quartets(basis, cls, n, seed=5000 + ci)
        k4q = np.prod(np.diff(basis["prim_off"])[q], axis=1)
        q = np.ascontiguousarray(q[np.argsort(-k4q, kind="stable")])
        info = rcg.class_info(cls)
        flops = info["flops_per_prim_quartet"] * int(k4q.sum()) + info["flops_per_quartet"] * n
        qd = torch.tensor(q, device="cuda")
        ws = torch.empty(max(1, rcg.eri_workspace_bytes(B, cls, n) // 8), dtype=torch.float64, device="cuda")
        out = rcg.eri_batch(B, cls, qd, workspace=ws)
        rcg.eri_batch(B, cls, qd, out=out, workspace=ws)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(5):
            rcg.eri_batch(B, cls, qd, out=out, workspace=ws)
        e1.record()
        torch.cuda.synchronize()
        t = e0.elapsed_time(e1) / 5 * 1e-3
        # oracle on a spread sample (every stride-th quartet, so the K4 mix is the list's), sized from a probe
        probe = q[:: max(1, n // 8)][:8]
        oracle.eri_batch(basis, probe)            # thread pool / page-in warm-up, untimed
        probe = q[:: max(1, n // 64)][:64]
        t0 = time.time()
        oracle.eri_batch(basis, probe)
        per = max(time.time() - t0, 1e-5) / len(probe)
        m = int(min(n, max(16, 0.3 / per)))
        idx = np.arange(0, n, max(1, n // m))[:m]
        t0 = time.time()
        ref = oracle.eri_batch(basis, q[idx])
        dt = max(time.time() - t0, 1e-6)
        got = out.cpu().numpy()[idx]
        d = np.abs(got - ref).reshape(len(idx), -1)
        r = np.abs(ref).reshape(len(idx), -1)
        err, scale = d.max(axis=1), r.max(axis=1)
        outside = int((~(d <= 1e-12 + 1e-10 * r).all(axis=1)).sum())        # north_star's criterion, componentwise
        bq = 16 + 8 * int(np.prod([2 * l + 1 for l in cls]))
        gbs = bq * n / t * 1e-9
        fa, fh = flops / t * 1e-12 / peak, gbs / hbm_peak()[0]
        lines.append("| (%d%d\\|%d%d) | %d | %d | %.1f | %.3e | %.1f | %.3f | %d | %.1f | %.3f | %s | %.3e | %d quartets, %.2f s | %.0fx | %.1e | %d |"
                     % (*cls, info["tier"], n, k4q.mean(), n / t, flops / t * 1e-9, fa, bq, gbs, fh, "hbm" if fh > fa else "alu",
                        len(idx) / dt, len(idx), dt, (n / t) / (len(idx) / dt), float(err.max()), outside))
        del out, ws
    txt = "\n".join(lines) + "\n"
    print(txt)
    if path and path != "-":
        with open(path, "w") as f:
            f.write(txt)
    return 0


def grad_flops(cls):
    """Algorithmic FP64 flops of the first-derivative path for one class (FMA = 2, MUL / ADD = 1), counted on the graph the kernel
    evaluates (csrc/eri_grad.cu): per PRIMITIVE quartet the pair set-up (70) and Boys values (2 x 9 per order), every vertex of the
    bra and ket levels of Eq. (2) (3 for the two leading terms, 4 for the lower term, 2 for the cross term where they exist) and one
    FMA per accumulated target and set; per CONTRACTED quartet the closed-form horizontal recurrences (2 per term), the combination
    (2 per Cartesian component and axis) and the non-zero coefficients of the four c2s steps (2 each)."""
    from paper_2605_10312_b200.gen import solid
    la, lb, lc, ld = cls
    E, F = la + lb + 1, lc + ld + 1
    M = E + F
    comps = [c for lev in range(10) for c in solid.cart_comps(lev)]
    ncum = lambda l: (l + 1) * (l + 2) * (l + 3) // 6 if l >= 0 else 0     # noqa: E731
    first = lambda c: 0 if c[0] else (1 if c[1] else 2)                   # noqa: E731
    prim = 70 + 18 * (M + 1)
    for n in range(E):
        for c in comps[ncum(n):ncum(n + 1)]:
            prim += (M - n) * (3 + (4 if c[first(c)] > 1 else 0))
    rect = [(max(la - 1, 0), la + lb, max(lc - 1, 0), lc + ld), (la + 1, la + lb + 1, lc, lc + ld),
            (la, la + lb + 1, lc, lc + ld), (la, la + lb, lc + 1, lc + ld + 1)]
    for f in range(F):
        nel = ncum(E - 1) if f + 1 == F else ncum(E)
        for c in comps[ncum(f):ncum(f + 1)]:
            i = first(c)
            cross = sum(1 for e in comps[:nel] if e[i] > 0)
            prim += (F - f) * (nel * (3 + (4 if c[i] > 1 else 0)) + 2 * cross)
    for (e0, e1, f0, f1) in rect:
        prim += 2 * (ncum(e1) - ncum(e0 - 1)) * (ncum(f1) - ncum(f0 - 1))
    nc = lambda l: (l + 1) * (l + 2) // 2                                  # noqa: E731
    terms = lambda l: sum((c[0] + 1) * (c[1] + 1) * (c[2] + 1) for c in solid.cart_comps(l))   # noqa: E731
    quartet = 0
    for p in range(3):
        for sh in (1, -1):
            m = [la, lb, lc, ld]
            m[p] += sh
            if m[p] < 0:
                continue
            nfr = ncum(m[2] + m[3]) - ncum(m[2] - 1)
            quartet += 2 * (nc(m[0]) * terms(m[1]) * nfr + nc(m[0]) * nc(m[1]) * nc(m[2]) * terms(m[3]))
    blk = nc(la) * nc(lb) * nc(lc) * nc(ld)
    quartet += 9 * 2 * blk
    dims = [nc(la), nc(lb), nc(lc), nc(ld)]
    for k, l in enumerate(cls):
        nnz = sum(len(r) for r in solid.c2s_rows(l))
        quartet += 9 * 2 * nnz * int(np.prod(dims[:k] + dims[k + 1:]))
        dims[k] = 2 * l + 1
    return prim, quartet


def run_grad_table(path):
    """rcg_eri_grad_batch per class -- quartets/s, algorithmic GFLOP/s and fraction of the FP64 peak, output
    GB/s, the integral call on the same list beside it, and the derivative oracle's rate and largest difference on a bounded sample."""
    import torch
    import oracle
    from paper_2605_10312_b200 import rcg, workloads
    oracle.build_grad()
    b3 = workloads.cfg3_basis()
    B3 = rcg.Basis(b3)
    peak = rcg.fp64_peak_tflops()
    cases = [("cfg1 shape", workloads.cfg1(10000), (1, 1, 1, 1)), ("cfg2 shape", workloads.cfg2(20000), (2, 2, 2, 2))]
    for cls in workloads.canonical_classes(2):
        n = 50000 if sum(cls) <= 6 else 20000
        q = workloads.sample_class_quartets(b3, cls, n, seed=7000 + sum(x * 5 ** i for i, x in enumerate(cls)))
        k4q = np.prod(np.diff(b3["prim_off"])[q], axis=1)
        cases.append(("water", (b3, np.ascontiguousarray(q[np.argsort(-k4q, kind="stable")])), cls))
    lines = ["# First-derivative ERIs per class (SURVEY 8(f) NEXT-4): `rcg_eri_grad_batch`, one class-independent kernel", "",
             "Command (under gpurun, one B200): `python bench.py --grad-table <this file>`", "",
             "cfg1 / cfg2 shapes: the BASELINE configs' bases and the first 10,000 / 20,000 quartets of their lists; water: K4-sorted seeded lists from the cfg3 water basis "
             "(s shells of 10 primitives: mean K4 in the thousands for the s-rich classes).  5 timed calls between CUDA events after 2 warm-up calls.  Flops: the static count of "
             "`bench.grad_flops` for the graph the kernel evaluates (FMA = 2); measured FP64 peak %.1f TFLOP/s; output = 12 blocks per quartet, HBM peak %.0f GB/s (%s).  "
             "Oracle: `oracle.eri_grad_batch` on %d host threads over an evenly spaced sample of the list (about 0.5 s)." % ((peak,) + hbm_peak() + (oracle.num_threads(),)), "",
             "| list | class | quartets | mean K4 | ms | quartets/s | GFLOP/s | frac of FP64 peak | output GB/s | frac of HBM peak | integrals ms (same list) | grad / integrals | oracle quartets/s | oracle sample | GPU / oracle | max diff / quartet scale |",
             "|---|---|---|---|---|---|---|---|---|---|---|---|---|---|---|---|"]
    for name, (basis, q), cls in cases:
        B = B3 if basis is b3 else rcg.Basis(basis)
        n = len(q)
        k4q = np.prod(np.diff(basis["prim_off"])[q], axis=1)
        fp, fq = grad_flops(cls)
        flops = fp * int(k4q.sum()) + fq * n
        qd = torch.tensor(q, device="cuda")
        out = rcg.eri_grad_batch(B, cls, qd)
        ref_out = rcg.eri_batch(B, cls, qd)
        ts = []
        for fn in (lambda: rcg.eri_grad_batch(B, cls, qd, out=out), lambda: rcg.eri_batch(B, cls, qd, out=ref_out)):
            fn()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(5):
                fn()
            e1.record()
            torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1) / 5 * 1e-3)
        t, ti = ts
        probe = q[:: max(1, n // 16)][:16]
        t0 = time.time()
        oracle.eri_grad_batch(basis, probe)
        per = max(time.time() - t0, 1e-5) / len(probe)
        m = int(min(n, max(16, 0.5 / per)))
        idx = np.arange(0, n, max(1, n // m))[:m]
        t0 = time.time()
        ref = oracle.eri_grad_batch(basis, q[idx])
        dt = max(time.time() - t0, 1e-6)
        got = out.cpu().numpy()[idx]
        sc = np.maximum(np.abs(ref).reshape(len(idx), -1).max(axis=1), 1e-300)
        rel = float((np.abs(got - ref).reshape(len(idx), -1).max(axis=1) / sc).max())
        gbs = (16 + 96 * int(np.prod([2 * l + 1 for l in cls]))) * n / t * 1e-9
        lines.append("| %s | (%d%d\\|%d%d) | %d | %.1f | %.3f | %.3e | %.1f | %.3f | %.1f | %.3f | %.3f | %.0fx | %.3e | %d quartets, %.2f s | %.0fx | %.1e |"
                     % (name, *cls, n, k4q.mean(), t * 1e3, n / t, flops / t * 1e-9, flops / t * 1e-12 / peak, gbs, gbs / hbm_peak()[0], ti * 1e3, t / ti,
                        len(idx) / dt, len(idx), dt, (n / t) / (len(idx) / dt), rel))
        del out, ref_out
    txt = "\n".join(lines) + "\n"
    print(txt)
    if path and path != "-":
        with open(path, "w") as f:
            f.write(txt)
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--class-table", default="", help="write the per-class table with the oracle beside it (markdown) and exit")
    ap.add_argument("--grad-table", default="", help="write the per-class table of the first-derivative entry point (markdown) and exit")
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours")
    ap.add_argument("--workload", default="cfg2")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.class_table:
        return run_class_table(args.class_table)
    if args.grad_table:
        return run_grad_table(args.grad_table)

    import torch
    import torch.distributed as dist
    from paper_2605_10312_b200 import rcg, sharding

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the library has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    W = max(3, args.warmup)
    basis, q, cls, wname = load_workload(args.workload)
    nq = len(q)
    B = rcg.Basis(basis)
    info = rcg.class_info(cls)
    flops_step = info["flops_per_prim_quartet"] * prim_quartets(basis, q) + info["flops_per_quartet"] * nq
    qd = torch.tensor(q, device="cuda")
    nout = int(np.prod([2 * l + 1 for l in cls]))
    out = torch.empty((nq,) + tuple(2 * l + 1 for l in cls), dtype=torch.float64, device="cuda")
    wsb = rcg.eri_workspace_bytes(B, cls, nq)
    ws = torch.empty(max(1, (wsb + 7) // 8), dtype=torch.float64, device="cuda")
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")      # > 126 MB L2
    stream = torch.cuda.current_stream()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident throughput: per-step CUDA events on the launching stream, L2 flushed between steps
    for _ in range(W):
        rcg.eri_batch(B, cls, qd, out=out, workspace=ws)
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    evs = []
    t_wall0 = time.time()
    for _ in range(args.steps):
        flush.zero_()
        e0 = torch.cuda.Event(enable_timing=True)
        e1 = torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        rcg.eri_batch(B, cls, qd, out=out, workspace=ws)
        e1.record(stream)
        evs.append((e0, e1))
    barrier()
    t_wall = time.time() - t_wall0
    ms_steps = [a.elapsed_time(b) for a, b in evs]
    ms_total = float(sum(ms_steps))
    ms_total_max = sharding.max_over_ranks(ms_total, device="cuda")
    ms_per_step = ms_total_max / args.steps
    value = world * nq / (ms_per_step * 1e-3)

    # ---- end to end through the host entry point (pinned host buffers; H2D + D2H inside the timed region)
    qh = torch.from_numpy(q).pin_memory()
    oh = torch.empty(out.shape, dtype=torch.float64).pin_memory()
    e2e_steps = max(1, min(args.steps, 5))
    rcg.eri_batch_host(B, cls, qh, out_host=oh)
    barrier()
    t0 = time.time()
    for _ in range(e2e_steps):
        rcg.eri_batch_host(B, cls, qh, out_host=oh)
    torch.cuda.synchronize()
    e2e_value = world * nq / sharding.max_over_ranks((time.time() - t0) / e2e_steps, device="cuda")
    # ---- end to end for a Fock build of the same batch (rcg_fock_batch: the integrals are digested on the chip):
    # per step H2D of the density from pinned host memory, the fused kernel, rcg_jk_finish, D2H of J and K
    nbf = int((2 * np.asarray(basis["shell_l"]) + 1).sum())
    bf_off = torch.tensor(np.concatenate([[0], np.cumsum(2 * np.asarray(basis["shell_l"]) + 1)])[:-1].astype(np.int32), device="cuda")
    Dh = torch.from_numpy(np.random.default_rng(0).normal(size=(nbf, nbf))).pin_memory()
    Dh.add_(Dh.t().clone())
    Dd = torch.empty((nbf, nbf), dtype=torch.float64, device="cuda")
    Jd, Kd = torch.empty_like(Dd), torch.empty_like(Dd)
    Jh, Kh = torch.empty((nbf, nbf), dtype=torch.float64).pin_memory(), torch.empty((nbf, nbf), dtype=torch.float64).pin_memory()
    fws = torch.empty(max(1, (rcg.fock_workspace_bytes(B, cls, nq, uniform=True) + 7) // 8), dtype=torch.float64, device="cuda")

    def fock_step():
        Dd.copy_(Dh, non_blocking=True)
        Jd.zero_()
        Kd.zero_()
        rcg.fock_batch(B, cls, qd, bf_off, Dd, Jd, Kd, workspace=fws, uniform=True)
        rcg.jk_finish(Jd, Kd)
        Jh.copy_(Jd, non_blocking=True)
        Kh.copy_(Kd, non_blocking=True)
        torch.cuda.synchronize()

    fock_step()
    barrier()
    t0 = time.time()
    for _ in range(e2e_steps):
        fock_step()
    fock_value = world * nq / sharding.max_over_ranks((time.time() - t0) / e2e_steps, device="cuda")
    sampler.stop.set()          # clocks were sampled over all timed regions (device-resident, e2e, Fock e2e)
    sampler.join()
    checksum = float(oh.reshape(nq, -1)[:: max(1, nq // 1000)].abs().sum())

    if rank == 0:
        peak_meas = rcg.fp64_peak_tflops()
        ach = flops_step / (ms_total / args.steps * 1e-3) * 1e-12
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": W,
                "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f64", "data": "synthetic",
                "config": {"workload": wname, "class": list(cls), "tier": info["tier"], "quartets_per_gpu": nq,
                           "l2": "256 MiB buffer rewritten between timed steps (L2 flush); output 500 MB/step > L2",
                           "timing": "per-step CUDA events on the launch stream, max over ranks"},
                "gflops": flops_step * world / (ms_per_step * 1e-3) * 1e-9,
                "roofline": {"bound": "alu", "achieved": ach, "peak": peak_meas, "unit": "TFLOP/s",
                             "frac": ach / peak_meas, "traffic": TRAFFIC.get(args.workload),
                             "peak_source": "FP64 DFMA microbenchmark run in this process (rcg_fp64_peak_tflops); "
                                            "nominal 148 SM x 64 FMA/clk x 2 x 1.965 GHz = 37.2",
                             "frac_of_nominal": ach / 37.2, "kernel": "rcg_eri_batch class kernel",
                             "algorithmic_flops_per_launch": flops_step,
                             "traffic_unit": "bytes per launch (ncu dram read+write)", "traffic_source": TRAFFIC_SOURCE,
                             "algorithmic_bytes_per_launch": (16 + 8 * nout) * nq,
                             "hbm_gbs": (16 + 8 * nout) * nq / (ms_total / args.steps * 1e-3) * 1e-9},
                "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(q.nbytes),
                        "d2h_bytes_per_step": int(nq * nout * 8), "checksum": checksum},
                "e2e_fock": {"value": fock_value, "unit": UNIT, "what": "Fock build of the same batch through rcg_fock_batch + rcg_jk_finish: "
                             "H2D of the density (pinned), integrals digested on the chip, D2H of J and K", "h2d_bytes_per_step": int(8 * nbf * nbf),
                             "d2h_bytes_per_step": int(16 * nbf * nbf), "checksum": float(Jh.abs().sum() + Kh.abs().sum())},
                "gpu_launches": args.steps, "clocks": sampler.summary(), "wall_s_timed_region": t_wall}
        if not args.no_cpu_baseline:
            v, n2, dt, cores = time_oracle(basis, q)
            line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
                                    "sample": "first %d quartets of the batch, %.1f s" % (n2, dt)}
        print(json.dumps(line))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
