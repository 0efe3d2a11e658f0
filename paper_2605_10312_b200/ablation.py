"""Ablation of the paper's Tier-1 ideas on the B200 (PAPER.md:311-345 is the A100 study):
for the 16 register-tier classes, the unrolled VRR graph emitted in the post-order, in the DSA order of Eq. (7)
(PAPER.md:168-177), and built by the literal Alg. 1 axis rule instead of the ket-first one (reading R-AXIS);
plus the warp tier forced on the same lists.  Reports PeakLive (Eq. (4)), ptxas registers / spill bytes and time.

    python -m paper_2605_10312_b200.ablation build            # CPU: variant libraries under csrc/build/ablation/
    python -m paper_2605_10312_b200.ablation run --md out.md  # GPU: times every variant

Lists: 200,000 seeded quartets per class over 30 shells per l = 0..3 with 2 primitives each (K4 = 16 everywhere, so the
register tier engages), exponents log-uniform in [0.2, 5], centres uniform in a 6-Bohr cube, seed 9.
"""
import glob
import json
import os
import re
import subprocess
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
OUT = os.path.join(HERE, "csrc", "build", "ablation")
VARIANTS = {"default": {}, "postorder": {"RCG_REG_ORDER": "post"}, "dsa": {"RCG_REG_ORDER": "dsa"},
            "alg1_axis": {"RCG_REG_AXIS": "alg1"}}


def reg_classes():
    from .gen import tiers
    from .gen.graph import canonical_classes
    return [c for c in canonical_classes() if tiers.choose_tier(c) == tiers.TIER_REGISTER]


def build():
    from . import build as b
    b.build_library()
    os.makedirs(OUT, exist_ok=True)
    classes = reg_classes()
    tags = ["%d%d%d%d" % c for c in classes]
    gen = os.path.join(HERE, "csrc", "gen")
    others = [o for o in glob.glob(os.path.join(b.OBJ, "*.o")) if not any(o.endswith("gen_eri_%s.o" % t) for t in tags)]
    info = {}
    try:
        for name, env in VARIANTS.items():
            e = dict(os.environ)
            e.update(env)
            subprocess.check_call([sys.executable, "-m", "paper_2605_10312_b200.gen.generate", "--only", ",".join(tags)],
                                  cwd=os.path.dirname(HERE), env=e, stdout=subprocess.DEVNULL)
            meta = {tuple(m["cls"]): m for m in json.load(open(os.path.join(gen, "classes.json")))}
            objs = []
            for cls, t in zip(classes, tags):
                obj = os.path.join(OUT, "%s_%s.o" % (name, t))
                p = subprocess.run([b.NVCC] + b.FLAGS + ["-c", os.path.join(gen, "eri_%s.cu" % t), "-o", obj], capture_output=True, text=True)
                if p.returncode:
                    raise RuntimeError(p.stderr[-2000:])
                m = re.search(r"rcg_eri_reg_%s.*?\n.*?(\d+) bytes stack frame, (\d+) bytes spill stores, (\d+) bytes spill loads\n.*?Used (\d+) registers" % t, p.stderr, re.S)
                info["%s/%s" % (name, t)] = dict(regs=int(m.group(4)), spill=int(m.group(2)) + int(m.group(3)), vertices=meta[cls]["reg_vertices"],
                                                 order=meta[cls]["reg_order"] if "RCG_REG_ORDER" not in env else env["RCG_REG_ORDER"],
                                                 pl_post=meta[cls]["reg_peaklive_postorder"], pl_dsa=meta[cls]["reg_peaklive_dsa"])
                objs.append(obj)
            subprocess.check_call([b.NVCC, "-shared", "-o", os.path.join(OUT, "librcg_%s.so" % name)] + others + objs + ["-lcudart"])
            for o in objs:
                os.remove(o)
    finally:      # the committed sources are the default variant
        subprocess.check_call([sys.executable, "-m", "paper_2605_10312_b200.gen.generate", "--only", ",".join(tags)],
                              cwd=os.path.dirname(HERE), stdout=subprocess.DEVNULL)
    json.dump(info, open(os.path.join(OUT, "ptxas.json"), "w"), indent=1)
    print("built %d variant libraries in %s" % (len(VARIANTS), OUT))


def uniform_basis():
    from . import workloads
    rng = np.random.default_rng(9)
    ls = [l for l in range(4) for _ in range(30)]
    exps = [np.exp(rng.uniform(np.log(0.2), np.log(5.0), 2)) for _ in ls]
    coefs = [workloads.normalise_shell(l, e, rng.uniform(0.1, 1.0, 2)) for l, e in zip(ls, exps)]
    return workloads.make_basis(ls, exps, coefs, rng.uniform(0.0, 6.0, (len(ls), 3))), rng


def time_variant(n=200000):
    """runs in a subprocess with RCG_LIB set; prints {tag: [ms own tier, ms warp tier forced]}"""
    import torch
    from . import rcg
    basis, rng = uniform_basis()
    B = rcg.Basis(basis)
    res = {}
    for cls in reg_classes():
        q = np.stack([30 * l + rng.integers(0, 30, n) for l in cls], axis=1).astype(np.int32)
        qd = torch.tensor(q, device="cuda")
        ms = []
        for tier in (0, rcg.TIER_WARP):
            out = rcg.eri_batch(B, cls, qd, tier=tier)
            rcg.eri_batch(B, cls, qd, out=out, tier=tier)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(5):
                rcg.eri_batch(B, cls, qd, out=out, tier=tier)
            e1.record()
            torch.cuda.synchronize()
            ms.append(e0.elapsed_time(e1) / 5)
        res["%d%d%d%d" % cls] = ms
    print("ABLATION " + json.dumps(res))


def run(md):
    info = json.load(open(os.path.join(OUT, "ptxas.json")))
    times = {}
    for name in VARIANTS:
        e = dict(os.environ)
        e["RCG_LIB"] = os.path.join(OUT, "librcg_%s.so" % name)
        p = subprocess.run([sys.executable, "-m", "paper_2605_10312_b200.ablation", "_time"], cwd=os.path.dirname(HERE), env=e,
                           capture_output=True, text=True)
        line = [ln for ln in p.stdout.splitlines() if ln.startswith("ABLATION ")]
        if not line:
            raise RuntimeError(p.stderr[-2000:])
        times[name] = json.loads(line[0][9:])
    lines = ["# Register tier (the paper's Tier 1) ablation on one B200: emission order and axis rule", "",
             "Commands: `python -m paper_2605_10312_b200.ablation build` (here, CPU) then, under gpurun, "
             "`python -m paper_2605_10312_b200.ablation run --md gpurun_out/r1_ablation_register_tier.md`.", "",
             "200,000 quartets per class, K4 = 16 (2 primitives per shell), 5 timed calls after 2 warm-up calls; ms per call.  "
             "PeakLive = Eq. (4) of the paper on the ket-first graph (post-order / DSA greedy of Eq. (7)); regs / spill = ptxas.  "
             "`default` = the committed kernels (the order with the lower PeakLive); `alg1_axis` = graph by the literal Alg. 1 "
             "(last hit wins) instead of ket-first; last column: the same list forced onto the warp tier.", "",
             "| class | vertices | PeakLive post / DSA | default: order, regs, spill, ms | post-order: regs, spill, ms | DSA: regs, spill, ms | alg1 axis: vertices, regs, spill, ms | warp tier ms |",
             "|---|---|---|---|---|---|---|---|"]
    for t in times["default"]:
        d, po, ds, ax = (info["%s/%s" % (v, t)] for v in ("default", "postorder", "dsa", "alg1_axis"))
        lines.append("| (%s%s\\|%s%s) | %d | %d / %d | %s, %d, %d, %.3f | %d, %d, %.3f | %d, %d, %.3f | %d, %d, %d, %.3f | %.3f |"
                     % (t[0], t[1], t[2], t[3], d["vertices"], d["pl_post"], d["pl_dsa"], d["order"], d["regs"], d["spill"], times["default"][t][0],
                        po["regs"], po["spill"], times["postorder"][t][0], ds["regs"], ds["spill"], times["dsa"][t][0],
                        ax["vertices"], ax["regs"], ax["spill"], times["alg1_axis"][t][0], times["default"][t][1]))
    txt = "\n".join(lines) + "\n"
    print(txt)
    if md:
        open(md, "w").write(txt)


if __name__ == "__main__":
    if len(sys.argv) > 1 and sys.argv[1] == "build":
        build()
    elif len(sys.argv) > 1 and sys.argv[1] == "_time":
        time_variant()
    elif len(sys.argv) > 1 and sys.argv[1] == "run":
        run(sys.argv[3] if len(sys.argv) > 3 and sys.argv[2] == "--md" else "")
    else:
        print(__doc__)
