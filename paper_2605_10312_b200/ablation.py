"""The paper's ablations on the B200 (PAPER.md:311-345 is the A100 study): axis-priority rule,
emission order (DSA, Eq. (7)), stepwise spherical fusion on/off, and the tier sweep (thread-per-quartet Tier 1 forced,
table-driven buffered tier forced, level-synchronous block tier instead of the chain one) on quartets of sum l = 2..12.

    python -m paper_2605_10312_b200.ablation build [--workdir DIR]     # CPU: variant libraries (generator flags, own directories)
    python -m paper_2605_10312_b200.ablation run --md out.md           # GPU: time every variant, compare with the default library

Every variant is generated into its OWN directory by `gen/generate.py --out-dir` and linked by `build.py --gen-dir --lib`;
the committed csrc/gen/ is never touched.  Each variant runs in a child process (RCG_LIB names its library); the table
reports time, ptxas registers and spill bytes, PeakLive (Eq. (4)) and the largest deviation of the variant's integrals
from the default library's, scaled by the quartet's largest integral (the oracle parity of the variants is
tests/test_gpu_variants.py).

Lists: seeded quartets per class over 30 shells per l = 0..3 with 2 primitives each (K4 = 16 everywhere), exponents
log-uniform in [0.2, 5], centres uniform in a 6-Bohr cube, seed 9.
"""
import json
import os
import re
import subprocess
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
WORK = os.path.join(HERE, "csrc", "build", "ablation")

# the quartets of the study (sum l = 2, 4, 6, 7, 8, 10, 12) and how many of each are timed
CLASSES = [((1, 0, 1, 0), 200000), ((1, 1, 1, 1), 200000), ((2, 1, 2, 1), 100000), ((2, 2, 2, 1), 50000), ((2, 2, 2, 2), 50000),
           ((3, 3, 2, 2), 10000), ((3, 3, 3, 3), 4000)]
TIER = {"register": 1, "warp": 2, "global": 3, "block": 4}
# name -> (generator arguments, run-time tier to force (0 = the class's own), classes it applies to (None = all))
VARIANTS = {
    "default": ([], 0, None),
    "no_sph_fusion": (["--no-spherical-fusion"], 0, [c for c, _ in CLASSES if sum(c) <= 8]),
    "tier1_thread": (["--force-tier", "register"], 1, [c for c, _ in CLASSES if sum(c) <= 7]),
    "tier1_thread_alg1_axis": (["--force-tier", "register", "--axis-rule", "alg1"], 1, [c for c, _ in CLASSES if sum(c) <= 7]),
    "tier1_thread_dsa": (["--force-tier", "register", "--order", "dsa"], 1, [c for c, _ in CLASSES if sum(c) <= 7]),
    "tier1_thread_postorder": (["--force-tier", "register", "--order", "post"], 1, [c for c, _ in CLASSES if sum(c) <= 7]),
    "tier1_thread_no_sph_fusion": (["--force-tier", "register", "--no-spherical-fusion"], 1, [c for c, _ in CLASSES if sum(c) <= 7]),
    "buffered_global": (["--force-tier", "global"], 3, None),
    "block_level_table": (["--set", "GEN_NO_SLAB=1"], 0, [c for c, _ in CLASSES if c[0] == 3]),
}


def tag(c):
    return "%d%d%d%d" % c


def variant_dir(name, workdir=None):
    return os.path.join(workdir or WORK, name)


def build_variant(name, classes=None, workdir=None, jobs=None):
    """generate + link one variant library; -> (library path, {class: ptxas / PeakLive facts})."""
    from . import build as b
    args, _, applies = VARIANTS[name]
    classes = [c for c in (classes or [c for c, _ in CLASSES]) if applies is None or c in applies]
    d = variant_dir(name, workdir)
    os.makedirs(d, exist_ok=True)
    if name == "default":
        lib = b.build_library()
    else:
        subprocess.check_call([sys.executable, "-m", "paper_2605_10312_b200.gen.generate", "--only", ",".join(tag(c) for c in classes),
                               "--out-dir", d] + args, cwd=ROOT, stdout=subprocess.DEVNULL)
        keep = {"eri_%s.cu" % tag(c) for c in classes}
        for f in os.listdir(d):
            if f.endswith(".cu") and f not in keep:
                os.remove(os.path.join(d, f))
        lib = b.build_library(gen_dir=d, lib=os.path.join(d, "librcg.so"), jobs=jobs)
    meta = {tuple(m["cls"]): m for m in json.load(open(os.path.join(d if name != "default" else os.path.join(HERE, "csrc", "gen"), "classes.json")))}
    logdir = os.path.join(d, "build") if name != "default" else b.OBJ
    facts = {}
    for c in classes:
        txt = open(os.path.join(logdir, "gen_eri_%s.o.log" % tag(c))).read()
        ks = re.findall(r"Compiling entry function '(\S+)' for 'sm_100a'.*?\n.*?(\d+) bytes stack frame, (\d+) bytes spill stores, (\d+) bytes spill loads\n.*?Used (\d+) registers", txt, re.S)
        ks = [k for k in ks if "side_kernel" not in k[0]]
        facts[c] = dict(kernels={re.sub(r"^_ZN?\d*[a-z]\d{4}\d*", "", k[0])[:28]: (int(k[4]), int(k[2]) + int(k[3])) for k in ks},
                        peaklive=(meta[c].get("peaklive_postorder"), meta[c].get("peaklive_dsa")), tier=meta[c]["tier"])
    json.dump({tag(c): v for c, v in facts.items()}, open(os.path.join(d, "facts.json"), "w"))
    return lib, facts


def make_basis():
    from . import workloads
    rng = np.random.default_rng(9)
    ls, exps, coefs, cen = [], [], [], []
    for l in range(4):
        for _ in range(30):
            e = np.exp(rng.uniform(np.log(0.2), np.log(5.0), 2))
            ls.append(l); exps.append(e); coefs.append(workloads.normalise_shell(l, e, rng.uniform(0.2, 1.0, 2)))
            cen.append(rng.uniform(0.0, 6.0, 3))
    return workloads.make_basis(ls, exps, coefs, np.array(cen))


def worker(tier, classes, dump):
    """child process: time the listed classes in the library RCG_LIB names; save the first 2,000 blocks of each to `dump`."""
    import torch
    from . import rcg, workloads
    basis = make_basis()
    B = rcg.Basis(basis)
    out = {}
    blocks = {}
    for ci, (cls, n) in enumerate(CLASSES):
        if cls not in classes:
            continue
        q = workloads.sample_class_quartets(basis, cls, n, seed=77 + ci)
        qd = torch.tensor(q, device="cuda")
        t = tier if (tier == 0 or rcg.class_info(cls)["tier"] == tier or tier == 3) else 0
        ws = torch.empty(max(1, rcg.eri_workspace_bytes(B, cls, n, t) // 8), dtype=torch.float64, device="cuda")
        o = rcg.eri_batch(B, cls, qd, workspace=ws, tier=t)
        rcg.eri_batch(B, cls, qd, out=o, workspace=ws, tier=t)
        best = 1e30
        for _ in range(5):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            rcg.eri_batch(B, cls, qd, out=o, workspace=ws, tier=t)
            e1.record()
            torch.cuda.synchronize()
            best = min(best, e0.elapsed_time(e1))
        info = rcg.class_info(cls)
        fl = (info["flops_per_prim_quartet"] * 16 + info["flops_per_quartet"]) * n
        out[tag(cls)] = dict(ms=best, n=n, tflops=fl / best * 1e-9, tier_run=t or info["tier"])
        blocks[tag(cls)] = o[:2000].cpu().numpy()
        del o, ws
    np.savez(dump, **blocks)
    print(json.dumps(out))


def run(md, workdir=None):
    import tempfile
    res, facts = {}, {}
    tmp = tempfile.mkdtemp()
    for name, (_, tier, applies) in VARIANTS.items():
        d = variant_dir(name, workdir)
        lib = os.path.join(HERE, "librcg.so") if name == "default" else os.path.join(d, "librcg.so")
        if not os.path.exists(lib):
            build_variant(name, workdir=workdir)
        facts[name] = json.load(open(os.path.join(d, "facts.json")))
        classes = [c for c, _ in CLASSES if applies is None or c in applies]
        env = dict(os.environ, RCG_LIB=lib)
        p = subprocess.run([sys.executable, "-m", "paper_2605_10312_b200.ablation", "worker", str(tier), ",".join(tag(c) for c in classes),
                            os.path.join(tmp, name + ".npz")], cwd=ROOT, env=env, capture_output=True, text=True)
        if p.returncode:
            raise RuntimeError("variant %s failed:\n%s" % (name, p.stderr[-3000:]))
        res[name] = json.loads(p.stdout.strip().splitlines()[-1])
    base = np.load(os.path.join(tmp, "default.npz"))
    lines = ["# Ablations on one B200 (SURVEY 8(f) NEXT-3; PAPER.md:311-345)", "",
             "Command (under gpurun): `python -m paper_2605_10312_b200.ablation run --md <this file>` (variant libraries: `... ablation build`).", "",
             "K4 = 16 everywhere; best of 5 calls between CUDA events.  `dev` = largest |variant - default| over the first 2,000 quartets, scaled by the "
             "quartet's largest integral.  regs / spill = ptxas registers and spill bytes of the class's kernel(s) in that variant.", "",
             "| class | sum l | variant | tier run | ms | TFLOP/s | x default | kernels: regs / spill B | PeakLive post / DSA | dev |", "|---|---|---|---|---|---|---|---|---|---|"]
    for cls, n in CLASSES:
        t = tag(cls)
        for name in VARIANTS:
            if t not in res[name]:
                continue
            r = res[name][t]
            v = np.load(os.path.join(tmp, name + ".npz"))[t]
            b0 = base[t]
            sc = np.abs(b0).reshape(len(b0), -1).max(axis=1) + 1e-300
            dev = float((np.abs(v - b0).reshape(len(b0), -1).max(axis=1) / sc).max())
            f = facts[name].get(t, {})
            ks = "; ".join("%s %d/%d" % (k, a, s) for k, (a, s) in sorted(f.get("kernels", {}).items()))
            pl = f.get("peaklive", [None, None])
            lines.append("| (%d%d\\|%d%d) | %d | %s | %d | %.3f | %.2f | %.2f | %s | %s / %s | %.1e |"
                         % (cls + (sum(cls), name, r["tier_run"], r["ms"], r["tflops"], res["default"][t]["ms"] / r["ms"], ks, pl[0], pl[1], dev)))
    txt = "\n".join(lines) + "\n"
    print(txt)
    if md:
        with open(md, "w") as f:
            f.write(txt)


def main(argv=None):
    argv = list(sys.argv[1:] if argv is None else argv)
    cmd = argv[0] if argv else ""
    workdir = argv[argv.index("--workdir") + 1] if "--workdir" in argv else None
    if cmd == "build":
        for name in VARIANTS:
            lib, facts = build_variant(name, workdir=workdir)
            print(name, lib)
            for c, f in facts.items():
                print("   ", tag(c), f["kernels"])
    elif cmd == "run":
        run(argv[argv.index("--md") + 1] if "--md" in argv else "", workdir)
    elif cmd == "worker":
        worker(int(argv[1]), [tuple(int(ch) for ch in t) for t in argv[2].split(",")], argv[3])
    else:
        print(__doc__)
        return 1
    return 0


if __name__ == "__main__":
    sys.exit(main())
