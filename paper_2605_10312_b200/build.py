"""Build the C-ABI library librcg.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2605_10312_b200.build [--force] [--gen-dir DIR --lib PATH]

--gen-dir / --lib: link a VARIANT library (generator options, gen/generate.py --out-dir) from the class sources in DIR; classes
missing there come from csrc/gen.  rcg.py loads it when RCG_LIB names it (ablation and sweep runs only).

Sources: csrc/*.cu plus the generated per-class csrc/gen/*.cu (committed; regenerate them with
`python -m paper_2605_10312_b200.gen.generate`).  Objects are cached in csrc/build/ by mtime.
"""
import glob
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(CSRC, "build")
LIB = os.path.join(HERE, "librcg.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
         "-Xcompiler", "-fPIC", "-Xptxas", "-v", "-I", CSRC]


def _newest_header():
    hs = glob.glob(os.path.join(CSRC, "*.h")) + glob.glob(os.path.join(CSRC, "*.cuh")) + \
        glob.glob(os.path.join(os.path.dirname(HERE), "include", "*.h"))
    return max(os.path.getmtime(h) for h in hs)


def _compile(src, force, hdr_time, objdir=None):
    objdir = objdir or OBJ
    rel = os.path.relpath(src, CSRC).replace(os.sep, "_") if objdir == OBJ else "gen_" + os.path.basename(src)
    obj = os.path.join(objdir, rel[:-3] + ".o")
    log = obj + ".log"
    if not force and os.path.exists(obj) and os.path.getmtime(obj) >= max(os.path.getmtime(src), hdr_time):
        return obj
    p = subprocess.run([NVCC] + FLAGS + ["-c", src, "-o", obj], capture_output=True, text=True)
    with open(log, "w") as f:
        f.write(p.stdout + p.stderr)
    if p.returncode != 0:
        raise RuntimeError("nvcc failed on %s:\n%s" % (src, p.stderr[-4000:]))
    return obj


def build_library(force=False, jobs=None, gen_dir=None, lib=None):
    os.makedirs(OBJ, exist_ok=True)
    srcs = sorted(glob.glob(os.path.join(CSRC, "*.cu")) + glob.glob(os.path.join(CSRC, "gen", "*.cu")))
    if not srcs:
        raise RuntimeError("no CUDA sources under %s" % CSRC)
    hdr_time = _newest_header()
    with ThreadPoolExecutor(jobs or os.cpu_count() or 1) as ex:
        objs = list(ex.map(lambda s: _compile(s, force, hdr_time), srcs))
        if gen_dir:          # variant library: its own objects for the sources present in gen_dir, the default ones for the rest
            vdir = os.path.join(os.path.abspath(gen_dir), "build")
            os.makedirs(vdir, exist_ok=True)
            vsrcs = sorted(glob.glob(os.path.join(os.path.abspath(gen_dir), "*.cu")))
            vobjs = dict(zip([os.path.basename(v) for v in vsrcs], ex.map(lambda s: _compile(s, force, hdr_time, vdir), vsrcs)))
            objs = [vobjs.get(os.path.basename(s), o) if os.path.dirname(s).endswith(os.path.join("csrc", "gen")) else o
                    for s, o in zip(srcs, objs)]
    lib = lib or LIB
    if gen_dir and os.path.abspath(lib) == LIB:
        raise RuntimeError("a variant build needs its own --lib path")
    if force or not os.path.exists(lib) or any(os.path.getmtime(o) > os.path.getmtime(lib) for o in objs):
        subprocess.check_call([NVCC, "-shared", "-o", lib] + objs + ["-lcudart"])
    return lib


def ptxas_report():
    """registers / spill bytes per kernel, parsed from the cached nvcc -Xptxas -v logs."""
    import re
    out = []
    for log in sorted(glob.glob(os.path.join(OBJ, "*.log"))):
        txt = open(log).read()
        for m in re.finditer(r"Compiling entry function '(\S+)' for 'sm_100a'.*?\n.*?(\d+) bytes stack frame, (\d+) bytes spill stores, (\d+) bytes spill loads\n.*?Used (\d+) registers", txt, re.S):
            out.append(dict(kernel=m.group(1), stack=int(m.group(2)), spill_st=int(m.group(3)),
                            spill_ld=int(m.group(4)), regs=int(m.group(5)), file=os.path.basename(log)))
    return out


if __name__ == "__main__":
    import argparse
    ap = argparse.ArgumentParser()
    ap.add_argument("--force", action="store_true")
    ap.add_argument("--gen-dir", default="")
    ap.add_argument("--lib", default="")
    ap.add_argument("--report", default="", help="write the ptxas table (registers, spill bytes per kernel) as markdown")
    a = ap.parse_args()
    print(build_library(force=a.force, gen_dir=a.gen_dir or None, lib=a.lib or None))
    if a.report:
        import re
        rows = ptxas_report()
        with open(a.report, "w") as f:
            f.write("# ptxas -v: registers and spill bytes of every kernel of librcg.so (sm_100a, nvcc %s)\n\n" % subprocess.run(
                [NVCC, "--version"], capture_output=True, text=True).stdout.strip().splitlines()[-2].split("release")[-1].strip())
            f.write("Command: `python -m paper_2605_10312_b200.build --report <this file>` (parses the cached `nvcc -Xptxas -v` logs of the build).\n\n")
            sp = [r for r in rows if r["spill_st"] or r["spill_ld"]]
            f.write("%d kernels; %d with spill bytes: %s.\n\n" % (len(rows), len(sp), ", ".join("`%s` (%d + %d B)" % (
                re.sub(r"^_Z+N?\d*[a-z]*\d*", "", r["kernel"])[:40], r["spill_st"], r["spill_ld"]) for r in sp) or "none"))
            f.write("| source | kernel | registers | stack | spill stores | spill loads |\n|---|---|---|---|---|---|\n")
            for r in rows:
                f.write("| %s | `%s` | %d | %d | %d | %d |\n" % (r["file"].replace(".o.log", ""), r["kernel"][:70], r["regs"], r["stack"], r["spill_st"], r["spill_ld"]))
