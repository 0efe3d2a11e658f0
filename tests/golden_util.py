"""Readers for the text fixtures under tests/golden/ (no arithmetic)."""
import os

import numpy as np

HERE = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def read_boys():
    rows = []
    for line in open(os.path.join(HERE, "boys_reference.txt")):
        if line.startswith("#") or not line.strip():
            continue
        T, m, v = line.split()
        rows.append((float(T), int(m), float(v)))
    return rows


def read_eri_golden():
    ls, cen, exps, coefs, sums, comps = [], [], [], [], [], []
    for line in open(os.path.join(HERE, "eri_golden.txt")):
        if line.startswith("#") or not line.strip():
            continue
        kind, rest = line.split(None, 1)
        parts = [p.split() for p in rest.split("|")]
        if kind == "shell":
            ls.append(int(parts[0][1])); cen.append([float(x) for x in parts[0][2:5]])
            exps.append([float(x) for x in parts[1]]); coefs.append([float(x) for x in parts[2]])
        elif kind == "sums":
            sums.append((tuple(int(x) for x in parts[0]), int(parts[1][0]), float(parts[1][1]), float(parts[1][2])))
        elif kind == "comp":
            comps.append((tuple(int(x) for x in parts[0]), tuple(int(x) for x in parts[1]), float(parts[2][0])))
    prim_off = np.zeros(len(ls) + 1, np.int32)
    prim_off[1:] = np.cumsum([len(e) for e in exps])
    basis = dict(shell_l=np.array(ls, np.int32), prim_off=prim_off, exps=np.concatenate(exps),
                 coefs=np.concatenate(coefs), centers=np.array(cen, float))
    return basis, sums, comps
