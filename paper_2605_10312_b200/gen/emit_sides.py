"""Emit csrc/gen/sides.cu: one "side" kernel per pair (l1, l2), l1 >= l2, l1 <= 4 -- one side of Phase 2 for the heavy
block tier (gen/emit_heavy.py), applied to 32 rows per block.

A side turns the contracted Cartesian targets (e0|, |e| = l1..l1+l2, of a row into the spherical pair (m1 m2|:
Eq. (3) (a, b+1i| = (a+1i, b| + X_i (a, b| unrolled to its closed form

    (a b| = sum_{k <= b} prod_i C(b_i, k_i) X_i^(b_i - k_i) (a + k, 0|          (X = A - B, or C - D: reading R-HRRK)

so that no intermediate (a, b'| with |b'| < l2 is ever held: the depth-first walk of the block tier needs 215 live
doubles per thread at (gg|, this form needs the 15 values of one b.  About 1.5x the additions of the recursion (1,890
against 1,269 at l1 = l2 = 4), on 1/6 of the registers.  Then T^(l1) on the first index (Eq. (11) / (15)) per b, the
half-transformed row parked in shared memory, and T^(l2) on the second (Eq. (12) / (16)).
Thread = (row = lane, warp = a share of the b's, then of the m1's); the rows of a block may belong to different
quartets (every lane builds the powers of its own displacement), so light classes fill their warps too.
"""
from math import comb

from .solid import cart_comps, ncart, c2s_rows
from .emit_warp import Prog

ROWS = 32
RST = 33            # odd row stride of the shared-memory tiles: conflict-free for lane = row and for the transposing load


def side_plan(l1, l2):
    B = cart_comps(l2)
    cost = [(b[0] + 1) * (b[1] + 1) * (b[2] + 1) for b in B]
    nw = max(1, min(4, len(B)))
    groups = [[] for _ in range(nw)]
    load = [0] * nw
    for jb in sorted(range(len(B)), key=lambda j: -cost[j]):
        g = min(range(nw), key=lambda i: load[i])
        groups[g].append(jb)
        load[g] += cost[jb]
    return nw, [sorted(g) for g in groups]


def emit_side(P, l1, l2):
    tag = "%d%d" % (l1, l2)
    idx = {}
    for e in range(l1, l1 + l2 + 1):
        for a in cart_comps(e):
            idx[a] = len(idx)
    NE = len(idx)
    A, B = cart_comps(l1), cart_comps(l2)
    T1, T2 = c2s_rows(l1), c2s_rows(l2)
    ns1, ns2, nb2 = 2 * l1 + 1, 2 * l2 + 1, len(B)
    nw, groups = side_plan(l1, l2)
    P.w("// ---- side (%d %d|: %d Cartesian targets -> %d x %d spherical, %d warps" % (l1, l2, NE, ns1, ns2, nw))
    P.w("__global__ void __launch_bounds__(%d) rcg_side_kernel_%s(RcgSideArgs s)" % (32 * nw, tag))
    P.w("{")
    P.ind = 1
    P.w("extern __shared__ double sm[];")
    P.w("double *Xs = sm, *SC = sm + %d;        // [%d][%d] inputs, [%d][%d] half-transformed" % (NE * RST, NE, RST, ns1 * nb2, RST))
    P.w("const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;")
    P.w("const int64_t R0 = (int64_t)blockIdx.x * %d;" % ROWS)
    P.w("for (int t = tid; t < %d; t += %d) {" % (ROWS * NE, 32 * nw))
    P.w("    const int r = t / %d, e = t - r * %d;" % (NE, NE))
    P.w("    Xs[e * %d + r] = R0 + r < s.nrows ? s.X[(R0 + r) * %d + e] : 0.0;" % (RST, NE))
    P.w("}")
    P.w("const bool valid = R0 + lane < s.nrows;")
    P.w("const int64_t R = valid ? R0 + lane : s.nrows - 1;")
    P.w("const int64_t ql = R / s.nR;")
    P.w("const int r = (int)(R - ql * s.nR);")
    P.w("const int32_t *qq = s.quartets + 4 * (s.q0 + ql);")
    P.w("const int s0 = qq[s.p0], s1 = qq[s.p1];")
    for i in range(3):
        P.w("const double X%d_1 = s.centers[3 * s0 + %d] - s.centers[3 * s1 + %d];" % (i, i, i))
        for p in range(2, l2 + 1):
            P.w("const double X%d_%d = X%d_%d * X%d_1;" % (i, p, i, p - 1, i))
    P.w("const double *xs = Xs + lane;")
    P.w("double *sc = SC + lane;")
    P.w("__syncthreads();")

    def lin(row, names):
        (k0, c0) = row[0]
        e = names[k0] if c0 == 1.0 else "%r * %s" % (float(c0), names[k0])
        for (k, c) in row[1:]:
            e = "fma(%r, %s, %s)" % (float(c), names[k], e)
        return e

    P.w("switch (warp) {")
    for g, jbs in enumerate(groups):
        P.w("case %d: {" % g)
        P.ind += 1
        # input-major order: every input (e0| of the row is read from shared memory ONCE per warp and scattered into the
        # (a b| of this warp's b's (registers), instead of being re-read for every (b, k) it occurs in
        terms = {}        # input index -> [(jb, ia, k)]
        for jb in jbs:
            b = B[jb]
            for kx in range(b[0] + 1):
                for ky in range(b[1] + 1):
                    for kz in range(b[2] + 1):
                        for ia, a in enumerate(A):
                            terms.setdefault(idx[(a[0] + kx, a[1] + ky, a[2] + kz)], []).append((jb, ia, (kx, ky, kz)))
        for jb in jbs:
            P.w("double " + ", ".join("o%d_%d" % (jb, ia) for ia in range(len(A))) + ";")
        cfname = {}
        for jb in jbs:
            b = B[jb]
            for kx in range(b[0] + 1):
                for ky in range(b[1] + 1):
                    for kz in range(b[2] + 1):
                        k = (kx, ky, kz)
                        if k == b:
                            continue
                        cst = comb(b[0], kx) * comb(b[1], ky) * comb(b[2], kz)
                        fac = [("X%d_%d" % (i, b[i] - k[i])) for i in range(3) if b[i] - k[i] > 0]
                        nm = "cf%d_%d%d%d" % (jb, kx, ky, kz)
                        P.w("const double %s = %s;" % (nm, " * ".join(([("%d.0" % cst)] if cst != 1 else []) + fac)))
                        cfname[(jb, k)] = nm
        init = set()
        for e in sorted(terms):
            P.w("{ const double x = xs[%d];" % (e * RST))
            for (jb, ia, k) in terms[e]:
                o = "o%d_%d" % (jb, ia)
                if k == B[jb]:
                    if o in init:
                        P.w("  %s += x;" % o)
                    else:
                        P.w("  %s = x;" % o)
                else:
                    if o in init:
                        P.w("  %s = fma(%s, x, %s);" % (o, cfname[(jb, k)], o))
                    else:
                        P.w("  %s = %s * x;" % (o, cfname[(jb, k)]))
                init.add(o)
            P.w("}")
        for jb in jbs:
            names = ["o%d_%d" % (jb, ia) for ia in range(len(A))]
            for ma, row in enumerate(T1):
                P.w("sc[%d] = %s;" % ((ma * nb2 + jb) * RST, lin(row, names)))
        P.ind -= 1
        P.w("} break;")
    P.w("default: break;")
    P.w("}")
    P.w("__syncthreads();")
    P.w("double *y = s.Y + ql * s.yq + (int64_t)(r / s.R2) * s.sr0 + (int64_t)(r % s.R2) * s.sr1;")
    P.w("if (valid)")
    P.w("switch (warp) {")
    for g in range(nw):
        P.w("case %d: {" % g)
        P.ind += 1
        for ma in range(g, ns1, nw):
            P.w("{")
            P.ind += 1
            names = []
            for jb in range(nb2):
                P.w("const double h%d = sc[%d];" % (jb, (ma * nb2 + jb) * RST))
                names.append("h%d" % jb)
            for mb, row in enumerate(T2):
                P.w("y[%d * s.so0 + %d * s.so1] = %s;" % (ma, mb, lin(row, names)))
            P.ind -= 1
            P.w("}")
        P.ind -= 1
        P.w("} break;")
    P.w("default: break;")
    P.w("}")
    P.ind = 0
    P.w("}")
    return NE, ns1 * nb2, nw


def emit(lmax=4):
    P = Prog()
    P.ind = 0
    P.w("// GENERATED by paper_2605_10312_b200/gen/emit_sides.py -- do not edit.")
    P.w('#include "rcg_sides.h"')
    meta = {}
    pairs = [(l1, l2) for l1 in range(lmax + 1) for l2 in range(l1 + 1)]
    for (l1, l2) in pairs:
        meta[(l1, l2)] = emit_side(P, l1, l2)
    P.w("cudaError_t rcg_side_launch(int l1, int l2, const RcgSideArgs &s, cudaStream_t stream)")
    P.w("{")
    P.w("    if (s.nrows <= 0) return cudaSuccess;")
    P.w("    const unsigned blocks = (unsigned)((s.nrows + %d) / %d);" % (ROWS - 1, ROWS))
    P.w("    cudaError_t e = cudaSuccess;")
    P.w("    switch (l1 * 8 + l2) {")
    for (l1, l2) in pairs:
        NE, nsc, nw = meta[(l1, l2)]
        smem = (NE + nsc) * RST * 8
        P.w("    case %d: {" % (l1 * 8 + l2))
        P.w("        static RcgOnce once;")
        P.w("        if ((e = rcg_prepare_kernel(once, (const void *)rcg_side_kernel_%d%d, %d, nullptr)) != cudaSuccess) return e;" % (l1, l2, smem))
        P.w("        rcg_side_kernel_%d%d<<<blocks, %d, %d, stream>>>(s);" % (l1, l2, 32 * nw, smem))
        P.w("    } break;")
    P.w("    default: return cudaErrorInvalidValue;")
    P.w("    }")
    P.w("    return cudaGetLastError();")
    P.w("}")
    return P.text() + "\n"
