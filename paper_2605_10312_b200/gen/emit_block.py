"""Emit the LEVEL-SYNCHRONOUS block tier kernel of one class: one thread BLOCK per shell quartet (round 1's block tier; superseded by the
slab layout of gen/emit_heavy.py, which keeps the ket chains in registers, and kept as the generator variant `--set GEN_NO_SLAB=1` for the
ablation of DESIGN.md 4.10; emit_side_dfs below is still the Phase 2 of the slab kernels).

For bra sides wider than a warp ((fd|, (ff|: 56 / 84 Cartesian components over all levels) with ket
tables too large for the register file.  The decomposition is the warp tier's carried
over to a block, with the ket table moved from registers into shared memory:
  * thread = one bra Cartesian component a, |a| in [0, la+lb] (targets AND lower components; the
    pruned graph gives lower levels smaller tables, so one uniform program serves every thread);
  * the pure-bra vertices [a0|00]^(m) are built thread-locally along the thread's own path
    (identity steps first, as in the warp tier), m = 0..L;
  * the ket table [a0|c0]^(m) of the thread lives in ITS column of a shared-memory table laid out
    [slot][thread] (conflict-free for own-column traffic); ket levels |c| = 1..lc+ld are built one
    after the other with a block barrier in between, the cross term [a-1i|c-1i]^(m+1) of Eq. (2)'s ket
    mirror (reading R-KET) is a gather from the column of the thread that owns a-1i;
    slots rotate over three level buffers (a level is read only by the next two: the lifetime packing of
    PAPER.md:265 in its level-synchronous form);
  * target threads keep the nC contraction accumulators H[a][.] (Alg. 2 line 7) in
    registers across the primitive loop;
  * Phase 2 (HRR + stepwise c2s) runs the class's table-driven node programs (csrc/rcg_phase2.cuh),
    warps taking ket columns / spherical bra rows round-robin, H and the half-transformed block in
    shared memory.
"""
import os

from . import options
from .graph import VrrGraph, hrr_c2s_program, reduction_axis, sub1
from .solid import cart_comps, ncart, c2s_rows
from .emit_warp import Prog


def block_layout(cls):
    """static sizes of the block kernel of one class (also used by tiers.py to decide eligibility)."""
    la, lb, lc, ld = cls
    g = VrrGraph(la, lb, lc, ld)
    nst, ctop = la + lb, lc + ld
    L = nst + ctop
    BC = [a for e in range(0, nst + 1) for a in cart_comps(e)]
    NB = len(BC)
    NTH = (NB + 31) // 32 * 32
    D = [0] * (ctop + 1)
    for (a, c, m) in g.nodes:
        D[sum(c)] = max(D[sum(c)], m + 1)
    D[0] = L + 1
    for k in range(1, ctop + 1):
        assert D[k - 1] >= D[k] + 1
    size = [ncart(k) * D[k] for k in range(ctop + 1)]
    size[0] = L + 1
    # a top-level vertex has no consumer and is not stored
    stored = [size[k] if k < ctop or ctop == 0 else 0 for k in range(ctop + 1)]
    reg = [0, 0, 0]
    for k in range(ctop + 1):
        reg[k % 3] = max(reg[k % 3], stored[k])
    base = [0, reg[0], reg[0] + reg[1]]
    nslot = sum(reg)
    nT = len(g.target_a)
    nC = len(g.target_c)
    nAB = (2 * la + 1) * (2 * lb + 1)
    bra = hrr_c2s_program(la, lb)
    ket = hrr_c2s_program(lc, ld)
    return dict(g=g, nst=nst, ctop=ctop, L=L, BC=BC, NB=NB, NTH=NTH, D=D, base=base, nslot=nslot,
                nT=nT, nC=nC, nAB=nAB, bra=bra, ket=ket)


def add1(t, i):
    return tuple(v + (1 if k == i else 0) for k, v in enumerate(t))


def side_live(l1, l2):
    """doubles live in registers along one depth-first path of emit_side_dfs."""
    return sum(sum(ncart(e) for e in range(l1, l1 + l2 - nb + 1)) for nb in range(1, l2 + 1))


def emit_side_dfs(P, l1, l2, inp, X, sc, outw, vp):
    """One side of Phase 2 for ONE thread (a fixed index of the other side), straight-line:
    HRR of Eq. (3) (a,b+1i| = (a+1i,b| + X_i (a,b| walked DEPTH-FIRST over the tree of
    b (axes added in non-decreasing order), so that only the arrays along the current path are live
    (46+25+10 doubles at (ff|) and nothing is recomputed; at a leaf |b| = l2 the first index is made
    spherical (T^(l1), Eq. (11)) and parked in the thread's scratch column; a second pass applies T^(l2)
    (Eq. (12)).  inp(k): expression of input k ((e0| in level-major order); sc(i): scratch lvalue;
    outw(r, expr): store of output r = ma*nsph(l2)+mb."""
    lev = list(range(l1, l1 + l2 + 1))
    iidx = {}
    for e in lev:
        for a in cart_comps(e):
            iidx[a] = len(iidx)
    A, B = cart_comps(l1), cart_comps(l2)
    T1, T2 = c2s_rows(l1), c2s_rows(l2)
    nb2 = len(B)

    def term(coef, name, first):
        if coef == 1.0:
            return name if first else " + %s" % name
        if coef == -1.0:
            return "-%s" % name if first else " - %s" % name
        return "%r * %s" % (float(coef), name) if first else " + %r * %s" % (float(coef), name)

    def lin(row, names):
        # sum_k coef_k * names[k] as nested fma
        (k0, c0) = row[0]
        e = names[k0] if c0 == 1.0 else "%r * %s" % (float(c0), names[k0])
        for (k, c) in row[1:]:
            e = "fma(%r, %s, %s)" % (float(c), names[k], e)
        return e

    def leaf(b, arr):
        jb = B.index(b)
        names = [arr(a) for a in A]
        for ma, row in enumerate(T1):
            P.w("%s = %s;" % (sc(ma * nb2 + jb), lin(row, names)))

    def rec(b, arr, depth):
        if sum(b) == l2:
            leaf(b, arr)
            return
        last = max([i for i in range(3) if b[i] > 0] + [0])
        for i in range(last, 3):
            b2 = add1(b, i)
            reg = [a for e in range(l1, l1 + l2 - sum(b2) + 1) for a in cart_comps(e)]
            P.w("{")
            P.ind += 1
            names = {}
            for n, a in enumerate(reg):
                nm = "%s%d_%d" % (vp, depth + 1, n)
                P.w("const double %s = fma(%s, %s, %s);" % (nm, X[i], arr(a), arr(add1(a, i))))
                names[a] = nm
            rec(b2, lambda a, names=names: names[a], depth + 1)
            P.ind -= 1
            P.w("}")

    rec((0, 0, 0), lambda a: inp(iidx[a]), 0)
    for ma in range(len(T1)):
        P.w("{")
        P.ind += 1
        names = []
        for j in range(nb2):
            P.w("const double %sr%d = %s;" % (vp, j, sc(ma * nb2 + j)))
            names.append("%sr%d" % (vp, j))
        for mb, row in enumerate(T2):
            outw(ma * len(T2) + mb, lin(row, names))
        P.ind -= 1
        P.w("}")


def emit_class(cls):
    la, lb, lc, ld = cls
    lay = block_layout(cls)
    g, nst, ctop, L = lay["g"], lay["nst"], lay["ctop"], lay["L"]
    BC, NB, NTH, D, base, NSLOT = lay["BC"], lay["NB"], lay["NTH"], lay["D"], lay["base"], lay["nslot"]
    nT, nC, nAB = lay["nT"], lay["nC"], lay["nAB"]
    tag = "%d%d%d%d" % cls
    nlowc = sum(ncart(e) for e in range(la))
    bidx = {a: i for i, a in enumerate(BC)}
    TC = [c for f in range(lc, lc + ld + 1) for c in cart_comps(f)]
    tpos = {c: t for t, c in enumerate(TC)}
    cidx = [{c: i for i, c in enumerate(cart_comps(k))} for k in range(ctop + 1)]

    def slot(c, m):
        k = sum(c)
        if k == 0:
            return base[0] + m
        return base[k % 3] + cidx[k][c] * D[k] + m

    # primitive record
    OFF_PA = L + 1
    OFF_WP = OFF_PA + 4
    OFF_HZN = OFF_WP + 4
    OFF_RZ = OFF_HZN + max(nst, 1)
    OFF_QC = OFF_RZ + 1
    OFF_WQ = OFF_QC + 3
    OFF_HE = OFF_WQ + 3
    OFF_RE = OFF_HE + 1
    OFF_HZE = OFF_RE + 1
    PRS = (OFF_HZE + 1) | 1
    PBS = 32
    # blocks per SM: what shared memory allows, but never so many that ptxas must squeeze the accumulators
    # (nC doubles) and the pure-bra chain (2(L+1) doubles) below what they need
    # (with few ket columns the bra side runs on few threads, but even one thread per column beats the
    # table-driven interpreter of rcg_phase2.cuh: measured 1.4-5x on (ff|ss)..(ff|fs))
    gen_p2 = nC >= options.geti("BLOCK_P2_MINCOLS", 1) and nC <= NTH and nAB <= NTH \
        and max(side_live(la, lb), side_live(lc, ld)) <= 90
    regs_needed = 2 * nC + 4 * (L + 1) + 100
    if gen_p2:
        regs_needed = max(regs_needed, 2 * max(side_live(la, lb), side_live(lc, ld)) + 56)
    regs_needed = min(255, regs_needed)
    # (ptxas budgets registers per block in units of 4 warps: 96 threads count as 128)
    nth_alloc = (NTH + 127) // 128 * 128
    minb = max(1, min(8, (227 * 1024) // ((NSLOT * NTH + PBS * PRS) * 8 + 1024),
                      65536 // (nth_alloc * ((regs_needed + 7) // 8 * 8))))
    if gen_p2 and nC < 20:
        # few ket columns: Phase 2 runs on few threads and is latency-bound, a third block per SM is worth more
        # than the ~350 spill bytes its depth-first (ff| program then has (measured 12-20% faster)
        minb = max(minb, min(3, (227 * 1024) // ((NSLOT * NTH + PBS * PRS) * 8 + 1024)))
    minb = options.geti("BLOCK_MINB", 0) or minb

    # thread table: ax ay az | source threads of a-1x, a-1y, a-1z | path selectors | path counts
    rows = []
    for t in range(NTH):
        a = BC[t] if t < NB else (0, 0, 0)
        src = [bidx[sub1(a, i)] if a[i] > 0 else t for i in range(3)]
        steps = [(ax, n) for ax in range(3) for n in range(a[ax])]
        pad = nst - len(steps)
        sel = [3] * pad + [ax for ax, _ in steps]
        nn = [0] * pad + [n for _, n in steps]
        rows.append(list(a) + src + sel + nn)
    NR = len(rows[0])

    P = Prog()
    P.ind = 0
    P.w("// ---- block tier kernel for (%d %d|%d %d): generated by gen/emit_block.py" % cls)
    P.w("// bra components (threads) %d of %d, ket levels 0..%d with depths %s, table %d slots/thread (%d B/block),"
        % (NB, NTH, ctop, D, NSLOT, NSLOT * NTH * 8))
    P.w("// accumulators/thread %d, blocks/SM %d" % (nC, minb))
    P.w('#include "rcg_device.cuh"')
    P.w('#include "rcg_phase2.cuh"')
    P.w("extern const RcgClassDesc rcg_class_%s;" % tag)
    P.w("namespace b%s {" % tag)
    P.w("constexpr int NTH = %d, NW = %d, NB = %d, NLOWC = %d, NSLOT = %d, PRS = %d, PBS = %d, NT = %d, NC = %d, NAB = %d;"
        % (NTH, NTH // 32, NB, nlowc, NSLOT, PRS, PBS, nT, nC, nAB))
    P.w("constexpr int VRR_DOUBLES = NSLOT * NTH + PBS * PRS;")
    # per-thread statics packed into three words (kept in registers; unpacked with shifts where used):
    # w0 = ax | ay<<4 | az<<8 ; w1 = source threads of a-1x | a-1y<<8 | a-1z<<16 ;
    # w2 = path selectors (2 bits per step) | path counts (3 bits per step) << 2*nst
    assert NTH <= 256 and 5 * nst <= 32
    P.w("__device__ const unsigned c_thr[%d][3] = {     // global, not __constant__: divergent constant-bank loads serialise" % NTH)
    for r in rows:
        w0 = r[0] | (r[1] << 4) | (r[2] << 8)
        w1 = r[3] | (r[4] << 8) | (r[5] << 16)
        w2 = 0
        for s_ in range(nst):
            w2 |= r[6 + s_] << (2 * s_)
            w2 |= r[6 + nst + s_] << (2 * nst + 3 * s_)
        P.w("  {%du,%du,%du}," % (w0, w1, w2))
    P.w("};")
    P.w("__global__ void __launch_bounds__(NTH, %d) rcg_eri_block_%s(GDev g, RcgLaunch a)" % (minb, tag))
    P.w("{")
    P.ind = 1
    P.w("extern __shared__ __align__(16) double smem[];")
    P.w("const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;")
    P.w("double *TAB = smem + tid;                  // own column of the [slot][thread] ket table")
    P.w("double *REC = smem + NSLOT * NTH;          // primitive records [PBS][PRS]")
    P.w("const RcgBasisDev &b = a.basis;")
    P.w("const unsigned tw0 = __ldg(&c_thr[tid][0]), tw1 = __ldg(&c_thr[tid][1]), tw2 = __ldg(&c_thr[tid][2]);")
    if nst:
        P.w("const double *X0 = smem + (tw1 & 255u), *X1 = smem + ((tw1 >> 8) & 255u), *X2 = smem + (tw1 >> 16);   // columns of a-1x, a-1y, a-1z")
    P.w("for (int64_t q = blockIdx.x; q < a.n; q += gridDim.x) {")
    P.w("const int sh0 = a.quartets[4 * q + a.perm[0]], sh1 = a.quartets[4 * q + a.perm[1]];")
    P.w("const int sh2 = a.quartets[4 * q + a.perm[2]], sh3 = a.quartets[4 * q + a.perm[3]];")
    P.w("const int pa0 = b.prim_off[sh0], Ka = b.prim_off[sh0 + 1] - pa0;")
    P.w("const int pb0 = b.prim_off[sh1], Kb = b.prim_off[sh1 + 1] - pb0;")
    P.w("const int pc0 = b.prim_off[sh2], Kc = b.prim_off[sh2 + 1] - pc0;")
    P.w("const int pd0 = b.prim_off[sh3], Kd = b.prim_off[sh3 + 1] - pd0;")
    P.w("const int K4 = Ka * Kb * Kc * Kd;")
    for t in range(nC):
        P.w("double acc%d = 0.0;" % t)
    P.w("for (int p0 = 0; p0 < K4; p0 += PBS) {")
    P.ind += 1
    P.w("const int cnt = min(PBS, K4 - p0);")
    P.w("__syncthreads();                        // the previous batch's records / Phase-2 buffers are no longer read")
    P.w("if (tid < cnt) {                        // primitive set-up, one primitive quartet per thread (Alg. 2 lines 4-5)")
    P.ind += 1
    P.w("double RA[3], RB[3], RC[3], RD[3];")
    P.w("#pragma unroll")
    P.w("for (int t = 0; t < 3; ++t) { RA[t] = b.centers[3 * sh0 + t]; RB[t] = b.centers[3 * sh1 + t]; RC[t] = b.centers[3 * sh2 + t]; RD[t] = b.centers[3 * sh3 + t]; }")
    P.w("int p = p0 + tid;")
    P.w("const float rKd = __fdividef(1.0f, (float)Kd), rKc = __fdividef(1.0f, (float)Kc), rKb = __fdividef(1.0f, (float)Kb);")
    P.w("int il, ik, ij; p = rcg_divmod(p, Kd, rKd, il); p = rcg_divmod(p, Kc, rKc, ik); const int ii = rcg_divmod(p, Kb, rKb, ij);")
    P.w("RcgPrim pq;")
    P.w("rcg_prim_setup(pq, RA, RB, RC, RD, b.exps[pa0 + ii], b.exps[pb0 + ij], b.exps[pc0 + ik], b.exps[pd0 + il],")
    P.w("               b.coefs[pa0 + ii] * b.coefs[pb0 + ij] * b.coefs[pc0 + ik] * b.coefs[pd0 + il]);")
    P.w("double F[%d];" % (L + 1))
    P.w("rcg_boys<%d>(%d, pq.T, pq.pref, b.boys, F);" % (L, L))
    P.w("double *pr = REC + tid * PRS;")
    P.w("#pragma unroll")
    P.w("for (int m = 0; m <= %d; ++m) pr[m] = F[m];" % L)
    P.w("pr[%d] = pq.PA[0]; pr[%d] = pq.PA[1]; pr[%d] = pq.PA[2]; pr[%d] = 1.0;" % (OFF_PA, OFF_PA + 1, OFF_PA + 2, OFF_PA + 3))
    P.w("pr[%d] = pq.WP[0]; pr[%d] = pq.WP[1]; pr[%d] = pq.WP[2]; pr[%d] = 0.0;" % (OFF_WP, OFF_WP + 1, OFF_WP + 2, OFF_WP + 3))
    for n in range(max(nst, 1)):
        P.w("pr[%d] = %d.0 * pq.hz;" % (OFF_HZN + n, n))
    P.w("pr[%d] = pq.rz;" % OFF_RZ)
    P.w("pr[%d] = pq.QC[0]; pr[%d] = pq.QC[1]; pr[%d] = pq.QC[2];" % (OFF_QC, OFF_QC + 1, OFF_QC + 2))
    P.w("pr[%d] = pq.WQ[0]; pr[%d] = pq.WQ[1]; pr[%d] = pq.WQ[2];" % (OFF_WQ, OFF_WQ + 1, OFF_WQ + 2))
    P.w("pr[%d] = pq.he; pr[%d] = pq.re; pr[%d] = pq.hze;" % (OFF_HE, OFF_RE, OFF_HZE))
    P.ind -= 1
    P.w("}")
    P.w("__syncthreads();")
    P.w("for (int jj = 0; jj < cnt; ++jj) {")
    P.ind += 1
    P.w("const double *pr = REC + jj * PRS;")
    # ---- pure-bra chain: every step computes all L+1 Boys orders (identity steps keep the full range)
    cur = []
    for m in range(L + 1):
        P.w("const double x0_%d = pr[%d];" % (m, m))
        cur.append("x0_%d" % m)
    prev = None
    if nst >= 2:
        P.w("const double rz = pr[%d];" % OFF_RZ)
    for s in range(1, nst + 1):
        P.w("const double *ps%d = pr + %d + ((tw2 >> %d) & 3u);" % (s, OFF_PA, 2 * (s - 1)))
        P.w("const double c1_%d = ps%d[0], c2_%d = ps%d[4];" % (s, s, s, s))
        if s >= 2:
            P.w("const double kn_%d = pr[%d + ((tw2 >> %d) & 7u)];" % (s, OFF_HZN, 2 * nst + 3 * (s - 1)))
        new = []
        for m in range(L + 1):
            nm = "x%d_%d" % (s, m)
            up = cur[m + 1] if m + 1 <= L else None
            if up:
                P.w("double %s = fma(c2_%d, %s, c1_%d * %s);" % (nm, s, up, s, cur[m]))
            else:
                P.w("double %s = c1_%d * %s;" % (nm, s, cur[m]))
            if s >= 2:
                pu = prev[m + 1] if m + 1 <= L else None
                u = "fma(-rz, %s, %s)" % (pu, prev[m]) if pu else prev[m]
                P.w("%s = fma(kn_%d, %s, %s);" % (nm, s, u, nm))
            new.append(nm)
        prev, cur = cur, new
    bvals = cur
    if (0, 0, 0) in tpos:
        P.w("acc%d += %s;" % (tpos[(0, 0, 0)], bvals[0]))
    if ctop >= 1:
        P.w("const double QC0 = pr[%d], QC1 = pr[%d], QC2 = pr[%d];" % (OFF_QC, OFF_QC + 1, OFF_QC + 2))
        P.w("const double WQ0 = pr[%d], WQ1 = pr[%d], WQ2 = pr[%d];" % (OFF_WQ, OFF_WQ + 1, OFF_WQ + 2))
        P.w("const double he = pr[%d], re = pr[%d];" % (OFF_HE, OFF_RE))
        for n in range(2, ctop):
            P.w("const double hen%d = %d.0 * he;" % (n, n))
        if nst:
            P.w("const double hze = pr[%d];" % OFF_HZE)
            P.w("const double ka0 = (double)(int)(tw0 & 15u) * hze, ka1 = (double)(int)((tw0 >> 4) & 15u) * hze, ka2 = (double)(int)(tw0 >> 8) * hze;")
        if (ctop - 1) % 3 == 0 and nst:
            P.w("__syncthreads();                    // the previous primitive's top-level gathers of this region are done")
        for m in range(L + 1):
            P.w("TAB[%d] = %s;" % ((base[0] + m) * NTH, bvals[m]))
    for k in range(1, ctop + 1):
        if nst:
            P.w("__syncthreads();                    // ket level %d: level %d of every thread is visible" % (k, k - 1))
        Dk = D[k]
        for c1 in cart_comps(k - 1):
            children = [(2, tuple(v + (1 if j == 2 else 0) for j, v in enumerate(c1)))]
            if c1[2] == 0:
                children.append((1, tuple(v + (1 if j == 1 else 0) for j, v in enumerate(c1))))
                if c1[1] == 0:
                    children.append((0, tuple(v + (1 if j == 0 else 0) for j, v in enumerate(c1))))
            for (i, c) in children:
                assert reduction_axis(c) == i and sub1(c, i) == c1
            P.w("{")
            P.ind += 1
            if k - 1 == 0:
                pn = bvals
            else:
                pn = []
                for m in range(Dk + 1):
                    P.w("const double p%d = TAB[%d];" % (m, slot(c1, m) * NTH))
                    pn.append("p%d" % m)
            for (i, c) in children:
                n2 = c1[i]
                P.w("{")
                P.ind += 1
                if n2:
                    c2 = sub1(c1, i)
                    if k - 2 == 0:
                        gn = bvals
                    else:
                        gn = []
                        for m in range(Dk + 1):
                            P.w("const double g%d = TAB[%d];" % (m, slot(c2, m) * NTH))
                            gn.append("g%d" % m)
                if nst:
                    for m in range(Dk):
                        P.w("const double x%d = X%d[%d];" % (m, i, slot(c1, m + 1) * NTH))
                hen = {0: None, 1: "he"}
                for m in range(Dk):
                    leaf = (k == ctop and m == 0 and c in tpos)
                    if leaf:
                        nm = "acc%d" % tpos[c]
                        P.w("%s = fma(QC%d, %s, %s);" % (nm, i, pn[m], nm))
                    else:
                        nm = "v%d" % m
                        P.w("double %s = QC%d * %s;" % (nm, i, pn[m]))
                    P.w("%s = fma(WQ%d, %s, %s);" % (nm, i, pn[m + 1], nm))
                    if n2:
                        P.w("%s = fma(%s, fma(-re, %s, %s), %s);" % (nm, hen.get(n2, "hen%d" % n2), gn[m + 1], gn[m], nm))
                    if nst:
                        P.w("%s = fma(ka%d, x%d, %s);" % (nm, i, m, nm))
                    if k < ctop:
                        P.w("TAB[%d] = %s;" % (slot(c, m) * NTH, nm))
                    if m == 0 and c in tpos and not leaf:
                        P.w("acc%d += %s;" % (tpos[c], nm))
                P.ind -= 1
                P.w("}")
            P.ind -= 1
            P.w("}")
    P.ind -= 1
    P.w("}")
    P.ind -= 1
    P.w("}")
    # ---------------- Phase 2
    nCD = (2 * lc + 1) * (2 * ld + 1)
    HST = max(nC, nCD) | 1               # odd row stride of H: conflict-free for thread = column and thread = row
    SCN = max((2 * la + 1) * ncart(lb), (2 * lc + 1) * ncart(ld))
    P2_DOUBLES = nT * HST + SCN * NTH
    if not gen_p2:
        P.w("__syncthreads();                            // table region becomes H | Bh | per-warp Phase-2 vectors")
        P.w("double *Hs = smem, *Bh = smem + NT * NC, *wbuf = Bh + NAB * NC;")
        P.w("if (tid >= NLOWC && tid < NB) {")
        P.ind += 1
        P.w("double *h = Hs + (tid - NLOWC) * NC;")
        for t in range(nC):
            P.w("h[%d] = acc%d;" % (t, t))
        P.ind -= 1
        P.w("}")
        P.w("double AB[3], CD[3];")
        P.w("#pragma unroll")
        P.w("for (int t = 0; t < 3; ++t) { AB[t] = b.centers[3 * sh0 + t] - b.centers[3 * sh1 + t]; CD[t] = b.centers[3 * sh2 + t] - b.centers[3 * sh3 + t]; }")
        P.w("__syncthreads();")
        P.w("rcg_phase2_block(g, a, q, Hs, Bh, wbuf, AB, CD, warp, lane, NW);")
    else:
        # generated Phase 2: thread = ket column runs the bra side, thread = spherical bra row runs the ket
        # side (Eqs. (11)-(16)), each as a depth-first straight-line program; the
        # half-transformed block and the result overwrite H in place (a thread only touches its own column / row)
        P.w("__syncthreads();                            // table region becomes H [NT][HST] | scratch columns [SCN][NTH]")
        P.w("double *Hs = smem, *SC = smem + NT * %d + tid;" % HST)
        P.w("if (tid >= NLOWC && tid < NB) {")
        P.ind += 1
        P.w("double *h = Hs + (tid - NLOWC) * %d;" % HST)
        for t in range(nC):
            P.w("h[%d] = acc%d;" % (t, t))
        P.ind -= 1
        P.w("}")
        P.w("__syncthreads();")
        P.w("if (tid < NC) {                             // bra HRR + Ta, Tb on ket column tid")
        P.ind += 1
        P.w("const double AB0 = b.centers[3 * sh0] - b.centers[3 * sh1], AB1 = b.centers[3 * sh0 + 1] - b.centers[3 * sh1 + 1], AB2 = b.centers[3 * sh0 + 2] - b.centers[3 * sh1 + 2];")
        P.w("double *hc = Hs + tid;")
        emit_side_dfs(P, la, lb, lambda k: "hc[%d]" % (k * HST), ["AB0", "AB1", "AB2"],
                      lambda i: "SC[%d]" % (i * NTH), lambda r, e: P.w("hc[%d] = %s;" % (r * HST, e)), "h")
        P.ind -= 1
        P.w("}")
        P.w("__syncthreads();")
        P.w("if (tid < NAB) {                            // ket HRR + Tc, Td on spherical bra row tid")
        P.ind += 1
        P.w("const double CD0 = b.centers[3 * sh2] - b.centers[3 * sh3], CD1 = b.centers[3 * sh2 + 1] - b.centers[3 * sh3 + 1], CD2 = b.centers[3 * sh2 + 2] - b.centers[3 * sh3 + 2];")
        P.w("double *hr = Hs + tid * %d;" % HST)
        emit_side_dfs(P, lc, ld, lambda k: "hr[%d]" % k, ["CD0", "CD1", "CD2"],
                      lambda i: "SC[%d]" % (i * NTH), lambda r, e: P.w("hr[%d] = %s;" % (r, e)), "g")
        P.ind -= 1
        P.w("}")
        P.w("__syncthreads();")
        nsb, nsc, nsd = 2 * lb + 1, 2 * lc + 1, 2 * ld + 1
        P.w("double *out = a.out + q * a.out_stride;")
        P.w("const bool canon = a.ostride[3] == 1 && a.ostride[2] == %d && a.ostride[1] == %d && a.ostride[0] == %d;"
            % (nsd, nsd * nsc, nsd * nsc * nsb))
        P.w("for (int e = tid; e < %d; e += NTH) {" % (nAB * nCD))
        P.w("    const int o = e / %d, r = e %% %d;" % (nCD, nCD))
        P.w("    const double v = Hs[o * %d + r];" % HST)
        P.w("    if (canon) out[e] = v;")
        P.w("    else {")
        P.w("        const int id = r %% %d, ic = r / %d, ib = o %% %d, ia = o / %d;" % (nsd, nsd, nsb, nsb))
        P.w("        out[ia * a.ostride[0] + ib * a.ostride[1] + ic * a.ostride[2] + id * a.ostride[3]] = v;")
        P.w("    }")
        P.w("}")
    P.w("}   // quartet loop")
    P.ind = 0
    P.w("}")
    P.w("}  // namespace b%s" % tag)
    P.w("static cudaError_t rcg_launch_block_%s(const RcgLaunch &a)" % tag)
    P.w("{")
    P.w("    using namespace b%s;" % tag)
    P.w("    GDev g;")
    P.w("    cudaError_t e = rcg_global_tables(rcg_class_%s, &g);" % tag)
    P.w("    if (e != cudaSuccess) return e;")
    if gen_p2:
        P.w("    size_t dbl = %d;      // generated Phase 2: H + scratch columns" % P2_DOUBLES)
    else:
        P.w("    size_t dbl = (size_t)NT * NC + (size_t)NAB * NC + (size_t)NW * g.p2_slots;")
    P.w("    if (dbl < (size_t)VRR_DOUBLES) dbl = VRR_DOUBLES;")
    P.w("    const size_t smem = sizeof(double) * dbl;")
    P.w("    static RcgOnce once;              // shared-memory limit raised once per device (thread-safe)")
    P.w("    if ((e = rcg_prepare_kernel(once, (const void *)rcg_eri_block_%s, smem, nullptr)) != cudaSuccess) return e;" % tag)
    P.w("    const int64_t blocks = a.n < (1ll << 30) ? a.n : (1ll << 30);     // one block per quartet: the hardware balances uneven K4")
    P.w("    rcg_eri_block_%s<<<(unsigned)blocks, NTH, smem, a.stream>>>(g, a);" % tag)
    P.w("    return cudaGetLastError();")
    P.w("}")
    meta = dict(block_threads=NTH, block_bra_components=NB, block_table_slots=NSLOT,
                block_table_bytes=NSLOT * NTH * 8, block_accumulators_per_thread=nC, block_ket_depths=D,
                block_blocks_per_sm=minb, block_generated_phase2=bool(gen_p2))
    return P.text() + "\n", "rcg_launch_block_%s" % tag, meta
