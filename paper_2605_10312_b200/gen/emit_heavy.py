"""Emit the block tiers for wide bra sides (RCG_TIER_BLOCK): one thread block per shell quartet, thread = bra component, the ket
recurrence CHAINS in registers.  Two layouts: emit_class (z-column layout: (gf|xx), (gg|xx); VRR + contraction in one kernel, Phase 2
in two class-independent side kernels, gen/emit_sides.py) and, further down, emit_class_slab (slab layout: bra sides up to la + lb = 6).

Why a third decomposition.  (gg|gg) has 165 bra components, 486 ket vertices per component and
145 x 145 contraction accumulators (Alg. 2 line 7): neither the accumulators (42 k registers of an
SM's 64 k) nor the level-synchronous shared-memory ket table of the block tier (373 KB) fit.  What does fit:

  * thread = one bra Cartesian component a, |a| in [0, la+lb], as in the block tier -- but the components are laid
    out so that the z-COLUMN of a (fixed ax, ay; az ascending) sits in consecutive lanes of one warp.  With the
    ket-first z -> y -> x axis rule a ket vertex [a|c] with cz > 0 reads [a|c-1z], [a|c-2z] (own
    thread) and the cross term [a-1z|c-1z]^(m+1) (Eq. (2)'s ket mirror, reading R-KET): lane - 1.  So every ket
    z-CHAIN (cx, cy, 0..) runs in REGISTERS, its cross terms by __shfl_up_sync -- two thirds of all vertices touch no
    shared memory;
  * only the chain HEADS (cx, cy, 0) -- reduced along y or x, cross terms from other warps -- go level by level
    (|c| = cx + cy) through a [slot][thread] shared-memory table with three rotating level buffers (the lifetime
    packing of PAPER.md:265 in level-synchronous form): 73 slots per thread at (gg|gg) instead of 243;
  * the accumulators stay in registers; when a thread would need more than ACC_CAP of them the ket side is cut into
    PASSES over x-slabs (sets of cx): a pass repeats the primitive loop for its slabs only (pure-bra chain and x-chain
    recomputed) and writes its columns of H to the launch's workspace;
  * H[quartet][ket target][bra target] then goes through the side kernels: bra HRR + Ta, Tb (Eqs. (3), (11)-(12)),
    ket HRR + Tc, Td (Eqs. (13)-(16)) -- the paper's Tier-2 shape (evaluation kernel, buffered hand-over, transform
    kernels), with the buffer sized to stay in the 126 MB L2.
"""
from . import options
from .solid import cart_comps, ncart
from .emit_warp import Prog

ACC_CAP = 76            # accumulators (doubles) a thread keeps per pass: measured on the B200 against 32, 48 and 100 ((gg|gg): 7.1 / 6.7 / 5.3 ms per 5,000
                        # quartets with 32 / 48 / 76; 100 spills at (gg|gf), (gg|gg)); two passes of at most 76 at (gg|gg), 254 registers, 0 spill bytes
# (chunks of a launch: csrc/rcg_sides.h, rcg_heavy_chunk -- whole waves of one block per SM, about 96 MB of hand-over buffer)


def zcol_layout(nst):
    """threads of the block: bra components 0..nst grouped into z-columns (ax, ay), az ascending, columns packed into
    warps first-fit by decreasing length (a column never straddles a warp).  -> list of components or None (idle lane)."""
    cols = [(ax, ay) for ax in range(nst + 1) for ay in range(nst + 1 - ax)]
    cols.sort(key=lambda c: (-(nst - c[0] - c[1] + 1), c))
    warps = []
    for col in cols:
        ln = nst - col[0] - col[1] + 1
        for w in warps:
            if len(w) + ln <= 32:
                break
        else:
            w = []
            warps.append(w)
        w.extend((col[0], col[1], az) for az in range(ln))
    thr = []
    for w in warps:
        thr.extend(w + [None] * (32 - len(w)))
    return thr


def slab_targets(lc, ctop, cx):
    """number of ket targets (levels lc..ctop) in the x-slab cx."""
    return sum(k - cx + 1 for k in range(max(lc, cx), ctop + 1))


def slab_families(ctop, cx):
    return (ctop - cx + 1) * (ctop - cx + 2) // 2


def slab_passes(lc, ld, cap=None):
    """partition of the x-slabs 0..ctop into passes with at most `cap` targets each (one slab may exceed it),
    longest-processing-time first on the family count."""
    cap = cap or options.geti("HEAVY_ACC_CAP", 0) or ACC_CAP
    ctop = lc + ld
    nC = sum(ncart(f) for f in range(lc, ctop + 1))
    npass = max(1, -(-nC // cap))
    while True:
        bins = [[] for _ in range(npass)]
        load = [0] * npass
        tgt = [0] * npass
        ok = True
        for cx in sorted(range(ctop + 1), key=lambda c: -slab_families(ctop, c)):
            t = slab_targets(lc, ctop, cx)
            cand = [i for i in range(npass) if tgt[i] + t <= cap or not bins[i]]
            if not cand:
                ok = False
                break
            i = min(cand, key=lambda j: load[j])
            bins[i].append(cx)
            load[i] += slab_families(ctop, cx)
            tgt[i] += t
        if ok:
            return [sorted(b) for b in bins if b]
        npass += 1


def ws_quartet_doubles(cls):
    la, lb, lc, ld = cls
    nT = sum(ncart(e) for e in range(la, la + lb + 1))
    nC = sum(ncart(f) for f in range(lc, lc + ld + 1))
    nAB = (2 * la + 1) * (2 * lb + 1)
    return nT * nC + nAB * nC


def emit_class(cls):
    la, lb, lc, ld = cls
    tag = "%d%d%d%d" % cls
    nst, ctop = la + lb, lc + ld
    L = nst + ctop
    thr = zcol_layout(nst)
    NTH = len(thr)
    NB = sum(1 for t in thr if t is not None)
    tid_of = {a: i for i, a in enumerate(thr) if a is not None}
    T = [a for e in range(la, nst + 1) for a in cart_comps(e)]
    tix_of = {a: i for i, a in enumerate(T)}
    nT = len(T)
    TC = [c for f in range(lc, ctop + 1) for c in cart_comps(f)]
    tpos = {c: t for t, c in enumerate(TC)}
    nC = len(TC)
    nAB = (2 * la + 1) * (2 * lb + 1)
    passes = slab_passes(lc, ld)
    D = [ctop - k + 1 for k in range(ctop + 1)]          # Boys orders m = 0..ctop-k kept at ket level k

    # ---- shared-memory table: level 0 (base values, m = 0..ctop) and the stored heads of every pass
    def pass_heads(Sx):
        """heads of a pass by level: [(cx, cy)] with the x-chain (cx, 0) first."""
        mx = max(Sx)
        out = {}
        for k in range(1, ctop + 1):
            hs = []
            if k <= mx:
                hs.append((k, 0))
            for cx in Sx:
                if cx < k:
                    hs.append((cx, k - cx))
            out[k] = hs
        return out

    def stored(Sx, cx, cy):
        k = cx + cy
        if k >= ctop:
            return False
        return (cx in Sx) or (cy == 0 and cx + 1 <= max(Sx))

    size = [0, 0, 0]
    size[0] = ctop + 1
    slot_of = []                      # per pass: {(cx, cy): first slot offset within its level buffer}
    for Sx in passes:
        so = {}
        hs = pass_heads(Sx)
        for k in range(1, ctop + 1):
            off = 0
            for (cx, cy) in hs[k]:
                if stored(Sx, cx, cy):
                    so[(cx, cy)] = off
                    off += D[k]
            size[k % 3] = max(size[k % 3], off)
        slot_of.append(so)
    base = [0, size[0], size[0] + size[1]]
    NSLOT = sum(size)

    # ---- primitive record (as in the block tier)
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
    smem_doubles = NSLOT * NTH + PBS * PRS
    maxacc = max(sum(slab_targets(lc, ctop, cx) for cx in Sx) for Sx in passes)
    regs_needed = min(255, 2 * maxacc + 6 * (ctop + 2) + 2 * (L + 2) + 64)
    nth_alloc = (NTH + 127) // 128 * 128
    minb = max(1, min(4, (227 * 1024) // (smem_doubles * 8 + 1024), 65536 // (nth_alloc * ((regs_needed + 7) // 8 * 8))))
    minb = options.geti("HEAVY_MINB", 0) or minb

    rows = []
    for t in range(NTH):
        a = thr[t] if thr[t] is not None else (0, 0, 0)
        sx = tid_of[(a[0] - 1, a[1], a[2])] if a[0] > 0 else t
        sy = tid_of[(a[0], a[1] - 1, a[2])] if a[1] > 0 else t
        if a[2] > 0:
            assert tid_of[(a[0], a[1], a[2] - 1)] == t - 1 and (t & 31) > 0
        steps = [(ax, n) for ax in range(3) for n in range(a[ax])]
        pad = nst - len(steps)
        sel = [3] * pad + [ax for ax, _ in steps]
        nn = [0] * pad + [n for _, n in steps]
        tix = tix_of[a] if (thr[t] is not None and sum(a) >= la) else 0xffff
        w0 = a[0] | (a[1] << 4) | (a[2] << 8)
        w1 = sx | (sy << 8) | (tix << 16)
        w2 = w3 = 0
        for s_ in range(nst):
            w2 |= sel[s_] << (2 * s_)
            w3 |= nn[s_] << (3 * s_)
        rows.append((w0, w1, w2, w3))
    assert NTH <= 256 and nT < 0xffff and 3 * nst <= 32

    P = Prog()
    P.ind = 0
    P.w("// ---- heavy block tier kernel for (%d %d|%d %d): generated by gen/emit_heavy.py" % cls)
    P.w("// bra components (threads) %d of %d in z-columns, ket levels 0..%d, head table %d slots/thread (%d B/block),"
        % (NB, NTH, ctop, NSLOT, NSLOT * NTH * 8))
    P.w("// passes over ket x-slabs %s, at most %d accumulators/thread, blocks/SM %d" % (passes, maxacc, minb))
    P.w('#include "rcg_device.cuh"')
    P.w('#include "rcg_sides.h"')
    P.w("namespace h%s {" % tag)
    P.w("constexpr int NTH = %d, NB = %d, NSLOT = %d, PRS = %d, PBS = %d, NT = %d, NC = %d, NAB = %d;"
        % (NTH, NB, NSLOT, PRS, PBS, nT, nC, nAB))
    P.w("constexpr int VRR_DOUBLES = NSLOT * NTH + PBS * PRS;")
    P.w("#define FULL 0xffffffffu")
    P.w("__device__ const unsigned c_thr[%d][4] = {     // ax|ay<<4|az<<8 ; thread of a-1x | a-1y<<8 | target index<<16 ; path selectors ; path counts" % NTH)
    for r in rows:
        P.w("  {%du,%du,%du,%du}," % r)
    P.w("};")
    P.w("__global__ void __launch_bounds__(NTH, %d) rcg_eri_heavy_%s(RcgLaunch a, int64_t q0, double *H)" % (minb, tag))
    P.w("{")
    P.ind = 1
    P.w("extern __shared__ __align__(16) double smem[];")
    P.w("const int tid = threadIdx.x;")
    P.w("double *TAB = smem + tid;                  // own column of the [slot][thread] head table")
    P.w("double *REC = smem + NSLOT * NTH;          // primitive records [PBS][PRS]")
    P.w("const RcgBasisDev &b = a.basis;")
    P.w("const unsigned tw0 = __ldg(&c_thr[tid][0]), tw1 = __ldg(&c_thr[tid][1]), tw2 = __ldg(&c_thr[tid][2]), tw3 = __ldg(&c_thr[tid][3]);")
    P.w("const double *X0 = smem + (tw1 & 255u), *X1 = smem + ((tw1 >> 8) & 255u);   // columns of a-1x, a-1y (a-1z is lane - 1)")
    P.w("const unsigned tix = tw1 >> 16;            // index among the bra targets, 0xffff: lower component or idle lane")
    P.w("const int64_t q = q0 + blockIdx.x;")
    P.w("double *Hq = H + (int64_t)blockIdx.x * (NT * NC);")
    P.w("const int sh0 = a.quartets[4 * q + a.perm[0]], sh1 = a.quartets[4 * q + a.perm[1]];")
    P.w("const int sh2 = a.quartets[4 * q + a.perm[2]], sh3 = a.quartets[4 * q + a.perm[3]];")
    P.w("const int pa0 = b.prim_off[sh0], Ka = b.prim_off[sh0 + 1] - pa0;")
    P.w("const int pb0 = b.prim_off[sh1], Kb = b.prim_off[sh1 + 1] - pb0;")
    P.w("const int pc0 = b.prim_off[sh2], Kc = b.prim_off[sh2 + 1] - pc0;")
    P.w("const int pd0 = b.prim_off[sh3], Kd = b.prim_off[sh3 + 1] - pd0;")
    P.w("const int K4 = Ka * Kb * Kc * Kd;")

    def slot(pi, cx, cy, m):
        k = cx + cy
        if k == 0:
            return base[0] + m
        return base[k % 3] + slot_of[pi][(cx, cy)] + m

    for pi, Sx in enumerate(passes):
        Sset = set(Sx)
        heads = pass_heads(Sx)
        # accumulators of this pass: targets (cx, cy, cz) with cx in Sx
        acc_of = {}
        for c in TC:
            if c[0] in Sset:
                acc_of[c] = len(acc_of)
        P.w("{   // ---- pass %d: ket x-slabs %s, %d accumulators" % (pi, Sx, len(acc_of)))
        P.ind += 1
        for t in range(len(acc_of)):
            P.w("double acc%d = 0.0;" % t)
        P.w("for (int p0 = 0; p0 < K4; p0 += PBS) {")
        P.ind += 1
        P.w("const int cnt = min(PBS, K4 - p0);")
        P.w("__syncthreads();                        // the previous batch's records are no longer read")
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
        # ---- pure-bra chain [a0|00]^(m): step s keeps the orders its successors need, m = 0..ctop+nst-s
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
                P.w("const double kn_%d = pr[%d + ((tw3 >> %d) & 7u)];" % (s, OFF_HZN, 3 * (s - 1)))
            new = []
            for m in range(ctop + nst - s + 1):
                nm = "x%d_%d" % (s, m)
                P.w("double %s = fma(c2_%d, %s, c1_%d * %s);" % (nm, s, cur[m + 1], s, cur[m]))
                if s >= 2:
                    P.w("%s = fma(kn_%d, fma(-rz, %s, %s), %s);" % (nm, s, prev[m + 1], prev[m], nm))
                new.append(nm)
            prev, cur = cur, new
        bvals = cur[: ctop + 1]
        if ctop >= 1:
            P.w("const double QC0 = pr[%d], QC1 = pr[%d], QC2 = pr[%d];" % (OFF_QC, OFF_QC + 1, OFF_QC + 2))
            P.w("const double WQ0 = pr[%d], WQ1 = pr[%d], WQ2 = pr[%d];" % (OFF_WQ, OFF_WQ + 1, OFF_WQ + 2))
            P.w("const double he = pr[%d], re = pr[%d];" % (OFF_HE, OFF_RE))
            for n in range(2, ctop):
                P.w("const double hen%d = %d.0 * he;" % (n, n))
            if nst:
                P.w("const double hze = pr[%d];" % OFF_HZE)
                P.w("const double ka0 = (double)(int)(tw0 & 15u) * hze, ka1 = (double)(int)((tw0 >> 4) & 15u) * hze, ka2 = (double)(int)(tw0 >> 8) * hze;")
                P.w("__syncthreads();                    // the previous primitive's gathers of the base row are done")
                for m in range(ctop + 1):
                    P.w("TAB[%d] = %s;" % ((base[0] + m) * NTH, bvals[m]))
        hen = {0: None, 1: "he"}

        def emit_target(c, nm):
            if c in acc_of:
                P.w("acc%d += %s;" % (acc_of[c], nm))

        def emit_zchain(cx, cy, head):
            """ket vertices (cx, cy, cz), cz = 1..ctop-cx-cy, in registers; head = names of (cx, cy, 0)^(m), m = 0..D-1."""
            k = cx + cy
            if cx not in Sset or k >= ctop:
                return
            P.w("{   // z-chain of (%d,%d,0)" % (cx, cy))
            P.ind += 1
            prev2, prev1 = None, head
            for cz in range(1, ctop - k + 1):
                kk = k + cz
                c = (cx, cy, cz)
                d = D[kk]
                names = []
                for m in range(d):
                    leaf = kk == ctop and c in acc_of
                    if leaf:
                        nm = "acc%d" % acc_of[c]
                        P.w("%s = fma(QC2, %s, %s);" % (nm, prev1[m], nm))
                    else:
                        nm = "z%d_%d" % (cz, m)
                        P.w("double %s = QC2 * %s;" % (nm, prev1[m]))
                    P.w("%s = fma(WQ2, %s, %s);" % (nm, prev1[m + 1], nm))
                    if cz >= 2:
                        P.w("%s = fma(%s, fma(-re, %s, %s), %s);" % (nm, hen.get(cz - 1, "hen%d" % (cz - 1)), prev2[m + 1], prev2[m], nm))
                    if nst:
                        P.w("%s = fma(ka2, __shfl_up_sync(FULL, %s, 1), %s);" % (nm, prev1[m + 1], nm))
                    names.append(nm)
                if kk >= lc and kk < ctop:
                    emit_target(c, names[0])
                elif kk == ctop and c not in acc_of:
                    pass
                prev2, prev1 = prev1, names
            P.ind -= 1
            P.w("}")

        if (0, 0, 0) in acc_of:
            P.w("acc%d += %s;" % (acc_of[(0, 0, 0)], bvals[0]))
        if ctop >= 1:
            emit_zchain(0, 0, bvals)
        for k in range(1, ctop + 1):
            if not heads[k]:
                continue
            if nst:
                P.w("__syncthreads();                    // head level %d: level %d of every thread is visible" % (k, k - 1))
            d = D[k]
            for (cx, cy) in heads[k]:
                i = 0 if cy == 0 else 1
                pc = (cx - 1, 0) if cy == 0 else (cx, cy - 1)
                n2 = pc[i]
                gc = (cx - 2, 0) if cy == 0 else (cx, cy - 2)
                c = (cx, cy, 0)
                P.w("{   // head (%d,%d,0), axis %s" % (cx, cy, "xy"[i]))
                P.ind += 1
                if k - 1 == 0:
                    pn = bvals
                else:
                    pn = []
                    for m in range(d + 1):
                        P.w("const double p%d = TAB[%d];" % (m, slot(pi, pc[0], pc[1], m) * NTH))
                        pn.append("p%d" % m)
                if n2:
                    if k - 2 == 0:
                        gn = bvals
                    else:
                        gn = []
                        for m in range(d + 1):
                            P.w("const double g%d = TAB[%d];" % (m, slot(pi, gc[0], gc[1], m) * NTH))
                            gn.append("g%d" % m)
                if nst:
                    for m in range(d):
                        P.w("const double x%d = X%d[%d];" % (m, i, slot(pi, pc[0], pc[1], m + 1) * NTH))
                names = []
                for m in range(d):
                    leaf = k == ctop and c in acc_of
                    if leaf:
                        nm = "acc%d" % acc_of[c]
                        P.w("%s = fma(QC%d, %s, %s);" % (nm, i, pn[m], nm))
                    else:
                        nm = "v%d" % m
                        P.w("double %s = QC%d * %s;" % (nm, i, pn[m]))
                    P.w("%s = fma(WQ%d, %s, %s);" % (nm, i, pn[m + 1], nm))
                    if n2:
                        P.w("%s = fma(%s, fma(-re, %s, %s), %s);" % (nm, hen.get(n2, "hen%d" % n2), gn[m + 1], gn[m], nm))
                    if nst:
                        P.w("%s = fma(ka%d, x%d, %s);" % (nm, i, m, nm))
                    if stored(Sx, cx, cy):
                        P.w("TAB[%d] = %s;" % (slot(pi, cx, cy, m) * NTH, nm))
                    names.append(nm)
                if k >= lc and k < ctop:
                    emit_target(c, names[0])
                emit_zchain(cx, cy, names)
                P.ind -= 1
                P.w("}")
        P.ind -= 1
        P.w("}")     # jj
        P.ind -= 1
        P.w("}")     # p0
        P.w("if (tix != 0xffffu) {                   // this pass's columns of H[ket target][bra target]")
        P.ind += 1
        for c, t in sorted(acc_of.items(), key=lambda kv: kv[1]):
            P.w("Hq[%d * NT + tix] = acc%d;" % (tpos[c], t))
        P.ind -= 1
        P.w("}")
        P.ind -= 1
        P.w("}")     # pass
    P.ind = 0
    P.w("}")
    P.w("#undef FULL")
    P.w("}  // namespace h%s" % tag)
    wsq = ws_quartet_doubles(cls)
    P.w("static cudaError_t rcg_launch_heavy_%s(const RcgLaunch &a)" % tag)
    P.w("{")
    P.w("    using namespace h%s;" % tag)
    P.w("    const size_t smem = sizeof(double) * VRR_DOUBLES;")
    P.w("    static RcgOnce once;")
    P.w("    cudaError_t e = rcg_prepare_kernel(once, (const void *)rcg_eri_heavy_%s, smem, nullptr);" % tag)
    P.w("    if (e != cudaSuccess) return e;")
    P.w("    const int64_t chunk = rcg_heavy_chunk(%dLL, a.n);" % wsq)
    P.w("    double *H = a.workspace, *Bh = a.workspace + chunk * (int64_t)(NT * NC);")
    P.w("    for (int64_t q0 = 0; q0 < a.n; q0 += chunk) {")
    P.w("        const int64_t qn = a.n - q0 < chunk ? a.n - q0 : chunk;")
    P.w("        rcg_eri_heavy_%s<<<(unsigned)qn, NTH, smem, a.stream>>>(a, q0, H);" % tag)
    P.w("        if ((e = cudaGetLastError()) != cudaSuccess) return e;")
    P.w("        if ((e = rcg_side_bra(%d, %d, a, q0, qn, H, NC, Bh)) != cudaSuccess) return e;" % (la, lb))
    P.w("        if ((e = rcg_side_ket(%d, %d, a, q0, qn, Bh, NAB)) != cudaSuccess) return e;" % (lc, ld))
    P.w("    }")
    P.w("    return cudaSuccess;")
    P.w("}")
    meta = dict(heavy_threads=NTH, heavy_bra_components=NB, heavy_table_slots=NSLOT, heavy_table_bytes=NSLOT * NTH * 8,
                heavy_passes=passes, heavy_accumulators_per_thread=maxacc, heavy_blocks_per_sm=minb,
                heavy_ws_doubles_per_quartet=wsq)
    return P.text() + "\n", "rcg_launch_heavy_%s" % tag, meta


# ======================================================================================================================
# Slab variant: bra sides with la + lb <= 6 ((fd|, (ff|, (gs|, (gp|, (gd|)
# ======================================================================================================================
SLAB_ACC_CAP = 80       # slab variant: one pass up to 80 accumulators per thread (measured: (ff|ff) 1.52 ms per 20,000 quartets in one pass of 74
                        # against 2.06 ms in two of 37 -- the second pass repeats the pure-bra chain and the x-chain)
SLAB_EXT_MAXCOLS = 10   # at most this many ket targets: Phase 2 in the side kernels (rows of many quartets per block) instead of in the
                        # kernel, where the bra side would run on nC threads only (measured: (gd|ps) 7.5e7 -> 1.3e8 quartets/s)


def slab_layout(nst):
    """threads of the block: the x-SLABS of the bra pyramid (all components with one ax) packed whole into warps, first-fit
    by decreasing size; inside a slab ay ascending, az ascending -- so a-1z is lane - 1 and a-1y is a lane of the same warp.
    Possible while the largest slab ((nst+1)(nst+2)/2 components) fits a warp: nst <= 6."""
    slabs = sorted(range(nst + 1), key=lambda ax: (-(nst - ax + 1) * (nst - ax + 2) // 2, ax))
    warps = []
    for ax in slabs:
        comps = [(ax, ay, az) for ay in range(nst - ax + 1) for az in range(nst - ax - ay + 1)]
        assert len(comps) <= 32
        for w in warps:
            if len(w) + len(comps) <= 32:
                break
        else:
            w = []
            warps.append(w)
        w.extend(comps)
    thr = []
    for w in warps:
        thr.extend(w + [None] * (32 - len(w)))
    return thr


def slab_eligible(cls):
    from .emit_block import side_live
    la, lb, lc, ld = cls
    return la + lb <= 6 and max(side_live(la, lb), side_live(lc, ld)) <= 90 and not options.flag("HEAVY_NO_SLAB")


def emit_class_slab(cls):
    """One kernel per class: x-chain heads (cx,0,0) level by level through shared memory (their cross terms come from
    another slab = possibly another warp), everything else in registers -- y-chains with the cross term [a-1y|c-1y]^(m+1)
    by __shfl_sync from the lane that owns a-1y, z-chains by __shfl_up_sync -- accumulators in registers (passes over ket
    x-slabs above ACC_CAP), H in shared memory, Phase 2 in the kernel (the block tier's depth-first programs)."""
    from .emit_block import emit_side_dfs, side_live
    from .solid import c2s_rows  # noqa: F401
    la, lb, lc, ld = cls
    tag = "%d%d%d%d" % cls
    nst, ctop = la + lb, lc + ld
    L = nst + ctop
    thr = slab_layout(nst)
    NTH = len(thr)
    NB = sum(1 for t in thr if t is not None)
    tid_of = {a: i for i, a in enumerate(thr) if a is not None}
    T = [a for e in range(la, nst + 1) for a in cart_comps(e)]
    tix_of = {a: i for i, a in enumerate(T)}
    nT = len(T)
    TC = [c for f in range(lc, ctop + 1) for c in cart_comps(f)]
    tpos = {c: t for t, c in enumerate(TC)}
    nC = len(TC)
    nAB = (2 * la + 1) * (2 * lb + 1)
    nCD = (2 * lc + 1) * (2 * ld + 1)
    passes = slab_passes(lc, ld, options.geti("SLAB_ACC_CAP", 0) or SLAB_ACC_CAP)
    ext = nC <= (options.geti("SLAB_EXT_MAXCOLS", -1) if options.geti("SLAB_EXT_MAXCOLS", -1) >= 0 else SLAB_EXT_MAXCOLS)
    D = [ctop - k + 1 for k in range(ctop + 1)]
    xslot = [0] * (ctop + 1)            # first slot of the x-chain head (cx,0,0): D[cx] orders each
    for cx in range(1, ctop + 1):
        xslot[cx] = xslot[cx - 1] + D[cx - 1]
    NSLOT = xslot[ctop] + D[ctop]
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
    HST = max(nC, nCD) | 1
    SCN = max((2 * la + 1) * ncart(lb), (2 * lc + 1) * ncart(ld))
    work = NSLOT * NTH + PBS * PRS if ext else max(NSLOT * NTH + PBS * PRS, SCN * NTH)
    smem_doubles = work + (0 if ext else nT * HST)
    maxacc = max(sum(slab_targets(lc, ctop, cx) for cx in Sx) for Sx in passes)
    regs_needed = min(255, max(2 * maxacc + 8 * (ctop + 2) + 90, 0 if ext else 2 * max(side_live(la, lb), side_live(lc, ld)) + 100))
    nth_alloc = (NTH + 127) // 128 * 128
    minb = max(1, min(8, (227 * 1024) // (smem_doubles * 8 + 1024), 65536 // (nth_alloc * ((regs_needed + 7) // 8 * 8))))
    minb = options.geti("SLAB_MINB", 0) or minb

    rows = []
    for t in range(NTH):
        a = thr[t] if thr[t] is not None else (0, 0, 0)
        sx = tid_of[(a[0] - 1, a[1], a[2])] if a[0] > 0 else t
        ysrc = (tid_of[(a[0], a[1] - 1, a[2])] & 31) if a[1] > 0 else (t & 31)
        if a[1] > 0:
            assert tid_of[(a[0], a[1] - 1, a[2])] // 32 == t // 32
        if a[2] > 0:
            assert tid_of[(a[0], a[1], a[2] - 1)] == t - 1 and (t & 31) > 0
        steps = [(ax, n) for ax in range(3) for n in range(a[ax])]
        pad = nst - len(steps)
        sel = [3] * pad + [ax for ax, _ in steps]
        nn = [0] * pad + [n for _, n in steps]
        tix = tix_of[a] if (thr[t] is not None and sum(a) >= la) else 0xffff
        w0 = a[0] | (a[1] << 4) | (a[2] << 8) | (ysrc << 12)
        w1 = sx | (tix << 16)
        w2 = w3 = 0
        for s_ in range(nst):
            w2 |= sel[s_] << (2 * s_)
            w3 |= nn[s_] << (3 * s_)
        rows.append((w0, w1, w2, w3))
    assert NTH <= 256 and 3 * nst <= 32

    P = Prog()
    P.ind = 0
    P.w("// ---- block tier kernel (slab layout) for (%d %d|%d %d): generated by gen/emit_heavy.py" % cls)
    P.w("// bra components (threads) %d of %d, one x-slab per warp segment; x-chain table %d slots/thread; passes over ket x-slabs %s,"
        % (NB, NTH, NSLOT, passes))
    P.w("// at most %d accumulators/thread, blocks/SM %d, shared memory %d B" % (maxacc, minb, smem_doubles * 8))
    P.w('#include "rcg_device.cuh"')
    P.w('#include "rcg_sides.h"')
    P.w("namespace s%s {" % tag)
    P.w("constexpr int NTH = %d, NB = %d, NSLOT = %d, PRS = %d, PBS = %d, NT = %d, NC = %d, NAB = %d, HST = %d, WORK = %d;"
        % (NTH, NB, NSLOT, PRS, PBS, nT, nC, nAB, HST, work))
    P.w("#define FULL 0xffffffffu")
    P.w("__device__ const unsigned c_thr[%d][4] = {     // ax|ay<<4|az<<8|lane of a-1y<<12 ; thread of a-1x | target index<<16 ; path selectors ; path counts" % NTH)
    for r in rows:
        P.w("  {%du,%du,%du,%du}," % r)
    P.w("};")
    if ext:
        P.w("__global__ void __launch_bounds__(NTH, %d) rcg_eri_slab_%s(RcgLaunch a, int64_t q0, double *H)" % (minb, tag))
    else:
        P.w("__global__ void __launch_bounds__(NTH, %d) rcg_eri_slab_%s(RcgLaunch a, int64_t q0)" % (minb, tag))
    P.w("{")
    P.ind = 1
    P.w("extern __shared__ __align__(16) double smem[];")
    P.w("const int tid = threadIdx.x;")
    P.w("double *TAB = smem + tid;                  // own column of the [slot][thread] x-chain table")
    P.w("double *REC = smem + NSLOT * NTH;          // primitive records [PBS][PRS]")
    if not ext:
        P.w("double *Hs = smem + WORK;                  // H [NT][HST], kept across the passes")
    P.w("const RcgBasisDev &b = a.basis;")
    P.w("const unsigned tw0 = __ldg(&c_thr[tid][0]), tw1 = __ldg(&c_thr[tid][1]), tw2 = __ldg(&c_thr[tid][2]), tw3 = __ldg(&c_thr[tid][3]);")
    P.w("const double *X0 = smem + (tw1 & 255u);    // column of a-1x")
    P.w("const int ysrc = (int)((tw0 >> 12) & 31u);  // lane of a-1y (same warp); a-1z is lane - 1")
    P.w("const unsigned tix = tw1 >> 16;")
    if ext:
        P.w("{")
        P.w("const int64_t q = q0 + blockIdx.x;")
        P.w("double *Hq = H + (int64_t)blockIdx.x * (NT * NC);      // H[ket target][bra target] of this quartet, for the side kernels")
    else:      # one block per quartet and no loop over quartets: block-invariant addresses are then formed where they are used instead
        P.w("{")   # of being hoisted, kept across the primitive loop and spilled (12-16 bytes at (ff|ff) with the loop)
        P.w("const int64_t q = q0 + blockIdx.x;")
    P.w("const int sh0 = a.quartets[4 * q + a.perm[0]], sh1 = a.quartets[4 * q + a.perm[1]];")
    P.w("const int sh2 = a.quartets[4 * q + a.perm[2]], sh3 = a.quartets[4 * q + a.perm[3]];")
    P.w("const int pa0 = b.prim_off[sh0], Ka = b.prim_off[sh0 + 1] - pa0;")
    P.w("const int pb0 = b.prim_off[sh1], Kb = b.prim_off[sh1 + 1] - pb0;")
    P.w("const int pc0 = b.prim_off[sh2], Kc = b.prim_off[sh2 + 1] - pc0;")
    P.w("const int pd0 = b.prim_off[sh3], Kd = b.prim_off[sh3 + 1] - pd0;")
    P.w("const int K4 = Ka * Kb * Kc * Kd;")
    hen = {0: None, 1: "he"}
    for pi, Sx in enumerate(passes):
        Sset = set(Sx)
        mx = max(Sx)
        acc_of = {}
        for c in TC:
            if c[0] in Sset:
                acc_of[c] = len(acc_of)
        P.w("{   // ---- pass %d: ket x-slabs %s, %d accumulators" % (pi, Sx, len(acc_of)))
        P.ind += 1
        for t in range(len(acc_of)):
            P.w("double acc%d = 0.0;" % t)
        P.w("for (int p0 = 0; p0 < K4; p0 += PBS) {")
        P.ind += 1
        P.w("const int cnt = min(PBS, K4 - p0);")
        P.w("__syncthreads();                        // the previous batch's records / the previous quartet's Phase-2 scratch are no longer read")
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
                P.w("const double kn_%d = pr[%d + ((tw3 >> %d) & 7u)];" % (s, OFF_HZN, 3 * (s - 1)))
            new = []
            for m in range(ctop + nst - s + 1):
                nm = "x%d_%d" % (s, m)
                P.w("double %s = fma(c2_%d, %s, c1_%d * %s);" % (nm, s, cur[m + 1], s, cur[m]))
                if s >= 2:
                    P.w("%s = fma(kn_%d, fma(-rz, %s, %s), %s);" % (nm, s, prev[m + 1], prev[m], nm))
                new.append(nm)
            prev, cur = cur, new
        bvals = cur[: ctop + 1]
        if ctop >= 1:
            P.w("const double QC0 = pr[%d], QC1 = pr[%d], QC2 = pr[%d];" % (OFF_QC, OFF_QC + 1, OFF_QC + 2))
            P.w("const double WQ0 = pr[%d], WQ1 = pr[%d], WQ2 = pr[%d];" % (OFF_WQ, OFF_WQ + 1, OFF_WQ + 2))
            P.w("const double he = pr[%d], re = pr[%d];" % (OFF_HE, OFF_RE))
            for n in range(2, ctop):
                P.w("const double hen%d = %d.0 * he;" % (n, n))
            P.w("const double hze = pr[%d];" % OFF_HZE)
            P.w("const double ka0 = (double)(int)(tw0 & 15u) * hze, ka1 = (double)(int)((tw0 >> 4) & 15u) * hze, ka2 = (double)(int)((tw0 >> 8) & 15u) * hze;")

        def emit_target(c, nm):
            if c in acc_of:
                P.w("acc%d += %s;" % (acc_of[c], nm))

        def vertex(nm, leafacc, i, p1, p1u, g, gu, n2, cross):
            """one Eq. (2) ket step along axis i: nm (or the accumulator leafacc) from parent p1^(m), p1^(m+1), grandparent, cross term."""
            if leafacc is not None:
                P.w("%s = fma(QC%d, %s, %s);" % (leafacc, i, p1, leafacc))
                nm = leafacc
            else:
                P.w("double %s = QC%d * %s;" % (nm, i, p1))
            P.w("%s = fma(WQ%d, %s, %s);" % (nm, i, p1u, nm))
            if n2:
                P.w("%s = fma(%s, fma(-re, %s, %s), %s);" % (nm, hen.get(n2, "hen%d" % n2), gu, g, nm))
            if cross is not None:
                P.w("%s = fma(ka%d, %s, %s);" % (nm, i, cross, nm))
            return nm

        def emit_zchain(cx, cy, head, pfx):
            k = cx + cy
            if k >= ctop:
                return
            P.w("{   // z-chain of (%d,%d,0)" % (cx, cy))
            P.ind += 1
            prev2, prev1 = None, head
            for cz in range(1, ctop - k + 1):
                kk = k + cz
                c = (cx, cy, cz)
                names = []
                for m in range(D[kk]):
                    leaf = "acc%d" % acc_of[c] if (kk == ctop and c in acc_of) else None
                    cross = "__shfl_up_sync(FULL, %s, 1)" % prev1[m + 1] if nst else None
                    names.append(vertex("%sz%d_%d" % (pfx, cz, m), leaf, 2, prev1[m], prev1[m + 1],
                                        prev2[m] if cz >= 2 else None, prev2[m + 1] if cz >= 2 else None, cz - 1, cross))
                if lc <= kk < ctop:
                    emit_target(c, names[0])
                prev2, prev1 = prev1, names
            P.ind -= 1
            P.w("}")

        # ---- x-chain heads (cx,0,0), cx = 1..mx, level by level through shared memory; slab cx - 1 (y- and z-chains, registers and
        # shuffles only) is worked off right after head cx has been published, so that the barrier of head cx + 1 finds the other
        # warps' values ready and only two heads (not all of them: 28 doubles at ctop = 6) are live at a time
        def emit_slab(cx, head):
            c0 = (cx, 0, 0)
            P.w("{   // slab cx = %d" % cx)
            P.ind += 1
            if cx >= lc and (cx < ctop or ctop == 0):      # (a top-level head is a leaf: folded into its accumulator above)
                emit_target(c0, head[0])
            emit_zchain(cx, 0, head, "a")
            y2, y1 = None, head
            for cy in range(1, ctop - cx + 1):
                k = cx + cy
                c = (cx, cy, 0)
                names = []
                P.w("{")
                P.ind += 1
                for m in range(D[k]):
                    leaf = "acc%d" % acc_of[c] if (k == ctop and c in acc_of) else None
                    cross = "__shfl_sync(FULL, %s, ysrc)" % y1[m + 1] if nst else None
                    names.append(vertex("y%d_%d" % (cy, m), leaf, 1, y1[m], y1[m + 1],
                                        y2[m] if cy >= 2 else None, y2[m + 1] if cy >= 2 else None, cy - 1, cross))
                if lc <= k < ctop:
                    emit_target(c, names[0])
                emit_zchain(cx, cy, names, "b")
                y2, y1 = y1, names
            for cy in range(1, ctop - cx + 1):
                P.ind -= 1
                P.w("}")
            P.ind -= 1
            P.w("}")

        interleave = not options.flag("SLAB_NO_INTERLEAVE")
        if nst and ctop >= 1 and mx >= 1:
            P.w("__syncthreads();                    // the previous primitive's gathers of the x-chain table are done")
            for m in range(1, ctop + 1):
                P.w("TAB[%d] = %s;" % ((xslot[0] + m) * NTH, bvals[m]))
        xh = {0: bvals}
        for cx in range(1, mx + 1):
            if nst:
                P.w("__syncthreads();                    // x-chain head %d: head %d of every thread is visible" % (cx, cx - 1))
            names = []
            for m in range(D[cx]):
                cross = None
                if nst:
                    P.w("const double xx%d_%d = X0[%d];" % (cx, m, (xslot[cx - 1] + m + 1) * NTH))
                    cross = "xx%d_%d" % (cx, m)
                leaf = "acc%d" % acc_of[(cx, 0, 0)] if (cx == ctop and (cx, 0, 0) in acc_of) else None
                names.append(vertex("xh%d_%d" % (cx, m), leaf, 0, xh[cx - 1][m], xh[cx - 1][m + 1],
                                    xh[cx - 2][m] if cx >= 2 else None, xh[cx - 2][m + 1] if cx >= 2 else None, cx - 1, cross))
                if nst and cx < mx and m >= 1:
                    P.w("TAB[%d] = %s;" % ((xslot[cx] + m) * NTH, names[-1]))
            xh[cx] = names
            if interleave and (cx - 1) in Sset:
                emit_slab(cx - 1, xh[cx - 1])
        for cx in Sx:
            if not interleave or cx == mx:
                emit_slab(cx, xh[cx])
        P.ind -= 1
        P.w("}")     # jj
        P.ind -= 1
        P.w("}")     # p0
        P.w("if (tix != 0xffffu) {                   // this pass's columns of H")
        P.ind += 1
        if ext:
            for c, t in sorted(acc_of.items(), key=lambda kv: kv[1]):
                P.w("Hq[%d * NT + tix] = acc%d;" % (tpos[c], t))
        else:
            P.w("double *h = Hs + tix * HST;")
            for c, t in sorted(acc_of.items(), key=lambda kv: kv[1]):
                P.w("h[%d] = acc%d;" % (tpos[c], t))
        P.ind -= 1
        P.w("}")
        P.ind -= 1
        P.w("}")     # pass
    if not ext:
        # ---------------- Phase 2 (the block tier's depth-first programs; emit_block.emit_side_dfs)
        P.w("__syncthreads();                            // H complete; the table region becomes the scratch columns [SCN][NTH]")
        P.w("double *SC = smem + tid;")
        P.w("for (int col = tid; col < NC; col += NTH) {     // bra HRR + Ta, Tb on ket column col")
        P.ind += 1
        P.w("const double AB0 = b.centers[3 * sh0] - b.centers[3 * sh1], AB1 = b.centers[3 * sh0 + 1] - b.centers[3 * sh1 + 1], AB2 = b.centers[3 * sh0 + 2] - b.centers[3 * sh1 + 2];")
        P.w("double *hc = Hs + col;")
        emit_side_dfs(P, la, lb, lambda k: "hc[%d]" % (k * HST), ["AB0", "AB1", "AB2"],
                      lambda i: "SC[%d]" % (i * NTH), lambda r, e: P.w("hc[%d] = %s;" % (r * HST, e)), "h")
        P.ind -= 1
        P.w("}")
        P.w("__syncthreads();")
        P.w("for (int row = tid; row < NAB; row += NTH) {    // ket HRR + Tc, Td on spherical bra row")
        P.ind += 1
        P.w("const double CD0 = b.centers[3 * sh2] - b.centers[3 * sh3], CD1 = b.centers[3 * sh2 + 1] - b.centers[3 * sh3 + 1], CD2 = b.centers[3 * sh2 + 2] - b.centers[3 * sh3 + 2];")
        P.w("double *hr = Hs + row * HST;")
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
        P.w("    const double v = Hs[o * HST + r];")
        P.w("    if (canon) out[e] = v;")
        P.w("    else {")
        P.w("        const int id = r %% %d, ic = r / %d, ib = o %% %d, ia = o / %d;" % (nsd, nsd, nsb, nsb))
        P.w("        out[ia * a.ostride[0] + ib * a.ostride[1] + ic * a.ostride[2] + id * a.ostride[3]] = v;")
        P.w("    }")
        P.w("}")
    P.w("}   // quartet loop")
    P.ind = 0
    P.w("}")
    P.w("#undef FULL")
    P.w("}  // namespace s%s" % tag)
    P.w("static cudaError_t rcg_launch_slab_%s(const RcgLaunch &a)" % tag)
    P.w("{")
    P.w("    using namespace s%s;" % tag)
    P.w("    const size_t smem = sizeof(double) * %d;" % smem_doubles)
    P.w("    static RcgOnce once;")
    P.w("    cudaError_t e = rcg_prepare_kernel(once, (const void *)rcg_eri_slab_%s, smem, nullptr);" % tag)
    P.w("    if (e != cudaSuccess) return e;")
    if ext:
        wsq = ws_quartet_doubles(cls)
        P.w("    const int64_t chunk = rcg_heavy_chunk(%dLL, a.n);" % wsq)
        P.w("    double *H = a.workspace, *Bh = a.workspace + chunk * (int64_t)(NT * NC);")
        P.w("    for (int64_t q0 = 0; q0 < a.n; q0 += chunk) {")
        P.w("        const int64_t qn = a.n - q0 < chunk ? a.n - q0 : chunk;")
        P.w("        rcg_eri_slab_%s<<<(unsigned)qn, NTH, smem, a.stream>>>(a, q0, H);" % tag)
        P.w("        if ((e = cudaGetLastError()) != cudaSuccess) return e;")
        P.w("        if ((e = rcg_side_bra(%d, %d, a, q0, qn, H, NC, Bh)) != cudaSuccess) return e;" % (la, lb))
        P.w("        if ((e = rcg_side_ket(%d, %d, a, q0, qn, Bh, NAB)) != cudaSuccess) return e;" % (lc, ld))
        P.w("    }")
        P.w("    return cudaSuccess;")
    else:
        P.w("    for (int64_t q0 = 0; q0 < a.n; q0 += (1ll << 30)) {             // one block per quartet: the hardware balances uneven K4")
        P.w("        const int64_t blocks = a.n - q0 < (1ll << 30) ? a.n - q0 : (1ll << 30);")
        P.w("        rcg_eri_slab_%s<<<(unsigned)blocks, NTH, smem, a.stream>>>(a, q0);" % tag)
        P.w("        if ((e = cudaGetLastError()) != cudaSuccess) return e;")
        P.w("    }")
        P.w("    return cudaSuccess;")
    P.w("}")
    meta = dict(slab_threads=NTH, slab_bra_components=NB, slab_table_slots=NSLOT, slab_smem_bytes=smem_doubles * 8,
                slab_passes=passes, slab_accumulators_per_thread=maxacc, slab_blocks_per_sm=minb, slab_external_phase2=bool(ext))
    if ext:
        meta["heavy_ws_doubles_per_quartet"] = ws_quartet_doubles(cls)
    return P.text() + "\n", "rcg_launch_slab_%s" % tag, meta
