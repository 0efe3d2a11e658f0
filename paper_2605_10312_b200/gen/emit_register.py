"""Emit the register tier (RCG_TIER_REGISTER) kernel of one class: one THREAD per shell quartet.

This is the paper's Tier 1 (Alg. 2 at :269-283) as it stands: the four primitive
loops run inside the thread, every VRR vertex of Eq. (2) is a register, the graph is
emitted fully unrolled in a liveness-aware topological order (the DSA greedy order of Eq. (7),
PAPER.md:168-177, or the post-order, whichever has the lower PeakLive of Eq. (4)), the contracted
targets H (Alg. 2 line 7) stay in registers across the loops, and Phase 2 (HRR Eq. (3) + stepwise c2s,
Eqs. (11)-(16)) runs on registers once after the loops.  On sm_100a it pays only for the lightest
classes (at most 56 Cartesian targets): there a warp per quartet leaves most lanes idle, while 32
quartets per warp use all of them -- provided the quartets of a warp have similar primitive counts
(threads loop to their own K4, a warp to its largest), which the launcher checks on the device
(csrc/pack_stats.cu with groups of 32) before it lets this kernel, and not the warp-tier one, do the
work.
"""
import os

from . import options
from .graph import VrrGraph, hrr_c2s_program, c2s_pair_program, peak_live, dsa_order
from .solid import cart_comps
from .emit_warp import Prog

REG_MAX_TARGETS = 100         # up to (pp|pp): measured with the forced-tier ablation (profiles/r2_ablation.md), 200,000 quartets, K4 = 16: the thread
                              # per quartet runs (pp|pp) 1.8x faster than the packed warp kernel (528 spill bytes in the DSA order); (dp|dp) and up lose
REG_H_REGS = 36               # accumulators H kept in registers; the ket columns beyond live in the thread's own shared-memory column
                              # ([slot][thread], conflict-free): explicit staging instead of the 300-1,600 spill bytes ptxas would emit
REG_EXCLUDED = set()
# classes above 100 targets whose thread-per-quartet kernel still compiles to 0 spill bytes with EVERY accumulator in shared memory (1.3-1.8x their
# warp kernels on K4 = 1 lists); (fd|ps), (fp|ds), (dd|ds) keep 120-360 spill bytes that way and stay in the warp tier
REG_EXTRA = {(2, 1, 1, 1), (3, 0, 2, 1)}
REG_SPLIT_EXCLUDED = {(3, 0, 2, 1)}      # its primitive-split and Fock variants keep 4 spill bytes: not generated (warp kernels take those lists)
REG_FOCK_EXCLUDED = {(3, 0, 2, 1)}    # their digestion epilogue would spill (236 / 8 bytes): rcg_fock_batch takes the L2-chunk path there
REG_ORDER_OF = {(2, 1, 2, 0): "dsa", (2, 1, 1, 1): "dsa"}     # (dp|ds): the DSA order of Eq. (7) compiles to 0 spill bytes, the post-order (lower PeakLive) to 8 + 12  # 96 targets, but 20 spill bytes remain even with every accumulator in shared memory: stays in the warp tier
REG_H_COLS = {(2, 2, 1, 0): 0, (3, 0, 3, 0): 1, (2, 1, 2, 0): 0}     # register-resident ket columns where the default still left spill bytes (ptxas)
REG_MIN_QUARTETS_HEAVY = 32768   # classes above 56 targets (shared-memory staged accumulators): cfg1 (10,000 (pp|pp) quartets, K4 = 81) runs 0.143 ms in the
                              # packed warp kernel against 0.170 ms with a thread per quartet; at 200,000 quartets the thread per quartet is 1.2-1.8x faster
REG_STAGE_MIN = 15         # blocks of at least this many doubles are stored through shared memory (staged stores); measured on the
REG_STAGE_DOUBLES = 16     # cfg5 pass: 1.04-1.40x per class with 16 doubles per thread and staging pass (two classes: 32), blocks of 9 lose
REG_STAGE_DOUBLES_OF = {(1, 1, 1, 1): 32, (3, 0, 1, 1): 32}
REG_STAGE_OFF = {(2, 1, 1, 1), (3, 0, 2, 1)}      # (dp|pp): every accumulator already in shared memory (144 per thread), staging on top loses 10%; (fs|dp) would spill 4 bytes
REG_SPLIT = 8                 # lanes per quartet of the primitive-split kernel
REG_MIN_QUARTETS = 8192       # measured on the B200 (K = 1 and 2 primitives per shell): from 8,192 quartets up a thread per quartet is
                              # never slower than a warp per quartet (1.3-6x faster at 16-32 k); below, both sit on the launch floor


def eligible(cls):
    la, lb, lc, ld = cls
    g = VrrGraph(la, lb, lc, ld)
    return (len(g.target_a) * len(g.target_c) <= options.geti("REG_MAX_TARGETS", REG_MAX_TARGETS) or cls in REG_EXTRA) and cls not in REG_EXCLUDED


def emit_lin_names(P, prog, inputs, prefix, X):
    """straight-line LinProgram on named registers; returns the output expressions."""
    name = {k: inputs[k] for k in range(prog.nin)}
    for (dst, src, coef, init) in prog.ops:
        if coef[0] == "one":
            cs = None
        elif coef[0] == "x":
            cs = X[coef[1]]
        elif coef[1] == 1.0:
            cs = None
        else:
            cs = repr(float(coef[1]))
        s = name[src]
        if init:
            d = "%s%d" % (prefix, dst)
            name[dst] = d
            P.w("double %s = %s;" % (d, s if cs is None else "%s * %s" % (cs, s)))
        else:
            d = name[dst]
            P.w("%s = %s;" % (d, "%s + %s" % (d, s) if cs is None else "fma(%s, %s, %s)" % (cs, s, d)))
    return [name[o] for o in prog.outputs]


def emit_class(cls):
    """the ERI kernel, the Fock kernel (same VRR and Phase 2, digestion in the epilogue) and their launchers."""
    t1, sym, meta = _emit_kernel(cls, False)
    t3, syms = "", None
    if cls not in REG_SPLIT_EXCLUDED:
        t3, syms, _ = _emit_kernel(cls, False, split=True)
        meta["reg_split_launcher"] = syms
    if cls in REG_FOCK_EXCLUDED:
        return t1 + t3, sym, meta
    t2, symf, _ = _emit_kernel(cls, True)
    meta["reg_fock_launcher"] = symf
    return t1 + t3 + t2, sym, meta


def _emit_kernel(cls, fock, split=False):
    """split: REG_SPLIT lanes per quartet, each taking every REG_SPLIT-th primitive quartet (primitive-level parallelism
    for short lists of deeply contracted shells, e.g. cfg1: 10,000 (pp|pp) quartets with K4 = 81); the contracted targets are summed
    over the lanes by shuffles, Phase 2 runs redundantly in every lane and each lane stores its share of the outputs."""
    la, lb, lc, ld = cls
    tag = "%d%d%d%d" % cls
    kname = "rcg_fock_reg_%s" % tag if fock else ("rcg_eri_regsplit_%s" % tag if split else "rcg_eri_reg_%s" % tag)
    ns = "rf%s" % tag if fock else ("rs%s" % tag if split else "r%s" % tag)
    S = REG_SPLIT
    # ablation switches (paper_2605_10312_b200/ablation.py; the defaults are the product): RCG_REG_AXIS=alg1 builds the graph by the
    # literal Alg. 1 (reading R-AXIS), RCG_REG_ORDER=dsa|post forces the emission order
    g = VrrGraph(la, lb, lc, ld, axis_rule=options.get("REG_AXIS", "side"))
    L = la + lb + lc + ld
    order_post = list(g.order)
    order_dsa = dsa_order(g)
    pl_post, pl_dsa = peak_live(g, order_post), peak_live(g, order_dsa)
    order = order_dsa if pl_dsa < pl_post else order_post
    forced = options.get("REG_ORDER", "") or REG_ORDER_OF.get(cls, "")
    if forced:
        order = order_dsa if forced == "dsa" else order_post
    TA, TCc = g.target_a, g.target_c
    nT, nC = len(TA), len(TCc)
    tindex = {(a, c): ia * nC + ic for ia, a in enumerate(TA) for ic, c in enumerate(TCc)}
    fused = options.get("SPH_FUSION", "1") != "0"      # ablation: bra pair Cartesian through the ket side, transformed last
    bra = hrr_c2s_program(la, lb, c2s=fused)
    ket = hrr_c2s_program(lc, ld)
    late = None if fused else c2s_pair_program(la, lb)
    nAB = (2 * la + 1) * (2 * lb + 1)
    nCD = (2 * lc + 1) * (2 * ld + 1)
    nsb, nsc, nsd = 2 * lb + 1, 2 * lc + 1, 2 * ld + 1
    # staged stores: a thread's block is contiguous in the output, so one store instruction of a warp touches 32 sectors (8 of 32 bytes
    # used): the kernels with large blocks wait on the load/store queue for half their time on K4 = 1 lists.  The warp parks STAGE_ROWS
    # bra rows of its 32 blocks in shared memory and copies them out together, 32 contiguous segments per pass
    stage = (not fock) and (not split) and options.geti(
        "REG_STAGE", 1 if nAB * nCD >= options.geti("REG_STAGE_MIN", REG_STAGE_MIN) and cls not in REG_STAGE_OFF else 0) == 1
    srows = max(1, min(nAB, options.geti("REG_STAGE_DOUBLES", REG_STAGE_DOUBLES_OF.get(cls, REG_STAGE_DOUBLES)) // nCD))
    SC = srows * nCD                   # doubles per thread and pass
    SCP = SC | 1                       # odd row stride: conflict-free column stores
    P = Prog()
    P.ind = 0
    P.w("// ---- register tier kernel for (%d %d|%d %d): generated by gen/emit_register.py" % cls)
    P.w("// %d VRR vertices per primitive quartet, order = %s (PeakLive post-order %d, DSA %d), %d accumulators"
        % (g.num_nodes(), "DSA" if order is order_dsa else "post-order", pl_post, pl_dsa, nT * nC))
    P.w("namespace %s {" % ns)
    minb = options.geti("SPLIT_MINB", 1) if split else 1
    P.w("__global__ void __launch_bounds__(128, %d) %s(RcgLaunch a)" % (minb, kname))
    P.w("{")
    P.ind = 1
    P.w("if (a.stat_reg != nullptr && !(a.stat_reg[0] * 10ull <= a.stat_reg[1] * 13ull)) return;   // lists with uneven K4 go to the warp tier")
    if fock:      # no thread leaves early: a thread past the end recomputes the last quartet with weight 0, so the full-warp shuffles below are legal
        P.w("const int64_t q_ = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;")
        P.w("const bool live = q_ < a.n;")
        P.w("const int64_t q = live ? q_ : a.n - 1;")
    elif split:   # no thread leaves early either (full-warp shuffles in the reduction)
        P.w("const int64_t t_ = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;")
        P.w("const int sl = (int)(t_ %% %d);              // this lane's slice of the primitive quartets" % S)
        P.w("const bool live = t_ / %d < a.n;" % S)
        P.w("const int64_t q = live ? t_ / %d : a.n - 1;" % S)
    elif stage:   # no thread leaves early: the warp copies its 32 blocks out together
        P.w("const int64_t q_ = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;")
        P.w("const int64_t q = q_ < a.n ? q_ : a.n - 1;")
    else:
        P.w("const int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;")
        P.w("if (q >= a.n) return;")
    P.w("const RcgBasisDev &b = a.basis;")
    P.w("const int sh0 = a.quartets[4 * q + a.perm[0]], sh1 = a.quartets[4 * q + a.perm[1]];")
    P.w("const int sh2 = a.quartets[4 * q + a.perm[2]], sh3 = a.quartets[4 * q + a.perm[3]];")
    P.w("double RA[3], RB[3], RC[3], RD[3];")
    P.w("#pragma unroll")
    P.w("for (int t = 0; t < 3; ++t) { RA[t] = b.centers[3 * sh0 + t]; RB[t] = b.centers[3 * sh1 + t]; RC[t] = b.centers[3 * sh2 + t]; RD[t] = b.centers[3 * sh3 + t]; }")
    P.w("const int pa0 = b.prim_off[sh0], pa1 = b.prim_off[sh0 + 1], pb0 = b.prim_off[sh1], pb1 = b.prim_off[sh1 + 1];")
    P.w("const int pc0 = b.prim_off[sh2], pc1 = b.prim_off[sh2 + 1], pd0 = b.prim_off[sh3], pd1 = b.prim_off[sh3 + 1];")
    # ket columns c < creg keep their nT accumulators in registers, the rest sit in shared memory (explicit, instead of spills)
    creg = nC if nT * nC <= 56 else REG_H_COLS.get(cls, max(1, REG_H_REGS // nT))
    if nT * nC > 100:          # the VRR frontier alone fills the registers there: every accumulator in shared memory
        creg = options.geti("REG_BIG_HCOLS", 0)
    if split and options.geti("SPLIT_HREGS", -1) >= 0:
        creg = min(nC, options.geti("SPLIT_HREGS", -1) // nT)
    nsm_slots = (nC - creg) * nT

    def Hx(t):
        ia, c = divmod(t, nC)
        return "H%d" % t if c < creg else "hsm[%d * RBS]" % ((c - creg) * nT + ia)

    if nsm_slots or stage:
        P.w("extern __shared__ double hs[];")
        P.w("const int RBS = blockDim.x;")
    if stage:
        P.w("double *ost = hs + %d * RBS + (threadIdx.x & ~31) * %d;      // this warp's staging rows [32][%d]" % (nsm_slots, SCP, SCP))
    if nsm_slots:
        P.w("double *hsm = hs + threadIdx.x;")
        P.w("#pragma unroll 1")
        P.w("for (int t = 0; t < %d; ++t) hsm[t * RBS] = 0.0;" % nsm_slots)
    for t in range(nT * nC):
        if (t % nC) < creg:
            P.w("double H%d = 0.0;" % t)
    if split:
        P.w("const int Kb_ = pb1 - pb0, Kc_ = pc1 - pc0, Kd_ = pd1 - pd0, K4_ = (pa1 - pa0) * Kb_ * Kc_ * Kd_;")
        P.w("const float rKd = __fdividef(1.0f, (float)Kd_), rKc = __fdividef(1.0f, (float)Kc_), rKb = __fdividef(1.0f, (float)Kb_);")
        P.w("for (int pp = sl; pp < K4_; pp += %d) {" % S)
        P.w("    int il_, ik_, ij_; int pr_ = rcg_divmod(pp, Kd_, rKd, il_); pr_ = rcg_divmod(pr_, Kc_, rKc, ik_); const int ii_ = rcg_divmod(pr_, Kb_, rKb, ij_);")
        P.w("    const int i = pa0 + ii_, j = pb0 + ij_, k = pc0 + ik_, l = pd0 + il_;")
    else:
        P.w("for (int i = pa0; i < pa1; ++i)")
        P.w("for (int j = pb0; j < pb1; ++j)")
        P.w("for (int k = pc0; k < pc1; ++k)")
        P.w("for (int l = pd0; l < pd1; ++l) {")
    P.ind += 1
    P.w("RcgPrim p;")
    P.w("rcg_prim_setup(p, RA, RB, RC, RD, b.exps[i], b.exps[j], b.exps[k], b.exps[l],")
    P.w("               b.coefs[i] * b.coefs[j] * b.coefs[k] * b.coefs[l]);")
    P.w("double F[%d];" % (L + 1))
    P.w("rcg_boys<%d>(%d, p.T, p.pref, b.boys, F);" % (L, L))
    hen = set()
    hzn = set()
    hxn = set()
    for key in order:
        n = g.nodes[key]
        if n.side is None:
            continue
        if n.p3 is not None:
            (hen if n.side == "ket" else hzn).add(n.n2)
        if n.p5 is not None:
            hxn.add(n.ncross)
    for v in sorted(hen):
        P.w("const double hen%d = %d.0 * p.he;" % (v, v))
    for v in sorted(hzn):
        P.w("const double hzn%d = %d.0 * p.hz;" % (v, v))
    for v in sorted(hxn):
        P.w("const double hxn%d = %d.0 * p.hze;" % (v, v))
    vid = {}

    def nm(key):
        n = g.nodes[key]
        if n.side is None:
            return "F[%d]" % n.m
        return "v%d" % vid[key]

    for key in order:
        n = g.nodes[key]
        if n.side is None:
            if (n.a, n.c) in tindex and n.m == 0:
                P.w("%s += F[0];" % Hx(tindex[(n.a, n.c)]))
            continue
        vid[key] = len(vid)
        i = n.axis
        c1, c2 = ("p.QC[%d]" % i, "p.WQ[%d]" % i) if n.side == "ket" else ("p.PA[%d]" % i, "p.WP[%d]" % i)
        r3 = "p.re" if n.side == "ket" else "p.rz"
        h3 = ("hen%d" if n.side == "ket" else "hzn%d") % n.n2
        v = "v%d" % vid[key]
        P.w("double %s = %s * %s;" % (v, c1, nm(n.p1)))
        P.w("%s = fma(%s, %s, %s);" % (v, c2, nm(n.p2), v))
        if n.p3 is not None:
            P.w("%s = fma(%s, fma(-%s, %s, %s), %s);" % (v, h3, r3, nm(n.p4), nm(n.p3), v))
        if n.p5 is not None:
            P.w("%s = fma(hxn%d, %s, %s);" % (v, n.ncross, nm(n.p5), v))
        if n.m == 0 and (n.a, n.c) in tindex:
            P.w("%s += %s;" % (Hx(tindex[(n.a, n.c)]), v))
    P.ind -= 1
    P.w("}")
    if split:     # contraction over the lanes of the quartet (Alg. 2 line 7): butterfly sums, every lane ends with the full H
        P.w("__syncwarp();")
        for t in range(nT * nC):
            hx = Hx(t)
            if hx.startswith("H"):
                for off in [o for o in (16, 8, 4, 2, 1) if o < S]:
                    P.w("%s += __shfl_xor_sync(0xffffffffu, %s, %d);" % (hx, hx, off))
            else:
                P.w("{ double v_ = %s;" % hx)
                for off in [o for o in (16, 8, 4, 2, 1) if o < S]:
                    P.w("  v_ += __shfl_xor_sync(0xffffffffu, v_, %d);" % off)
                P.w("  %s = v_; }" % hx)
    # ---- Phase 2 on registers: bra HRR + Ta,Tb per ket column, then ket HRR + Tc,Td per spherical bra row
    P.w("const double AB0 = RA[0] - RB[0], AB1 = RA[1] - RB[1], AB2 = RA[2] - RB[2];")
    P.w("const double CD0 = RC[0] - RD[0], CD1 = RC[1] - RD[1], CD2 = RC[2] - RD[2];")
    half = []        # half[c][o]
    for c in range(nC):
        if c >= creg:
            for ia in range(nT):
                P.w("const double hc%d_%d = %s;" % (c, ia, Hx(ia * nC + c)))
            ins = ["hc%d_%d" % (c, ia) for ia in range(nT)]
        else:
            ins = ["H%d" % (ia * nC + c) for ia in range(nT)]
        outs = emit_lin_names(P, bra, ins, "b%d_" % c, ["AB0", "AB1", "AB2"])
        if c >= creg and len(outs) <= nT:        # a shared-memory column: its half-transformed values go back into its own slots
            for o, e in enumerate(outs):
                P.w("%s = %s;" % (Hx(o * nC + c), e))
            outs = [Hx(o * nC + c) for o in range(len(outs))]
        half.append(outs)
    nsa = 2 * la + 1
    if fock:
        # J/K digestion in the thread (PAPER.md:259 "inline atomicAdd scatter", :291 scale factors; Alg. 2 line 10): the block never
        # leaves the registers.  Jt_ab += 2w sum_cd D_cd I, Jt_cd += 2w sum_ab D_ab I, Kt_ac += w sum_bd D_bd I, Kt_ad, Kt_bc, Kt_bd alike
        # (csrc/jk_digest.cu has the derivation); consecutive quartets of a pass share the bra pair, so Jt_ab is summed over the
        # warp by shuffles first when all 32 lanes hold the same (a, b)
        P.w("const int oa = a.bf_off[sh0], ob = a.bf_off[sh1], oc = a.bf_off[sh2], od = a.bf_off[sh3];")
        P.w("double wq = live ? 1.0 : 0.0;")
        P.w("if (sh0 == sh1) wq *= 0.5;")
        P.w("if (sh2 == sh3) wq *= 0.5;")
        P.w("if (sh0 == sh2 && sh1 == sh3) wq *= 0.5;")
        P.w("const double *Dm = a.D;")
        P.w("const int64_t nbf = a.nbf;")
        P.w("__syncwarp();                           // the warp is whole again after the primitive loops (every thread reaches this point)")
        P.w("const int sh0_l0 = __shfl_sync(0xffffffffu, sh0, 0), sh1_l0 = __shfl_sync(0xffffffffu, sh1, 0);   // both shuffles by EVERY lane (no short-circuit)")
        P.w("const bool same_ab = __all_sync(0xffffffffu, sh0 == sh0_l0 && sh1 == sh1_l0);")
        for r in range(nCD):
            ic, idd = divmod(r, nsd)
            P.w("const double dcd%d = __ldg(Dm + (oc + %d) * nbf + od + %d);" % (r, ic, idd))
            P.w("double jcd%d = 0.0;" % r)
        for ic in range(nsc):         # Kt_ac, Kt_ad: one row (fixed ia) at a time -- complete after the nsb rows (ia, .) of the block, flushed then
            P.w("double kac%d = 0.0;" % ic)
        for idd in range(nsd):
            P.w("double kad%d = 0.0;" % idd)
        for ib in range(nsb):
            for ic in range(nsc):
                P.w("double kbc%d_%d = 0.0;" % (ib, ic))
            for idd in range(nsd):
                P.w("double kbd%d_%d = 0.0;" % (ib, idd))
    else:
        P.w("double *out = a.out + q * a.out_stride;")
        P.w("const bool canon = a.ostride[3] == 1 && a.ostride[2] == %d && a.ostride[1] == %d && a.ostride[0] == %d;"
            % (nsd, nsd * nsc, nsd * nsc * nsb))
    if late is not None:      # all Cartesian bra rows through the ket side first, then Ta (x) Tb per output column
        nABc = len(half[0])
        kout = [emit_lin_names(P, ket, [half[c][o] for c in range(nC)], "kc%d_" % o, ["CD0", "CD1", "CD2"]) for o in range(nABc)]
        fin = [emit_lin_names(P, late, [kout[o][r] for o in range(nABc)], "t%d_" % r, ["0", "0", "0"]) for r in range(nCD)]
    for o in range(nAB):
        P.w("{")
        P.ind += 1
        if late is not None:
            outs = [fin[r][o] for r in range(nCD)]
        else:
            kin = []
            for c in range(nC):
                if c >= creg and half[c][o].startswith("hsm["):
                    P.w("const double kin%d = %s;" % (c, half[c][o]))
                    kin.append("kin%d" % c)
                else:
                    kin.append(half[c][o])
            outs = emit_lin_names(P, ket, kin, "k", ["CD0", "CD1", "CD2"])
        ia, ib = divmod(o, nsb)
        if fock:
            P.w("const double dab = __ldg(Dm + (oa + %d) * nbf + ob + %d);" % (ia, ib))
            for idd in range(nsd):
                P.w("const double dbd%d = __ldg(Dm + (ob + %d) * nbf + od + %d), dad%d = __ldg(Dm + (oa + %d) * nbf + od + %d);" % (idd, ib, idd, idd, ia, idd))
            for ic in range(nsc):
                P.w("const double dbc%d = __ldg(Dm + (ob + %d) * nbf + oc + %d), dac%d = __ldg(Dm + (oa + %d) * nbf + oc + %d);" % (ic, ib, ic, ic, ia, ic))
            P.w("double jab = 0.0;")
            for r, e in enumerate(outs):
                ic, idd = divmod(r, nsd)
                P.w("{ const double v = %s;" % e)
                P.w("  jab = fma(dcd%d, v, jab); jcd%d = fma(dab, v, jcd%d);" % (r, r, r))
                P.w("  kac%d = fma(dbd%d, v, kac%d); kad%d = fma(dbc%d, v, kad%d);" % (ic, idd, ic, idd, ic, idd))
                P.w("  kbc%d_%d = fma(dad%d, v, kbc%d_%d); kbd%d_%d = fma(dac%d, v, kbd%d_%d); }" % (ib, ic, idd, ib, ic, ib, idd, ic, ib, idd))
            P.w("jab *= 2.0 * wq;")
            P.w("if (same_ab) {                          // one bra pair in the whole warp (the lists of a pass are sorted by bra pair): one atomic")
            P.w("    for (int off = 16; off > 0; off >>= 1) jab += __shfl_xor_sync(0xffffffffu, jab, off);")
            P.w("    if ((threadIdx.x & 31) == 0) atomicAdd(a.Jt + (oa + %d) * nbf + ob + %d, jab);" % (ia, ib))
            P.w("} else atomicAdd(a.Jt + (oa + %d) * nbf + ob + %d, jab);" % (ia, ib))
            if ib == nsb - 1:
                for ic in range(nsc):
                    P.w("atomicAdd(a.Kt + (oa + %d) * nbf + oc + %d, wq * kac%d); kac%d = 0.0;" % (ia, ic, ic, ic))
                for idd in range(nsd):
                    P.w("atomicAdd(a.Kt + (oa + %d) * nbf + od + %d, wq * kad%d); kad%d = 0.0;" % (ia, idd, idd, idd))
        else:
            def mine(idx):
                return "if (live && sl == %d) " % (idx % S) if split else ""
            P.w("if (canon) {")
            for r, e in enumerate(outs):
                if stage:
                    P.w("    ost[(threadIdx.x & 31) * %d + %d] = %s;" % (SCP, (o % srows) * nCD + r, e))
                else:
                    P.w("    %sout[%d] = %s;" % (mine(o * nCD + r), o * nCD + r, e))
            P.w("} else {")
            P.w("    double *ob = out + %d * a.ostride[0] + %d * a.ostride[1];" % (ia, ib))
            for r, e in enumerate(outs):
                ic, idd = divmod(r, nsd)
                P.w("    %sob[%d * a.ostride[2] + %d * a.ostride[3]] = %s;" % (mine(o * nCD + r), ic, idd, e))       # (staged kernels: a thread past the end rewrites the last block with the same values)
            P.w("}")
        P.ind -= 1
        P.w("}")
        if stage and ((o + 1) % srows == 0 or o == nAB - 1):
            o0 = (o // srows) * srows
            cnt = (o + 1 - o0) * nCD
            P.w("if (canon) {      // rows %d..%d of the warp's 32 blocks: 32 segments of %d doubles" % (o0, o, cnt))
            P.w("    __syncwarp();")
            P.w("    const int lane_ = threadIdx.x & 31;")
            P.w("    const int64_t qw = q_ - lane_;")
            P.w("    const int nv = (int)min((int64_t)32, a.n - qw);")
            P.w("    double *og = a.out + qw * a.out_stride + %d;" % (o0 * nCD))
            P.w("    #pragma unroll")
            P.w("    for (int k = 0; k < %d; ++k) {" % cnt)
            P.w("        const int e = lane_ + 32 * k, tq = e / %d, ix = e - tq * %d;" % (cnt, cnt))
            P.w("        if (tq < nv) og[tq * a.out_stride + ix] = ost[tq * %d + ix];" % SCP)
            P.w("    }")
            P.w("    __syncwarp();")
            P.w("}")
    if fock:
        for r in range(nCD):
            ic, idd = divmod(r, nsd)
            P.w("atomicAdd(a.Jt + (oc + %d) * nbf + od + %d, 2.0 * wq * jcd%d);" % (ic, idd, r))
        for ib in range(nsb):
            for ic in range(nsc):
                P.w("atomicAdd(a.Kt + (ob + %d) * nbf + oc + %d, wq * kbc%d_%d);" % (ib, ic, ib, ic))
            for idd in range(nsd):
                P.w("atomicAdd(a.Kt + (ob + %d) * nbf + od + %d, wq * kbd%d_%d);" % (ib, idd, ib, idd))
    P.ind = 0
    P.w("}")
    P.w("}  // namespace %s" % ns)
    lname = "rcg_launch_fock_reg_%s" % tag if fock else ("rcg_launch_regsplit_%s" % tag if split else "rcg_launch_reg_%s" % tag)
    P.w("static cudaError_t %s(const RcgLaunch &a)" % lname)
    P.w("{")
    P.w("    int nsm = 0, bs = 128;                    // short lists: smaller blocks, so that every SM gets at least two")
    P.w("    cudaError_t e = rcg_sm_count(&nsm);")
    P.w("    if (e != cudaSuccess) return e;")
    P.w("    const int64_t nthr = a.n * %d;" % (S if split else 1))
    P.w("    while (bs > 32 && nthr / bs < 2 * (int64_t)nsm) bs >>= 1;")
    smt = nsm_slots + (SCP if stage else 0)          # doubles of shared memory per thread
    if smt * 8 * 128 > 72 * 1024:
        P.w("    while (bs > 32 && (size_t)bs * %d > 72 * 1024) bs >>= 1;      // three blocks per SM by shared memory" % (smt * 8))
    bs_max = 128
    while bs_max > 32 and smt * 8 * 128 > 72 * 1024 and smt * 8 * bs_max > 72 * 1024:
        bs_max >>= 1
    if smt * bs_max * 8 > 48 * 1024:
        P.w("    static RcgOnce once;")
        P.w("    if ((e = rcg_prepare_kernel(once, (const void *)%s::%s, sizeof(double) * %d * %d, nullptr)) != cudaSuccess) return e;" % (ns, kname, smt, bs_max))
    P.w("    %s::%s<<<(unsigned)((nthr + bs - 1) / bs), bs, sizeof(double) * %d * bs, a.stream>>>(a);" % (ns, kname, smt))
    P.w("    return cudaGetLastError();")
    P.w("}")
    if fock or split:
        return P.text() + "\n", lname, {}
    meta = dict(reg_smem_accumulators=nsm_slots, reg_vertices=g.num_nodes(), reg_order="dsa" if order is order_dsa else "postorder",
                reg_peaklive_postorder=pl_post, reg_peaklive_dsa=pl_dsa, reg_accumulators=nT * nC)
    return P.text() + "\n", "rcg_launch_reg_%s" % tag, meta


def emit_auto(cls, warp_text, warp_sym, reg_text, reg_sym):
    """both tiers in one source + the launcher that picks per call (no host synchronisation)."""
    tag = "%d%d%d%d" % cls
    w = []
    w.append("static cudaError_t rcg_launch_%s_regauto(const RcgLaunch &a)" % tag)
    w.append("{")
    w.append("    if (a.force_tier == RCG_TIER_WARP) return %s(a);" % warp_sym)
    w.append("    if (a.force_tier == RCG_TIER_REGISTER) return %s(a);" % reg_sym)
    la, lb, lc, ld = cls
    g = VrrGraph(la, lb, lc, ld)
    heavy = len(g.target_a) * len(g.target_c) > 56      # 250+ registers per thread: one block of 128 per SM, needs a longer list to win
    minq = REG_MIN_QUARTETS_HEAVY if heavy else REG_MIN_QUARTETS
    w.append("    {   // short list of evenly and deeply contracted shells: %d lanes per quartet, each taking every %d-th primitive quartet" % (REG_SPLIT, REG_SPLIT))
    w.append("        bool even = true; int64_t k4 = 1;")
    w.append("        for (int k = 0; k < 4; ++k) { even = even && a.kmin[a.lcan[k]] == a.kmax[a.lcan[k]]; k4 *= a.kmax[a.lcan[k]]; }")
    if cls not in REG_SPLIT_EXCLUDED:
        w.append("        if (even && k4 >= %d && a.n < %d && a.n * %d >= %d) return rcg_launch_regsplit_%s(a);" % (4 * REG_SPLIT, minq, REG_SPLIT, minq, tag))
    w.append("    }")
    w.append("    if (a.n < %d) return %s(a);        // too few quartets for one thread each to fill the GPU" % (minq, warp_sym))
    w.append("    if (a.uniform_k4) return %s(a);     // the caller's promise (rcg_eri_batch_uniform): one K4 in the whole list" % reg_sym)
    w.append("    double spread = 1.0;      // bound on max K4 / min K4 over the quartets of this class in this basis")
    w.append("    for (int k = 0; k < 4; ++k) spread *= (double)a.kmax[a.lcan[k]] / (double)a.kmin[a.lcan[k]];")
    w.append("    if (spread <= 1.3) return %s(a);" % reg_sym)
    w.append("    // uneven contraction depths: measure, on THIS list, what looping 32 consecutive quartets to their")
    w.append("    // largest K4 would waste; both tiers are enqueued, the loser of the device-side test returns at once")
    w.append("    RcgLaunch b = a;")
    w.append("    cudaError_t e = rcg_pack_stats(a, 32, 1, &b.stat_reg);")
    w.append("    if (e != cudaSuccess) return e;")
    w.append("    e = %s(b);" % reg_sym)
    w.append("    return e != cudaSuccess ? e : %s(b);" % warp_sym)
    w.append("}")
    return warp_text + reg_text + "\n".join(w) + "\n", "rcg_launch_%s_regauto" % tag
