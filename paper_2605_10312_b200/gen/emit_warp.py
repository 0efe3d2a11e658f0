"""Emit the warp tier (RCG_TIER_WARP) kernel of one class: straight-line CUDA for sm_100a.

Work decomposition (replaces the paper's thread-per-quartet Tier 1,
PAPER.md:259-261, whose frontier + accumulators need ~3,300 registers at (dd|dd)):
  * one warp per shell quartet; lane = one bra Cartesian component a with |a| in [la,la+lb]
    ("target" lanes); the lane keeps the whole ket table [a0|c0]^(m) of ITS component in
    registers and owns the nC contraction accumulators H[a][.] (Alg. 2 line 7).
  * with the ket-first axis rule a ket step of Eq. (2) reads [a|c-1i], [a|c-2i]
    (same lane) and ONE cross term [a-1i|c-1i]^(m+1), fetched from the lane that owns a-1i by
    __shfl_sync; every lane executes the same (c,m) schedule (the Boys order a vertex needs depends
    on c only), so the generated code is one straight-line program per class, not one per vertex.
  * the pure-bra vertices [a0|00]^(m) are built lane-locally along the lane's own path
    x^ax y^ay z^az (la+lb steps; lanes with shorter paths take identity steps first).
  * components below la ("lower" lanes, needed only as cross-term sources) are evaluated for PB
    primitive quartets at once (lane = (primitive, lower component)) in a lower pass whose results
    go through shared memory; primitive-quartet set-up (pair quantities, Boys) is likewise done for
    PBS primitives at once, one per lane, and broadcast through shared memory.
  * Phase 2 (HRR + stepwise c2s, Eqs. (11)-(16)) transposes H through shared memory: lane = ket
    column for the bra side, lane = spherical bra row for the ket side, then a coalesced store.
"""
import os

from . import options
from .graph import VrrGraph, hrr_c2s_program, c2s_pair_program, reduction_axis, sub1
from .solid import cart_comps


# Cross-term loads issued together per ket level (chunk sizes by level), where a sweep on the B200 found better than the
# uniform default of 8: ptxas' schedule falls into one of two modes and inside the fast one the split of a
# level matters by 2%.  (dd|dd), levels of 12 / 18 / 20 / 15 vertices: 8+4, 9+9, 8+8+4, 8+7 -> 1.849 ms against 1.887 ms.
WARP_CHUNKS = {(2, 2, 2, 2): "8,9,8,8"}
ACC_REG_MAX, ACC_REG_KEEP = 36, 30
# lane tables staged in shared memory (a lane-indexed __constant__ read serialises over the lanes): 4-26% on the K4 <= 10 lists of the
# screened passes; measured slower (3-14%) for these kernels, which keep the __constant__ reads
TAB_CONST = {(2, 2, 2, 1), (1, 0, 3, 2), (1, 1, 3, 2), (2, 0, 3, 2)}
TAB_CONST_FOCK = {(3, 1, 2, 2)}       # Fock variants that would spill (16 bytes) with the staged tables
GRP_RECS = 16          # grouped set-up: records kept beside the first quartet's (quartets per group: 1 + GRP_RECS / K4, at most 32 / K4)      # accumulators per lane kept in registers (all, if at most ACC_REG_MAX)
ACC_KEEP_OF = {(1, 1, 3, 2): 14, (3, 0, 3, 2): 22}      # kernels (generated for the swapped quartet) that need more room for 0 spill bytes (ptxas)


def path_steps(a):
    """the lane's own bra path: x's first, then y's, then z's -> [(axis, n_before)]."""
    out = []
    for ax in range(3):
        for n in range(a[ax]):
            out.append((ax, n))
    return out


def bra_pyramid(nst, ctop):
    """Pure-bra vertices [a0|00]^(m), |a| <= nst, shared between lanes: one representative per orbit of
    the cyclic axis rotation x->y->z->x, each with a parent (and grandparent) that is itself a
    representative, so ONE straight-line program run by three lanes with rotated axes (PA, WP
    permuted) yields every component.  Returns ([(rep, axis, parent, n, grandparent, mmax)], mmax of F)."""
    rot = lambda a: (a[2], a[0], a[1])                      # noqa: E731
    reps = {(0, 0, 0)}
    out = []
    for e in range(1, nst + 1):
        seen = set()
        for a in cart_comps(e):
            if a in seen:
                continue
            orbit = [a, rot(a), rot(rot(a))]
            seen.update(orbit)
            choice = None
            for cand in orbit:
                for i in range(3):
                    if cand[i] == 0:
                        continue
                    par = sub1(cand, i)
                    gp = sub1(par, i) if par[i] > 0 else None
                    if par in reps and (gp is None or gp in reps):
                        choice = (cand, i, par, par[i], gp)
                        break
                if choice:
                    break
            assert choice, "no closed representative for orbit of %s" % (a,)
            out.append(choice)
        reps.update(c[0] for c in out)
    need = {r[0]: ctop for r in out}
    need[(0, 0, 0)] = ctop
    for (rep, i, par, n, gp) in reversed(out):
        need[par] = max(need[par], need[rep] + 1)
        if gp is not None:
            need[gp] = max(need[gp], need[rep] + 1)
    return [(rep, i, par, n, gp, need[rep]) for (rep, i, par, n, gp) in out], need[(0, 0, 0)]


class Prog:
    def __init__(self):
        self.lines = []
        self.ind = 1

    def w(self, s=""):
        self.lines.append("    " * self.ind + s if s else "")

    def text(self):
        return "\n".join(self.lines)


def ket_nodes(S, ctop):
    """non-base vertices of the (c,m) set S in dependency order: by |c|, then component, then m."""
    out = []
    for k in range(1, ctop + 1):
        for c in cart_comps(k):
            ms = sorted(m for (cc, m) in S if cc == c)
            for m in ms:
                out.append((c, m))
    return out


def emit_lin(P, prog, src_expr, var, X):
    """straight-line code for a LinProgram; inputs via src_expr(k); X = names of the 3 displacements."""
    for k in range(prog.nin):
        P.w("double %s%d = %s;" % (var, k, src_expr(k)))
    defined = set(range(prog.nin))
    for (dst, src, coef, init) in prog.ops:
        if coef[0] == "one":
            cs = None
        elif coef[0] == "x":
            cs = X[coef[1]]
        elif coef[1] == 1.0:
            cs = None
        else:
            cs = repr(float(coef[1]))
        s = "%s%d" % (var, src)
        d = "%s%d" % (var, dst)
        if init:
            assert dst not in defined
            defined.add(dst)
            P.w("double %s = %s;" % (d, s if cs is None else "%s * %s" % (cs, s)))
        else:
            assert dst in defined
            P.w("%s = %s;" % (d, "%s + %s" % (d, s) if cs is None else "fma(%s, %s, %s)" % (cs, s, d)))


def _has_register_tier(cls):
    from .tiers import register_eligible
    return register_eligible(cls) or register_eligible((cls[2], cls[3], cls[0], cls[1]))


def _emit_variant(cls, qforce, suffix, warps=None, minblocks=None, fock=False):
    # warps per (persistent, one per SM) block: 8 where the kernel needs the full 255 registers; classes with at
    # most 10 ket targets per lane stay below 168 registers (ptxas) and run 12 -- their lists are mostly K4 = 1
    # and latency-bound, a third warp per scheduler gave 20-25% on the cfg3 pass
    nC_ = sum(len(cart_comps(f)) for f in range(cls[2], cls[2] + cls[3] + 1))
    warps = warps or options.geti("WARP_WARPS", 0) or (12 if nC_ <= 10 else 8)
    minblocks = minblocks or options.geti("WARP_MINBLOCKS", 1)
    la, lb, lc, ld = cls
    tag = "%d%d%d%d%s" % (cls + (suffix,))
    g = VrrGraph(la, lb, lc, ld)
    nst, ctop = la + lb, lc + ld
    L = nst + ctop
    T = [a for e in range(la, la + lb + 1) for a in cart_comps(e)]
    LW = [a for e in range(0, la) for a in cart_comps(e)]
    nT, nLow = len(T), len(LW)
    assert nT <= 32
    # Q quartets per warp, G lanes per quartet ("group"): light bra sides pack several quartets into a warp
    Q = qforce or (32 // max(nT, nLow, 1) if max(nT, nLow) <= 16 else 1)
    Q = min(Q, options.geti("WARP_QCAP", 4))
    if nT < 3 and not qforce:
        Q = 1              # (ss|ss): set-up bound, 16 primitives per pass beat 4 quartets x 8 lanes (measured)
    G = 32 // Q
    KC = [c for k in range(ctop + 1) for c in cart_comps(k)]
    kidx = {c: i for i, c in enumerate(KC)}
    TC = [c for f in range(lc, lc + ld + 1) for c in cart_comps(f)]
    nC = len(TC)
    tset, lset = set(T), set(LW)
    S_main = {(c, m) for (a, c, m) in g.nodes if a in tset}
    S_low = {(c, m) for (a, c, m) in g.nodes if a in lset}
    main_nodes = ket_nodes(S_main, ctop)
    low_nodes = ket_nodes(S_low, ctop)
    for S in (S_main, S_low):
        for (c, m) in S:
            if sum(c) == 0:
                continue
            i = reduction_axis(c)
            c1 = sub1(c, i)
            assert (c1, m) in S and (c1, m + 1) in S
            if c1[i] > 0:
                assert (sub1(c1, i), m) in S and (sub1(c1, i), m + 1) in S
    # values exchanged between lanes through shared memory: every cross-term source (c-1i, m+1)
    EX = []
    if nst:
        for (c, m) in main_nodes:
            c1 = sub1(c, reduction_axis(c))
            if (c1, m + 1) not in EX:
                EX.append((c1, m + 1))
    exidx = {k: i for i, k in enumerate(EX)}
    NEX = len(EX)
    # exchange-row strides chosen so that every cross-term gather (a 64-bit load per lane) is free of
    # shared-memory bank conflicts: model = per half-warp, max number of distinct addresses per 8-byte bank
    L1C = cart_comps(la - 1) if la >= 1 else []       # lower components the target lanes read (level la-1)
    nL1 = len(L1C)

    def src_desc(lane, i):
        a = T[lane] if lane < nT else None
        if a is None or a[i] == 0:
            half = lane & 16
            act = [ln for ln in range(half, half + 16) if ln < nT and T[ln][i] > 0]
            if not act:
                return ("M", lane)
            a = T[act[0]]
        am = sub1(a, i)
        return ("M", T.index(am)) if am in tset else ("L", L1C.index(am))

    def wavefronts(addrs):
        tot = 0
        for h in (0, 16):
            banks = {}
            for x in set(addrs[h:h + 16]):
                banks.setdefault(x % 16, set()).add(x)
            tot += max(len(v) for v in banks.values())
        return tot

    def wavefronts16(addrs):          # one half-warp, predicated-off lanes left out
        banks = {}
        for x in set(addrs):
            banks.setdefault(x % 16, set()).add(x)
        return max([len(v) for v in banks.values()] + [0])

    NEXs, NLS, PADX, JST = NEX | 1, NEX | 1, 0, nL1 * (NEX | 1)
    JSTH, jnest = 0, False
    if nst:
        desc = [[src_desc(ln, i) for i in range(3)] for ln in range(32)]
        pbg = min(G // nLow, options.geti("WARP_PB", 8)) if nLow else 1
        # weights: a (jj, axis) gather pattern runs once per ket vertex reduced along that axis; the lower
        # pass's store pattern runs once per exported lower value per PB primitives.  Only the strides
        # mod 16 matter for the banks, so the search runs over residues and takes the smallest strides.
        n_ax = [len([1 for (c, m) in main_nodes if reduction_axis(c) == i]) for i in range(3)]
        n_lst = len([1 for k in EX if k in S_low])
        best = None
        for sx in range(NEX | 1, NEX + 3, 2):                    # odd: conflict-free exports of the target lanes
            for sl in (range(NEX, NEX + 16) if nLow else [NEX]):
                for dj in (range(0, 16) if nLow else [0]):       # extra skew per primitive of the lower tables
                    jst = nL1 * sl + dj
                    for dl in (range(16) if nLow else [0]):
                        tot = 0
                        if nLow:   # the lower pass's stores: lane (jj, level la-1 comp) writes row jj*jst + comp*sl
                            rows_l = [dl + (ln // nLow) * jst + L1C.index(LW[ln % nLow]) * sl
                                      if LW[ln % nLow] in L1C else None for ln in range(pbg * nLow)]
                            rows_l += [None] * (32 - len(rows_l))
                            tot += n_lst * sum(wavefronts16([x for x in rows_l[h:h + 16] if x is not None]) for h in (0, 16))
                        for jj in range(pbg):
                            if best is not None and tot > best[0]:
                                break
                            for i in range(3):
                                if n_ax[i]:
                                    tot += n_ax[i] * wavefronts([(r * sx) if k == "M" else ((1 << 20) + dl + jj * jst + r * sl)
                                                                 for (k, r) in (desc[ln][i] for ln in range(32))])
                        key = (tot, jst, sl, sx)
                        if best is None or key < best[0:1] + best[5:]:
                            best = (tot, sx, sl, dl, jst, jst, sl, sx)
        best = best[:5]
        if options.flag("GEN_VERBOSE"):
            print('layout search', cls, 'Q', Q, 'best', best, 'ideal', 2 * pbg * sum(n_ax) + n_lst)
        _, NEXs, NLS, PADX, JST = best
        # second family (two-level strides): the lower table of primitive jj sits at (jj >> 2) * JSTH + (jj & 3) * JST with
        # JSTH = 0 (mod 16).  One linear stride cannot keep the level la-1 rows of all PB tables off the banks of the
        # main rows ((dd|dd): 2 of 8 tables cost a third wavefront per gather); a run of four can, and the second
        # four repeat the residues of the first.  The primitive loop becomes a 2 x 4 nest, still affine for ptxas.
        if nLow and pbg == 8 and options.get("WARP_JNEST", "0") == "1":
            bestf = None
            for sx in range(NEX | 1, NEX + 3, 2):
                for sl in range(NEX, NEX + 16):
                    gcost = []
                    for d in range(16):
                        gcost.append(sum(n_ax[i] * wavefronts([(r * sx) if k == "M" else ((1 << 20) + d + r * sl)
                                                               for (k, r) in (desc[ln][i] for ln in range(32))])
                                         for i in range(3) if n_ax[i]))

                    def store_cost(ds):
                        rows_l = [(ln // nLow) * 4096 + ds[ln // nLow] + L1C.index(LW[ln % nLow]) * sl
                                  if LW[ln % nLow] in L1C else None for ln in range(pbg * nLow)]
                        rows_l += [None] * (32 - len(rows_l))
                        return n_lst * sum(wavefronts16([x for x in rows_l[h:h + 16] if x is not None]) for h in (0, 16))

                    for dlt in range(16):
                        for dl in range(16):
                            ds = [(dl + (jj & 3) * dlt) % 16 for jj in range(pbg)]
                            key = (sum(gcost[x] for x in ds) + store_cost(ds), sl, sx, dlt, dl)
                            if bestf is None or key < bestf:
                                bestf = key
            if options.flag("GEN_VERBOSE"):
                print('two-level search', cls, 'Q', Q, 'best', bestf)
            if bestf[0] < best[0]:
                _, NLS, NEXs, dlt, PADX = bestf
                JST = nL1 * NLS + (dlt - nL1 * NLS) % 16
                JSTH = (4 * JST + 15) // 16 * 16
                jnest = True
    PB = min(G // nLow, options.geti("WARP_PB", 8)) if nLow else 0
    PBS = min(options.geti("WARP_PBS", 16), G)   # primitives set up per pass (one per lane)
    if nLow:
        PBS = max(PB, PBS // PB * PB)
    # pure-bra values the ket programs read: [a0|00]^(m), m <= ctop (main) / mb_low (lower lanes)
    assert max([m + 1 for (c, m) in main_nodes if sum(c) == 1] + [0]) == ctop
    mb_low = max([m + 1 for (c, m) in low_nodes if sum(c) == 1] + [m for (c, m) in EX if sum(c) == 0 and (c, m) in S_low] + [0])
    nstl = max(la - 1, 0)
    # primitive record layout
    OFF_F = 0
    OFF_PA = L + 1
    OFF_WP = OFF_PA + 4
    OFF_HZN = OFF_WP + 4
    n_hzn = max(nst, 1)
    OFF_RZ = OFF_HZN + n_hzn
    pairs = Q == 1                       # 16-byte broadcast loads only when the whole warp reads ONE record
    OFF_QC = (OFF_RZ + 2) & ~1 if pairs else OFF_RZ + 1
    OFF_WQ = OFF_QC + 3
    OFF_HEN = OFF_WQ + 3
    OFF_RE = OFF_HEN + ctop + 1
    OFF_HZEN = OFF_RE + 1
    NREC = OFF_HZEN + nst + 1
    PRS = (NREC + 1) & ~1 if pairs else NREC | 1     # even keeps 16-byte alignment; odd spreads the groups' records over banks
    if pairs and (PRS // 2) % 2 == 0 and options.get("WARP_PRS_SKEW", "1") == "1":
        PRS += 2      # set-up stores: lane p writes record p, stride PRS; PRS = 2 * odd puts 16 lanes on 8 distinct 8-byte banks
                      # (2 wavefronts per store) where PRS = 0 mod 4 leaves 4 or fewer (PRS = 40 at (dd|dd): 8 wavefronts)
    nAB = (2 * la + 1) * (2 * lb + 1)
    nCD = (2 * lc + 1) * (2 * ld + 1)
    # ablation "no spherical fusion" (SPH_FUSION=0): the bra pair stays Cartesian through the ket side
    # (ncart(la) ncart(lb) rows instead of (2la+1)(2lb+1)) and is transformed last, Eq. (17)'s order for the bra
    fused = options.get("SPH_FUSION", "1") != "0"
    nABc = nAB if fused else len(cart_comps(la)) * len(cart_comps(lb))
    bra = hrr_c2s_program(la, lb, c2s=fused)
    ket = hrr_c2s_program(lc, ld)
    late = None if fused else c2s_pair_program(la, lb)
    HS = nC | 1                         # row stride of H and B in Phase 2: odd, so that the lane-per-row accesses (H store, ket program) are
    #                                     free of bank conflicts (stride 16 of the (xx|dp) classes: 16-way conflicts, 75% of the shared-memory
    #                                     bandwidth of the SM on K4 = 1 lists)
    SA = max(nT * HS, nABc * nCD)
    SB = nABc * HS
    OFF_LOW = PBS * PRS                 # lower tables [PB][nLow][NEXs] (+1 dump row)
    OFF_XM = OFF_LOW + (PB * JST if not jnest else (PB + 3) // 4 * JSTH)     # lower tables [PB] x JST, then main rows [nxrow][NEXs]
    if nLow:
        OFF_XM += (OFF_LOW - PADX - OFF_XM) % 16   # (OFF_LOW - OFF_XM) = PADX (mod 16), as the search assumed
    nexp = len([a for a in T if sum(a) < la + lb])      # target lanes that are cross-term sources
    nxrow = max(nexp, 1)
    OFF_BT = OFF_XM + (nxrow * NEXs if nst else 0)
    use_pyr = Q == 1 and nst >= 2 and nLow > 0 and options.flag("WARP_PYRAMID")   # measured slower at (dd|dd): off
    BTS = ((nLow + nT) * (ctop + 1)) | 1              # pure-bra table [PB][all components][ctop+1]
    if use_pyr:     # per-primitive stride of the table chosen against bank conflicts of the bra pass's stores
        pyr0, _ = bra_pyramid(nst, ctop)
        allc = LW + T
        rot1 = lambda a: (a[2], a[0], a[1])                 # noqa: E731
        bestb = None
        for cand in range(BTS, BTS + 32, 2):
            tot = 0
            for (rep_, _i, _p, _n, _g, _mm) in pyr0:
                comps = [rep_, rot1(rep_), rot1(rot1(rep_))]
                tot += wavefronts([min(ln // 3, PB - 1) * cand + allc.index(comps[ln % 3]) * (ctop + 1) for ln in range(32)])
            if bestb is None or tot < bestb[0]:
                bestb = (tot, cand)
        BTS = bestb[1]
    NVRR = OFF_BT + (PB * BTS if use_pyr else 0)
    R1 = max(NVRR - SA, SB, 0)          # Phase 2 aliases the VRR region: [B | H/out]
    nsa_, nsb_, nsc_, nsd_ = 2 * la + 1, 2 * lb + 1, 2 * lc + 1, 2 * ld + 1
    # Fock variant: the six density sub-blocks D_cd, D_ab, D_bd, D_ad, D_bc, D_ac are staged in the B region once Phase 2 is through with it
    DOFF = [0, nCD, nCD + nAB, nCD + nAB + nsb_ * nsd_, nCD + nAB + nsb_ * nsd_ + nsa_ * nsd_, nCD + nAB + nsb_ * nsd_ + nsa_ * nsd_ + nsb_ * nsc_]
    DSZ = DOFF[5] + nsa_ * nsc_
    if fock:
        assert fused, "the Fock epilogue is generated for the default (fused c2s) Phase 2 only"
        R1 = max(R1, DSZ)
    WSM = max(NVRR, R1 + SA)            # doubles of shared memory per warp
    # lanes with more than ACC_REG_MAX accumulators (the swapped (xx|fd) kernels: 46) keep the last ones in their own shared-memory column
    # [slot][lane], outside the aliased regions: explicit staging where ptxas otherwise spills 76-230 bytes
    nacc_reg = nC if nC <= ACC_REG_MAX else options.geti("WARP_ACC_KEEP", ACC_KEEP_OF.get(cls, ACC_REG_KEEP))
    OFF_ASM = WSM
    WSM += (nC - nacc_reg) * G
    WSM = (WSM + 1) & ~1 if pairs else WSM | 1
    # grouped set-up (lists with one K4 <= 16): one set-up pass prepares the records of several consecutive quartets, the first
    # quartet's in the usual place, the others' in GRP_RECS records behind everything Phase 2 aliases
    grouped = Q == 1 and not fock and options.flag("WARP_GROUP")
    OFF_RG = WSM
    if grouped:
        WSM += GRP_RECS * PRS
        WSM = (WSM + 1) & ~1 if pairs else WSM | 1

    def A(t):
        return "acc%d" % t if t < nacc_reg else "ASM[%d]" % ((t - nacc_reg) * G)

    # ---- lane tables
    def pack_main(a):
        steps = path_steps(a)
        pad = nst - len(steps)
        sel = [OFF_PA + 3] * pad + [OFF_PA + ax for ax, _ in steps]
        nn = [0] * pad + [n for _, n in steps]
        src, low = [], []
        for i in range(3):
            if a[i] > 0:
                am = sub1(a, i)
                if am in tset:
                    src.append(OFF_XM + T.index(am) * NEXs)      # row of the owning target lane
                    low.append(0)
                else:
                    src.append(OFF_LOW + L1C.index(am) * NLS)    # lower table (+ jj * JST at run time)
                    low.append(1)
            else:
                src.append(-1)                                   # own row, coefficient 0
                low.append(0)
        return sel, nn, src, low

    rows_main = []
    for lane in range(32):
        a = T[lane] if lane < nT else T[0]
        sel, nn, src, low = pack_main(a)
        src = [s if s >= 0 else OFF_XM + lane * NEXs for s in src]
        if lane >= nT:
            src = [OFF_XM + lane * NEXs] * 3
            low = [0, 0, 0]
        rows_main.append(list(a) + src + low + sel + nn)
    # lanes with a_i = 0 (coefficient 0) read the SAME address as an active lane of their half-warp:
    # a shared-memory broadcast instead of an extra bank conflict
    for half in (0, 16):
        for i in range(3):
            act = [ln for ln in range(half, half + 16) if ln < nT and T[ln][i] > 0]
            if not act:
                continue
            for ln in range(half, half + 16):
                if ln >= nT or T[ln][i] == 0:
                    rows_main[ln][3 + i] = rows_main[act[0]][3 + i]
                    rows_main[ln][6 + i] = rows_main[act[0]][6 + i]
    for ln in range(32):                                  # rows that do not exist (top-level / idle lanes)
        for i in range(3):
            if rows_main[ln][6 + i] == 0 and rows_main[ln][3 + i] >= OFF_XM + nxrow * NEXs:
                rows_main[ln][3 + i] = OFF_XM
    # lower pass lanes: lane = jj*nLow + comp
    rows_low = []
    for lane in range(32):
        if nLow and lane < PB * nLow:
            jj, comp = divmod(lane, nLow)
            exoff = (jj * JST if not jnest else (jj >> 2) * JSTH + (jj & 3) * JST) + L1C.index(LW[comp]) * NLS if LW[comp] in L1C else -1
        else:
            jj, comp = 0, 0
            exoff = -1                     # idle lane: no export
        a = LW[comp] if nLow else (0, 0, 0)
        steps = path_steps(a)
        pad = nstl - len(steps)
        sel = [OFF_PA + 3] * pad + [OFF_PA + ax for ax, _ in steps]
        nn = [0] * pad + [n for _, n in steps]
        src = []
        for i in range(3):
            if nLow and a[i] > 0 and lane < PB * nLow:
                src.append(jj * nLow + LW.index(sub1(a, i)))     # group-local lane that owns a-1i (shuffle source)
            else:
                src.append(lane % G)
        rows_low.append(list(a) + src + [jj, exoff] + sel + nn)
    NM = len(rows_main[0])
    NL = len(rows_low[0])

    tab_smem = options.geti("WARP_TAB_SMEM", 0 if (cls in TAB_CONST or (fock and cls in TAB_CONST_FOCK)) else 1) == 1
    TABD = ((NM + NL) * 32 * 4 + 7) // 8 if tab_smem else 0     # the lane tables, staged in shared memory: doubles behind the warps' regions
    warps = max(1, min(warps, (225 * 1024 - TABD * 8 * minblocks) // (WSM * Q * 8 * minblocks)))    # fit the SM's 227 KB of shared memory
    P = Prog()
    def emit_quartet_loads():
        P.w("const int sh0 = a.quartets[4 * q + a.perm[0]], sh1 = a.quartets[4 * q + a.perm[1]];")
        P.w("const int sh2 = a.quartets[4 * q + a.perm[2]], sh3 = a.quartets[4 * q + a.perm[3]];")
        P.w("double RA[3], RB[3], RC[3], RD[3];")
        P.w("#pragma unroll")
        P.w("for (int t = 0; t < 3; ++t) { RA[t] = b.centers[3 * sh0 + t]; RB[t] = b.centers[3 * sh1 + t]; RC[t] = b.centers[3 * sh2 + t]; RD[t] = b.centers[3 * sh3 + t]; }")
        P.w("const int pa0 = b.prim_off[sh0], Ka = b.prim_off[sh0 + 1] - pa0;")
        P.w("const int pb0 = b.prim_off[sh1], Kb = b.prim_off[sh1 + 1] - pb0;")
        P.w("const int pc0 = b.prim_off[sh2], Kc = b.prim_off[sh2 + 1] - pc0;")
        P.w("const int pd0 = b.prim_off[sh3], Kd = b.prim_off[sh3 + 1] - pd0;")
        P.w("const int K4 = Ka * Kb * Kc * Kd;")

    def emit_setup(pexpr, dest):
        """set-up of primitive quartet `pexpr` of the quartet whose shells are in scope: Boys values and VRR coefficients -> record at `dest`"""
        P.w("int p = %s;" % pexpr)
        if options.flag("WARP_IDIV"):
            P.w("const int il = p % Kd; p /= Kd; const int ik = p % Kc; p /= Kc; const int ij = p % Kb; const int ii = p / Kb;")
        else:
            P.w("const float rKd = __fdividef(1.0f, (float)Kd), rKc = __fdividef(1.0f, (float)Kc), rKb = __fdividef(1.0f, (float)Kb);")
            P.w("int il, ik, ij; p = rcg_divmod(p, Kd, rKd, il); p = rcg_divmod(p, Kc, rKc, ik); const int ii = rcg_divmod(p, Kb, rKb, ij);")
        P.w("RcgPrim pq;")
        P.w("rcg_prim_setup(pq, RA, RB, RC, RD, b.exps[pa0 + ii], b.exps[pb0 + ij], b.exps[pc0 + ik], b.exps[pd0 + il],")
        P.w("               b.coefs[pa0 + ii] * b.coefs[pb0 + ij] * b.coefs[pc0 + ik] * b.coefs[pd0 + il]);")
        P.w("double F[%d];" % (L + 1))
        P.w("rcg_boys<%d>(%d, pq.T, pq.pref, b.boys, F);" % (L, L))
        P.w("double *pr = %s;" % dest)
        rec = {m: "F[%d]" % m for m in range(L + 1)}
        for t in range(3):
            rec[OFF_PA + t] = "pq.PA[%d]" % t
            rec[OFF_WP + t] = "pq.WP[%d]" % t
            rec[OFF_QC + t] = "pq.QC[%d]" % t
            rec[OFF_WQ + t] = "pq.WQ[%d]" % t
        rec[OFF_PA + 3], rec[OFF_WP + 3] = "1.0", "0.0"             # identity step of the pure-bra chain
        mult = lambda n, x: "0.0" if n == 0 else (x if n == 1 else "%d.0 * %s" % (n, x))     # noqa: E731
        for n in range(n_hzn):
            rec[OFF_HZN + n] = mult(n, "pq.hz")
        rec[OFF_RZ] = "pq.rz"
        for n in range(ctop + 1):
            rec[OFF_HEN + n] = mult(n, "pq.he")
        rec[OFF_RE] = "pq.re"
        for n in range(nst + 1):
            rec[OFF_HZEN + n] = mult(n, "pq.hze")
        assert max(rec) == NREC - 1
        if pairs:        # the record is 16-byte aligned (PRS and WSM even): 16-byte stores, half the store instructions
            for k in range(0, NREC, 2):
                P.w("*reinterpret_cast<double2 *>(pr + %d) = make_double2(%s, %s);" % (k, rec.get(k, "0.0"), rec.get(k + 1, "0.0")))
        else:
            for k in sorted(rec):
                P.w("pr[%d] = %s;" % (k, rec[k]))

    P.ind = 0
    P.w("// ---- warp tier kernel for (%d %d|%d %d): generated by gen/emit_warp.py" % cls)
    P.w("// target lanes %d, lower components %d (PB=%d), ket table %d vertices, accumulators/lane %d,"
        % (nT, nLow, PB, len(main_nodes), nC))
    P.w("// lower-pass vertices %d, exported lower values %d, shared memory %d B/warp" % (len(low_nodes), NEX, WSM * 8))
    P.w('#include "rcg_device.cuh"')
    P.w("namespace w%s {" % tag)
    P.w("constexpr int Q = %d, G = %d;     // quartets per warp, lanes per quartet" % (Q, G))
    P.w("constexpr int WARPS = %d, WSM = %d, PRS = %d, PBS = %d, PB = %d, NLOW = %d, NEXS = %d, NLS = %d, JST = %d, OFF_LOW = %d, OFF_XM = %d, OFF_BT = %d, BTS = %d, R1 = %d;"
        % (warps, WSM, PRS, PBS, PB, nLow, NEXs, NLS, JST, OFF_LOW, OFF_XM, OFF_BT, BTS, R1))
    P.w("__constant__ int c_main[32][%d] = {" % NM)
    for r in rows_main:
        P.w("  {" + ",".join(str(v) for v in r) + "},")
    P.w("};")
    P.w("__constant__ int c_low[32][%d] = {" % NL)
    for r in rows_low:
        P.w("  {" + ",".join(str(v) for v in r) + "},")
    P.w("};")
    P.w("#define FULL 0xffffffffu")
    P.w("__global__ void __launch_bounds__(WARPS * 32, %d) rcg_eri_warp_%s(RcgLaunch a)" % (minblocks, tag))
    P.w("{")
    P.ind = 1
    P.w("extern __shared__ __align__(16) double smem[];")
    P.w("const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;")
    P.w("const int grp = min(lane / G, Q - 1), gl = lane < Q * G ? lane % G : G - 1;   // spare lanes shadow the last one")
    if tab_smem:
        P.w("// lane tables [entry][lane] in shared memory: a lane-indexed read of __constant__ memory serialises over the 32 lanes, once per")
        P.w("// entry and quartet (16% of the stall samples of the (dd|ds) kernel on K4 = 1 lists); from here it is one conflict-free load")
        P.w("int *TMs = reinterpret_cast<int *>(smem + WSM * Q * WARPS), *TLs = TMs + %d * 32;" % NM)
        P.w("for (int i = threadIdx.x; i < %d * 32; i += WARPS * 32) TMs[i] = c_main[i & 31][i >> 5];" % NM)
        P.w("for (int i = threadIdx.x; i < %d * 32; i += WARPS * 32) TLs[i] = c_low[i & 31][i >> 5];" % NL)
        P.w("__syncthreads();")
        P.w("#define TM(k) TMs[(k) * 32 + gl]")
        P.w("#define TL(k) TLs[(k) * 32 + gl]")
    else:        # entry k of this lane: c_main[gl][k] (a lane's entries are contiguous: 64- and 128-bit constant loads)
        P.w("#define TM(k) c_main[gl][k]")
        P.w("#define TL(k) c_low[gl][k]")
    P.w("double *S1 = smem + (warp * Q + grp) * WSM;      // primitive records | lower tables | exchange rows (later: B)")
    P.w("double *SA = S1 + R1;                // Phase 2: H, later the output block (aliases the VRR region)")
    P.w("const RcgBasisDev &b = a.basis;")
    P.w("const bool canon = a.ostride[3] == 1 && a.ostride[2] == %d && a.ostride[1] == %d && a.ostride[0] == %d;"
        % (2 * ld + 1, (2 * ld + 1) * (2 * lc + 1), (2 * ld + 1) * (2 * lc + 1) * (2 * lb + 1)))
    if _has_register_tier(cls):
        P.w("if (a.stat_reg != nullptr && a.stat_reg[0] * 10ull <= a.stat_reg[1] * 13ull) return;   // the register-tier kernel takes this list")
    P.w("if (a.stat != nullptr) {           // device-side choice between the packed and the one-quartet-per-warp kernel")
    P.w("    const bool want_packed = a.stat[0] * 10ull <= a.stat[1] * 13ull;   // padded primitive work <= 1.3 x real work")
    P.w("    if (want_packed != (Q > 1)) return;")
    P.w("}")
    if grouped:
        P.w("// grouped set-up: on a list with one K4 <= 16 (uniform basis, or the caller's promise) one set-up pass serves NQ consecutive quartets")
        P.w("int k4u = 1;")
        P.w("{")
        P.w("    bool even = true;")
        P.w("    for (int k = 0; k < 4; ++k) { even = even && a.kmin[a.lcan[k]] == a.kmax[a.lcan[k]]; k4u *= a.kmax[a.lcan[k]]; }")
        P.w("    if (!even && a.uniform_k4) {")
        P.w("        k4u = 1;")
        P.w("        for (int k = 0; k < 4; ++k) { const int sh = a.quartets[a.perm[k]]; k4u *= b.prim_off[sh + 1] - b.prim_off[sh]; }")
        P.w("    } else if (!even) k4u = 0;")
        P.w("    if (k4u > %d) k4u = 0;       // one set-up pass per quartet (PBS) and the records beside the first quartet's" % min(GRP_RECS, PBS))
        P.w("}")
        P.w("const int64_t nwarps = (int64_t)gridDim.x * WARPS;")
        P.w("const int NQ = k4u ? (int)max((int64_t)1, min((int64_t)min(32 / k4u, 1 + %d / k4u), a.n / nwarps)) : 1;" % GRP_RECS)
        P.w("double *RG = S1 + %d;" % OFF_RG)
        P.w("for (int64_t qg = ((int64_t)blockIdx.x * WARPS + warp) * NQ; qg < a.n; qg += nwarps * NQ) {")
        P.w("if (NQ > 1) {")
        P.ind += 1
        P.w("const int hq = lane / k4u, hp = lane - hq * k4u;      // lane = (quartet of the group, primitive)")
        P.w("if (hq < NQ && qg + hq < a.n) {")
        P.ind += 1
        P.w("const int64_t q = qg + hq;")
        emit_quartet_loads()
        emit_setup("hp", "(hq == 0 ? S1 + hp * PRS : RG + (lane - k4u) * PRS)")
        P.ind -= 1
        P.w("}")
        P.w("__syncwarp();")
        P.ind -= 1
        P.w("}")
        P.w("for (int h = 0; h < NQ; ++h) {")
        P.w("const int64_t qb = qg + h;")
        P.w("if (qb >= a.n) break;")
        P.w("const double *REC = (h == 0) ? S1 : RG + (h - 1) * k4u * PRS;")
    else:
        P.w("for (int64_t qb = ((int64_t)blockIdx.x * WARPS + warp) * Q; qb < a.n; qb += (int64_t)gridDim.x * WARPS * Q) {")
    P.w("const bool qvalid = qb + grp < a.n;")
    P.w("const int64_t q = qvalid ? qb + grp : a.n - 1;     // a group past the end recomputes the last quartet, stores nothing")
    emit_quartet_loads()
    # lane statics (main)
    if nst:
        P.w("const int xo0 = TM(3), xo1 = TM(4), xo2 = TM(5);   // exchange rows of a-1x, a-1y, a-1z")
        if jnest:
            P.w("const int xl0 = TM(6), xl1 = TM(7), xl2 = TM(8);   // 1: the source is a lower table")
        else:
            P.w("const int xl0 = TM(6) * JST, xl1 = TM(7) * JST, xl2 = TM(8) * JST;")
    if nst:
        P.w("const int kax0 = %d + TM(0), kax1 = %d + TM(1), kax2 = %d + TM(2);" % (OFF_HZEN, OFF_HZEN, OFF_HZEN))
    for s in (range(nst) if not use_pyr else []):
        P.w("const int sel%d = TM(%d), nix%d = %d + TM(%d);" % (s + 1, 9 + s, s + 1, OFF_HZN, 9 + nst + s))
    if nacc_reg < nC:
        P.w("double *ASM = S1 + %d + gl;" % OFF_ASM)
    for t in range(nC):
        P.w("double acc%d = 0.0;" % t if t < nacc_reg else "%s = 0.0;" % A(t))
    P.w("const int K4w = __reduce_max_sync(FULL, K4);       // the groups of a warp loop together")
    P.w("for (int p0 = 0; p0 < K4w; p0 += PBS) {")
    P.ind += 1
    P.w("const int cnt = max(0, min(PBS, K4 - p0));")
    P.w("const int cntw = __reduce_max_sync(FULL, cnt);")
    # ---------------- setup pass
    if grouped:
        P.w("if (NQ == 1) {")
        P.ind += 1
    P.w("if (gl >= cnt && gl < cntw) {      // this group has fewer primitives left: all-zero records contribute nothing")
    P.w("    double *pz = S1 + gl * PRS;")
    P.w("    for (int m = 0; m < PRS; ++m) pz[m] = 0.0;")
    P.w("}")
    P.w("if (gl < cnt) {")
    P.ind += 1
    emit_setup("p0 + gl", "S1 + gl * PRS")
    P.ind -= 1
    P.w("}")
    P.w("__syncwarp();")
    if grouped:
        P.ind -= 1
        P.w("}")

    def emit_chain(nsteps, mfinal, selname, nixname, out_prefix):
        """lane-local pure-bra chain; returns names of [a0|00]^(m), m=0..mfinal."""
        top = mfinal + nsteps
        for k in (range(0, top + 1, 2) if pairs else []):
            P.w("const double2 %sf%d = *reinterpret_cast<const double2 *>(pr + %d);" % (out_prefix, k, k))
        names = {0: ["%sf%d.%s" % (out_prefix, m & ~1, "xy"[m & 1]) if pairs else "pr[%d]" % m for m in range(top + 1)]}
        P.w("const double rz = pr[%d];" % OFF_RZ) if nsteps >= 2 else None
        for s in range(1, nsteps + 1):
            P.w("const double %sc1_%d = pr[%s%d], %sc2_%d = pr[%s%d + 4];" % (out_prefix, s, selname, s, out_prefix, s, selname, s))
            if s >= 2:
                P.w("const double %skn_%d = pr[%s%d];" % (out_prefix, s, nixname, s))
            cur = names[s - 1]
            new = []
            for m in range(top - s + 1):
                nm = "%s%d_%d" % (out_prefix, s, m)
                if s == 1:
                    P.w("double %s = fma(%sc2_1, %s, %sc1_1 * %s);" % (nm, out_prefix, cur[m + 1], out_prefix, cur[m]))
                else:
                    prev = names[s - 2]
                    P.w("double %s = fma(%sc2_%d, %s, %sc1_%d * %s);" % (nm, out_prefix, s, cur[m + 1], out_prefix, s, cur[m]))
                    P.w("%s = fma(%skn_%d, fma(-rz, %s, %s), %s);" % (nm, out_prefix, s, prev[m + 1], prev[m], nm))
                new.append(nm)
            names[s] = new
        return names[nsteps][: mfinal + 1]

    def emit_ket(nodes, base_names, S, is_main, vp):
        """ket table in registers; cross terms [a-1i|c-1i]^(m+1) read from the owning lane's exchange row
        in shared memory (rows xb0/xb1/xb2), own exchangeable values written to row `xrow`."""
        val = {}
        for m, nm in enumerate(base_names):
            val[((0, 0, 0), m)] = nm
            if nst and ((0, 0, 0), m) in exidx and ((0, 0, 0), m) in S:
                P.w("if (xp) xrow[%d] = %s;" % (exidx[((0, 0, 0), m)], nm))
        udef = {}
        tpos = {c: t for t, c in enumerate(TC)}
        # nodes are emitted level by level in chunks: first the chunk's cross-term loads (so they are all
        # in flight together and not ordered behind the exchange stores), then the arithmetic, then the
        # chunk's exchange stores
        chunk = options.geti("WARP_CHUNK", 8)
        levels = {}
        for (c, m) in nodes:
            levels.setdefault(sum(c), []).append((c, m))
        for level in sorted(levels):
            if nst and is_main:
                P.w("__syncwarp();")
            lv = levels[level]
            if is_main:      # emission order inside a level is free (a level reads only lower levels): knobs for the schedule search
                order = options.get("WARP_ORDER", "cm")
                if order == "mc":
                    lv = sorted(lv, key=lambda n: (n[1], kidx[n[0]]))
                elif order == "mcr":
                    lv = sorted(lv, key=lambda n: (-n[1], kidx[n[0]]))
                elif order == "ax":
                    lv = sorted(lv, key=lambda n: (reduction_axis(n[0]), kidx[n[0]], n[1]))
                elif order == "rev":
                    lv = lv[::-1]
                chs = options.get("WARP_CHUNKS", "") or WARP_CHUNKS.get(cls, "")
                if chs and Q == 1:
                    chunk = int(chs.split(",")[min(level, len(chs.split(","))) - 1])
            prefetch = options.flag("WARP_PREFETCH") and is_main
            parts = [lv[c0:c0 + chunk] for c0 in range(0, len(lv), chunk)]
            xname = {}

            def emit_loads(part):
                if not nst:
                    return
                for (c, m) in part:
                    i = reduction_axis(c)
                    c1 = sub1(c, i)
                    xname[(c, m)] = "%sx%d_%d" % (vp, kidx[c], m)
                    if is_main:
                        P.w("const double %s = xb%d[%d];" % (xname[(c, m)], i, exidx[(c1, m + 1)]))
                    else:      # lower pass: the few lower lanes exchange by shuffle
                        P.w("const double %s = __shfl_sync(FULL, %s, lsrc%d);" % (xname[(c, m)], val[(c1, m + 1)], i))

            if prefetch and parts:
                emit_loads(parts[0])
            for pi, part in enumerate(parts):
                if prefetch:
                    if pi + 1 < len(parts):
                        emit_loads(parts[pi + 1])      # next chunk's cross terms in flight during this chunk's arithmetic
                else:
                    emit_loads(part)
                stores = []
                for (c, m) in part:
                    i = reduction_axis(c)
                    c1 = sub1(c, i)
                    n2 = c1[i]
                    nm = "%s%d_%d" % (vp, kidx[c], m)
                    # a top-level ket target has no consumer: fold the contraction add (Alg. 2 line 7) into its FMAs
                    leaf = is_main and m == 0 and c in tpos and sum(c) == ctop and (c, m) not in exidx and tpos[c] < nacc_reg
                    if leaf:
                        nm = "acc%d" % tpos[c]
                        P.w("%s = fma(QC%d, %s, %s);" % (nm, i, val[(c1, m)], nm))
                    else:
                        P.w("double %s = QC%d * %s;" % (nm, i, val[(c1, m)]))
                    P.w("%s = fma(WQ%d, %s, %s);" % (nm, i, val[(c1, m + 1)], nm))
                    if n2:
                        c2 = sub1(c1, i)
                        ukey = (c2, m)
                        if ukey not in udef:
                            un = "%su%d_%d" % (vp, kidx[c2], m)
                            P.w("const double %s = fma(-re, %s, %s);" % (un, val[(c2, m + 1)], val[(c2, m)]))
                            udef[ukey] = un
                        P.w("%s = fma(hen%d, %s, %s);" % (nm, n2, udef[ukey], nm))
                    if nst:
                        P.w("%s = fma(ka%d, %s, %s);" % (nm, i, xname[(c, m)], nm))
                        if (c, m) in exidx:
                            stores.append("if (xp) xrow[%d] = %s;" % (exidx[(c, m)], nm))
                    val[(c, m)] = nm
                    if is_main and m == 0 and c in tpos and not leaf:
                        P.w("%s += %s;" % (A(tpos[c]), nm))
                for st in stores:
                    P.w(st)
        return val

    def load_ket_consts():
        # QC0 QC1 | QC2 WQ0 | WQ1 WQ2 | he*0 he*1 | ... | rho/eta : 16-byte broadcast loads
        nd = OFF_RE + 1 - OFF_QC
        names = ["QC0", "QC1", "QC2", "WQ0", "WQ1", "WQ2"] + ["hen%d" % n for n in range(ctop + 1)] + ["re"]
        assert len(names) == nd and OFF_WQ == OFF_QC + 3 and OFF_HEN == OFF_WQ + 3 and OFF_RE == OFF_HEN + ctop + 1
        if not pairs:
            for k, nm_ in enumerate(names):
                P.w("const double %s = pr[%d];" % (nm_, OFF_QC + k))
        for k in (range(0, nd, 2) if pairs else []):
            P.w("const double2 kc%d = *reinterpret_cast<const double2 *>(pr + %d);" % (k, OFF_QC + k))
            P.w("const double %s = kc%d.x;" % (names[k], k))
            if k + 1 < nd:
                P.w("const double %s = kc%d.y;" % (names[k + 1], k))

    # ---------------- lower pass
    P.w("for (int l0 = 0; l0 < cntw; l0 += %s) {" % ("PB" if nLow else "PBS"))
    P.ind += 1
    P.w("const int cntl = min(%s, cntw - l0);" % ("PB" if nLow else "PBS"))
    if use_pyr:
        pyr, f_need = bra_pyramid(nst, ctop)
        ALLC = LW + T
        rotn = lambda a, r: a if r == 0 else rotn((a[2], a[0], a[1]), r - 1)     # noqa: E731
        P.w("{   // bra pass: lane = (primitive jj, axis rotation r): pure-bra vertices [a0|00]^(m) of every component")
        P.ind += 1
        P.w("const int jj = min(lane / 3, cntl - 1), r = lane % 3;")
        P.w("const double *pr = %s + (l0 + jj) * PRS;" % ("REC" if grouped else "S1"))
        P.w("double *bt = S1 + OFF_BT + jj * BTS;")
        P.w("const int ax0 = %d + r, ax1 = %d + (r + 1) %% 3, ax2 = %d + (r + 2) %% 3;   // rotated axes" % (OFF_PA, OFF_PA, OFF_PA))
        P.w("const double pa0 = pr[ax0], pa1 = pr[ax1], pa2 = pr[ax2], wp0 = pr[ax0 + 4], wp1 = pr[ax1 + 4], wp2 = pr[ax2 + 4];")
        P.w("const double rz = pr[%d];" % OFF_RZ)
        pname = {(0, 0, 0): ["pr[%d]" % m for m in range(f_need + 1)]}
        for m in range(ctop + 1):
            P.w("bt[%d] = pr[%d];" % (ALLC.index((0, 0, 0)) * (ctop + 1) + m, m))
        for k, (rep_, i, par, n, gp, mmax) in enumerate(pyr):
            offs = [ALLC.index(rotn(rep_, r)) * (ctop + 1) for r in range(3)]
            P.w("const int po%d = r == 0 ? %d : (r == 1 ? %d : %d);" % (k, offs[0], offs[1], offs[2]))
            names = []
            for m in range(mmax + 1):
                nm = "py%d_%d" % (k, m)
                P.w("double %s = fma(wp%d, %s, pa%d * %s);" % (nm, i, pname[par][m + 1], i, pname[par][m]))
                if n:
                    P.w("%s = fma(pr[%d], fma(-rz, %s, %s), %s);" % (nm, OFF_HZN + n, pname[gp][m + 1], pname[gp][m], nm))
                if m <= ctop:
                    P.w("bt[po%d + %d] = %s;" % (k, m, nm))
                names.append(nm)
            pname[rep_] = names
        P.ind -= 1
        P.w("}")
        P.w("__syncwarp();")
    if nLow:
        P.w("{   // lower pass: lane = (primitive jj, lower component)")
        P.ind += 1
        P.w("const int jj = min(TL(6), cntl - 1);")
        P.w("const double *pr = %s + (l0 + jj) * PRS;" % ("REC" if grouped else "S1"))
        P.w("const int lsrc0 = lane - gl + TL(3), lsrc1 = lane - gl + TL(4), lsrc2 = lane - gl + TL(5);")
        P.w("const bool xp = TL(7) >= 0;      // only level la-1 components are read by the target lanes")
        P.w("double *xrow = S1 + OFF_LOW + TL(7);")
        P.w("const double ka0 = pr[%d + TL(0)], ka1 = pr[%d + TL(1)], ka2 = pr[%d + TL(2)];" % (OFF_HZEN, OFF_HZEN, OFF_HZEN))
        for s in range(nstl):
            P.w("const int lsel%d = TL(%d), lnix%d = %d + TL(%d);" % (s + 1, 8 + s, s + 1, OFF_HZN, 8 + nstl + s))
        if use_pyr:
            P.w("const double *bt = S1 + OFF_BT + jj * BTS + (gl %% NLOW) * %d;" % (ctop + 1))
            base = ["bt[%d]" % m for m in range(mb_low + 1)]
        else:
            base = emit_chain(nstl, mb_low, "lsel", "lnix", "lb")
        if ctop >= 1 and low_nodes:
            load_ket_consts()
        emit_ket(low_nodes, base, S_low, False, "lv")
        P.ind -= 1
        P.w("}")
        P.w("__syncwarp();")
    # ---------------- main passes
    if jnest:
        P.w("for (int jh = 0; jh < cntl; jh += 4) {       // lower tables in runs of four: (jj >> 2) * JSTH + (jj & 3) * JST")
        P.w("const int cn4 = min(4, cntl - jh);")
        P.w("for (int j4 = 0; j4 < cn4; ++j4) {")
        P.ind += 1
        P.w("const int jj = jh + j4;")
    else:
        P.w("for (int jj = 0; jj < cntl; ++jj) {")
        P.ind += 1
    P.w("const double *pr = %s + (l0 + jj) * PRS;" % ("REC" if grouped else "S1"))
    if nst:
        if jnest:
            P.w("const int jo = (jh >> 2) * %d + j4 * JST;" % JSTH)
            P.w("const double *xb0 = S1 + xo0 + jo * xl0, *xb1 = S1 + xo1 + jo * xl1, *xb2 = S1 + xo2 + jo * xl2;")
        else:
            P.w("const double *xb0 = S1 + xo0 + jj * xl0, *xb1 = S1 + xo1 + jj * xl1, *xb2 = S1 + xo2 + jj * xl2;")
        P.w("double *xrow = S1 + OFF_XM + gl * NEXS;")
        P.w("const bool xp = gl < %d;       // only lanes below the top bra level are cross-term sources" % nexp)
        P.w("const double ka0 = pr[kax0], ka1 = pr[kax1], ka2 = pr[kax2];")
    if use_pyr:
        P.w("const double *bt = S1 + OFF_BT + jj * BTS + (NLOW + (gl < %d ? gl : 0)) * %d;" % (nT, ctop + 1))
        base = ["bt[%d]" % m for m in range(ctop + 1)]
    else:
        base = emit_chain(nst, ctop, "sel", "nix", "b")
    if ctop >= 1:
        load_ket_consts()
    tpos = {c: t for t, c in enumerate(TC)}
    if (0, 0, 0) in tpos:
        P.w("%s += %s;" % (A(tpos[(0, 0, 0)]), base[0]))
    emit_ket(main_nodes, base, S_main, True, "v")
    P.ind -= 1
    P.w("}")
    if jnest:
        P.w("}")
    P.w("__syncwarp();")
    P.ind -= 1
    P.w("}")
    P.ind -= 1
    P.w("}")
    # ---------------- Phase 2
    P.w("// Phase 2: H -> shared, bra HRR + Ta,Tb per ket column, ket HRR + Tc,Td per bra row")
    P.w("if (gl < %d) {" % nT)
    P.ind += 1
    for t in range(nC):
        P.w("SA[gl * %d + %d] = %s;" % (HS, t, A(t)))
    P.ind -= 1
    P.w("}")
    P.w("__syncwarp();")
    if fock:
        # the density sub-blocks are fetched NOW (the accumulators have just died, registers are free) and parked in shared memory after
        # Phase 2: their L2 / HBM latency hides behind the bra and ket programs instead of stalling the epilogue
        nsa = 2 * la + 1
        DPF = (DSZ + G - 1) // G
        P.w("const int oa = a.bf_off[sh0], ob = a.bf_off[sh1], oc = a.bf_off[sh2], od = a.bf_off[sh3];")
        P.w("const int64_t nbf = a.nbf;")
        P.w("double dpf[%d];" % DPF)
        P.w("#pragma unroll")
        P.w("for (int k = 0; k < %d; ++k) {" % DPF)
        P.w("    const int e = gl + k * G;")
        P.w("    int r = 0, c = 0;")
        segs = ((nCD, "oc", "od", 2 * ld + 1), (nAB, "oa", "ob", 2 * lb + 1), ((2 * lb + 1) * (2 * ld + 1), "ob", "od", 2 * ld + 1),
                (nsa * (2 * ld + 1), "oa", "od", 2 * ld + 1), ((2 * lb + 1) * (2 * lc + 1), "ob", "oc", 2 * lc + 1), (nsa * (2 * lc + 1), "oa", "oc", 2 * lc + 1))
        for si, (cnt, o1, o2, n2) in enumerate(segs):
            P.w("    %sif (e < %d) { r = %s + (e - %d) / %d; c = %s + (e - %d) %% %d; }" % ("else " if si else "", DOFF[si] + cnt, o1, DOFF[si], n2, o2, DOFF[si], n2))
        P.w("    dpf[k] = e < %d ? __ldg(a.D + r * nbf + c) : 0.0;" % DSZ)
        P.w("}")
    P.w("const double AB0 = RA[0] - RB[0], AB1 = RA[1] - RB[1], AB2 = RA[2] - RB[2];")
    P.w("const double CD0 = RC[0] - RD[0], CD1 = RC[1] - RD[1], CD2 = RC[2] - RD[2];")
    P.w("for (int c0 = 0; c0 < %d; c0 += G) {" % nC)
    P.ind += 1
    P.w("const int col = c0 + gl;")
    P.w("if (col < %d) {" % nC)
    P.ind += 1
    emit_lin(P, bra, lambda k: "SA[%d + col]" % (k * HS), "h", ["AB0", "AB1", "AB2"])
    for r, s in enumerate(bra.outputs):
        P.w("S1[%d + col] = h%d;" % (r * HS, s))
    P.ind -= 1
    P.w("}")
    P.ind -= 1
    P.w("}")
    P.w("__syncwarp();")
    P.w("for (int r0 = 0; r0 < %d; r0 += G) {" % nABc)
    P.ind += 1
    P.w("const int row = r0 + gl;")
    P.w("if (row < %d) {" % nABc)
    P.ind += 1
    emit_lin(P, ket, lambda k: "S1[row * %d + %d]" % (HS, k), "g", ["CD0", "CD1", "CD2"])
    for r, s in enumerate(ket.outputs):
        P.w("SA[row * %d + %d] = g%d;" % (nCD, r, s))
    P.ind -= 1
    P.w("}")
    P.ind -= 1
    P.w("}")
    P.w("__syncwarp();")
    if late is not None:
        P.w("for (int c0 = 0; c0 < %d; c0 += G) {      // deferred Ta (x) Tb on the Cartesian bra rows, per output column" % nCD)
        P.ind += 1
        P.w("const int col = c0 + gl;")
        P.w("if (col < %d) {" % nCD)
        P.ind += 1
        emit_lin(P, late, lambda k: "SA[%d + col]" % (k * nCD), "t", ["0", "0", "0"])
        for r, s_ in enumerate(late.outputs):
            P.w("S1[%d + col] = t%d;" % (r * nCD, s_))
        P.ind -= 1
        P.w("}")
        P.ind -= 1
        P.w("}")
        P.w("__syncwarp();")
    P.w("const double *OB = %s;                  // the finished spherical block" % ("S1" if late is not None else "SA"))
    nsb, nsc, nsd = 2 * lb + 1, 2 * lc + 1, 2 * ld + 1
    if fock:
        # J/K digestion of the block where it lies (formulas: csrc/jk_digest.cu): the G lanes of the quartet share the
        # output elements; every element is a short dot product -> one atomicAdd per OUTPUT element.  nsph is odd, so a lane-per-row
        # walk of the [nAB][nCD] block (stride nCD) is free of bank conflicts.
        nsa = 2 * la + 1
        P.w("{")
        P.ind += 1
        P.w("double *DS = S1;                         // density sub-blocks (the B region is free now)")
        P.w("#pragma unroll")
        P.w("for (int k = 0; k < %d; ++k) if (gl + k * G < %d) DS[gl + k * G] = dpf[k];" % (DPF, DSZ))
        P.w("const bool adds = qvalid && lane < Q * G;      // spare lanes (Q = 3: lanes 30, 31) shadow a real lane: they must not repeat its atomics")
        P.w("double wq = 1.0;")
        P.w("if (sh0 == sh1) wq *= 0.5;")
        P.w("if (sh2 == sh3) wq *= 0.5;")
        P.w("if (sh0 == sh2 && sh1 == sh3) wq *= 0.5;")
        P.w("__syncwarp();")
        P.w("for (int e = gl; e < %d; e += G) {          // Jt_ab += 2w sum_cd D_cd I" % nAB)
        P.w("    double s = 0.0;")
        P.w("    #pragma unroll")
        P.w("    for (int t = 0; t < %d; ++t) s = fma(DS[%d + t], OB[e * %d + t], s);" % (nCD, DOFF[0], nCD))
        P.w("    if (adds) atomicAdd(a.Jt + (oa + e / %d) * nbf + ob + e %% %d, 2.0 * wq * s);" % (nsb, nsb))
        P.w("}")
        P.w("for (int t = gl; t < %d; t += G) {          // Jt_cd += 2w sum_ab D_ab I" % nCD)
        P.w("    double s = 0.0;")
        P.w("    #pragma unroll")
        P.w("    for (int e = 0; e < %d; ++e) s = fma(DS[%d + e], OB[e * %d + t], s);" % (nAB, DOFF[1], nCD))
        P.w("    if (adds) atomicAdd(a.Jt + (oc + t / %d) * nbf + od + t %% %d, 2.0 * wq * s);" % (nsd, nsd))
        P.w("}")
        for (nm, n1, n2, o1, o2, doff, idx, cmt) in (
                ("ac", nsa, nsc, "oa", "oc", DOFF[2], "((i1 * %d + j1) * %d + i2) * %d + j2" % (nsb, nsc, nsd), "Kt_ac += w sum_bd D_bd I"),
                ("ad", nsa, nsd, "oa", "od", DOFF[4], "((i1 * %d + j1) * %d + j2) * %d + i2" % (nsb, nsc, nsd), "Kt_ad += w sum_bc D_bc I"),
                ("bc", nsb, nsc, "ob", "oc", DOFF[3], "((j1 * %d + i1) * %d + i2) * %d + j2" % (nsb, nsc, nsd), "Kt_bc += w sum_ad D_ad I"),
                ("bd", nsb, nsd, "ob", "od", DOFF[5], "((j1 * %d + i1) * %d + j2) * %d + i2" % (nsb, nsc, nsd), "Kt_bd += w sum_ac D_ac I")):
            m1 = nsb if nm[0] == "a" else nsa          # summed indices (j1, j2): the two NOT in the output pair; D block [m1][m2]
            m2 = nsd if nm[1] == "c" else nsc
            P.w("for (int e = gl; e < %d; e += G) {          // %s" % (n1 * n2, cmt))
            P.w("    const int i1 = e / %d, i2 = e %% %d;" % (n2, n2))
            P.w("    double s = 0.0;")
            P.w("    #pragma unroll")
            P.w("    for (int j1 = 0; j1 < %d; ++j1) {" % m1)
            P.w("        #pragma unroll")
            P.w("        for (int j2 = 0; j2 < %d; ++j2) s = fma(DS[%d + j1 * %d + j2], OB[%s], s);" % (m2, doff, m2, idx))
            P.w("    }")
            P.w("    if (adds) atomicAdd(a.Kt + (%s + i1) * nbf + %s + i2, wq * s);" % (o1, o2))
            P.w("}")
        P.ind -= 1
        P.w("}")
    else:
        P.w("double *out = a.out + q * a.out_stride;")
        P.w("if (qvalid && canon) {                 // caller order == canonical order: plain coalesced copy")
        P.w("    for (int e = gl; e < %d; e += G) out[e] = OB[e];" % (nAB * nCD))
        P.w("} else if (qvalid)")
        P.w("for (int e = gl; e < %d; e += G) {" % (nAB * nCD))
        P.w("    const int id = e %% %d, ic = (e / %d) %% %d, ib = (e / %d) %% %d, ia = e / %d;"
            % (nsd, nsd, nsc, nsd * nsc, nsb, nsd * nsc * nsb))
        P.w("    out[ia * a.ostride[0] + ib * a.ostride[1] + ic * a.ostride[2] + id * a.ostride[3]] = OB[e];")
        P.w("}")
    P.w("__syncwarp();")
    if grouped:
        P.w("}   // quartets of the group")
    P.w("}   // quartet loop")
    P.ind = 0
    P.w("}")
    P.w("#undef TM")
    P.w("#undef TL")
    P.w("}  // namespace w%s" % tag)
    P.w("static cudaError_t rcg_launch_warp_%s(const RcgLaunch &a)" % tag)
    P.w("{")
    P.w("    using namespace w%s;" % tag)
    P.w("    const size_t smem = sizeof(double) * (WSM * Q * WARPS + %d);" % TABD)
    P.w("    static RcgOnce once;              // shared-memory limit raised once per device (thread-safe), SM count cached")
    P.w("    int nsm = 0;")
    P.w("    cudaError_t e = rcg_prepare_kernel(once, (const void *)rcg_eri_warp_%s, smem, &nsm);" % tag)
    P.w("    if (e != cudaSuccess) return e;")
    P.w("    int64_t blocks = (a.n + WARPS * Q - 1) / (WARPS * Q), cap = (int64_t)nsm * %d;   // persistent: one wave" % minblocks)
    P.w("    if (blocks > cap) blocks = cap;")
    P.w("    rcg_eri_warp_%s<<<(unsigned)blocks, WARPS * 32, smem, a.stream>>>(a);" % tag)
    P.w("    return cudaGetLastError();")
    P.w("}")
    meta = dict(warp_target_lanes=nT, warp_lower_components=nLow, warp_PB=PB, warp_ket_vertices=len(main_nodes),
                warp_lower_vertices=len(low_nodes), warp_smem_bytes_per_warp=WSM * 8, warp_accumulators_per_lane=nC)
    meta["warp_quartets_per_warp"] = Q
    return P.text() + "\n", "rcg_launch_warp_%s" % tag, meta, Q


def emit_class(cls, fock=False):
    """One-quartet-per-warp kernel, plus (light bra sides) a packed kernel with Q quartets per warp.
    The packed one is used when the batch is large and the contraction depths of the shells involved
    are uniform enough (all groups of a warp loop to the largest K4 among them): launcher below."""
    t1, sym1, meta, _ = _emit_variant(cls, 1, "")
    tq, symq, metaq, Q = _emit_variant(cls, 0, "p")
    strip = lambda t: t.replace('#include "rcg_device.cuh"\n', "")      # noqa: E731
    tag = "%d%d%d%d" % cls
    ftext = ""
    if fock:     # the same kernels with the J/K digestion as their epilogue (rcg_fock_batch)
        f1, fsym1, _, _ = _emit_variant(cls, 1, "f", fock=True)
        ftext = strip(f1)
        fl = ["cudaError_t rcg_launch_fock_warp_%s(const RcgLaunch &a)" % tag, "{"]
        if Q > 1:
            fq, fsymq, _, _ = _emit_variant(cls, 0, "pf", fock=True)
            ftext += strip(fq)
            fl += ["    int nsm = 0;", "    cudaError_t e = rcg_sm_count(&nsm);", "    if (e != cudaSuccess) return e;",
                   "    double spread = 1.0;", "    for (int k = 0; k < 4; ++k) spread *= (double)a.kmax[a.lcan[k]] / (double)a.kmin[a.lcan[k]];",
                   "    if (a.n >= (int64_t)nsm * 8 * %d && (spread <= 1.3 || a.uniform_k4)) return %s(a);      // even lists: Q quartets per warp" % (Q, fsymq)]
        fl += ["    return %s(a);" % fsym1, "}"]
        ftext += "static " + "\n".join(fl) + "\n"
        meta["warp_fock_launcher"] = "rcg_launch_fock_warp_%s" % tag
    if Q == 1:
        return t1 + ftext, sym1, meta
    meta["warp_packed_quartets_per_warp"] = Q
    disp = []
    disp.append("static cudaError_t rcg_launch_warp_%s_auto(const RcgLaunch &a)" % tag)
    disp.append("{")
    disp.append("    int nsm = 0;")
    disp.append("    cudaError_t e = rcg_sm_count(&nsm);")
    disp.append("    if (e != cudaSuccess) return e;")
    disp.append("    if (a.n < (int64_t)nsm * 8 * %d) return %s(a);        // too few quartets to fill the SMs when packed" % (Q, sym1))
    disp.append("    double spread = 1.0;      // bound on max K4 / min K4 over the quartets of this class in this basis")
    disp.append("    for (int k = 0; k < 4; ++k) spread *= (double)a.kmax[a.lcan[k]] / (double)a.kmin[a.lcan[k]];")
    disp.append("    if (spread <= 1.3 || a.uniform_k4) return %s(a);      // uniform contraction (or the caller's promise of one K4): always packed" % symq)
    disp.append("    // variable contraction depths: a statistics pass measures the padding the packed grouping (Q consecutive")
    disp.append("    // quartets loop to their largest K4) would cost on THIS list; both kernels are enqueued and the one")
    disp.append("    // that loses the device-side test returns at once (no host synchronisation)")
    disp.append("    RcgLaunch b = a;")
    disp.append("    e = rcg_pack_stats(a, %d, 0, &b.stat);" % Q)
    disp.append("    if (e != cudaSuccess) return e;")
    disp.append("    e = %s(b);" % symq)
    disp.append("    return e != cudaSuccess ? e : %s(b);" % sym1)
    disp.append("}")
    return t1 + strip(tq) + ftext + "\n".join(disp) + "\n", "rcg_launch_warp_%s_auto" % tag, meta


def emit_class_swapped(cls, fock=False):
    """kernel generated for the swapped quartet (lc ld|la lb); the launcher swaps the roles of the index
    pairs (quartet columns, output strides) so that the caller sees class `cls`."""
    la, lb, lc, ld = cls
    text, sym, meta = emit_class((lc, ld, la, lb), fock=fock)
    tag = "%d%d%d%d" % cls
    w = []
    w.append("static cudaError_t rcg_launch_warp_%s_swapped(const RcgLaunch &a)" % tag)
    w.append("{")
    w.append("    RcgLaunch b = a;      // (ab|cd) = (cd|ab): the kernel's bra is this class's ket")
    w.append("    for (int k = 0; k < 4; ++k) {")
    w.append("        const int s = (k + 2) & 3;")
    w.append("        b.perm[k] = a.perm[s]; b.nsph[k] = a.nsph[s]; b.lcan[k] = a.lcan[s]; b.ostride[k] = a.ostride[s];")
    w.append("    }")
    w.append("    return %s(b);" % sym)
    w.append("}")
    meta["warp_swapped"] = True
    if fock:      # (ab|cd) -> (cd|ab) maps Jt_ab <-> Jt_cd and Kt_ac -> Kt_ca, ...: the same J and K after rcg_jk_finish's symmetrisation
        inner = meta["warp_fock_launcher"]
        w += ["static cudaError_t rcg_launch_fock_warp_%s_swapped(const RcgLaunch &a)" % tag, "{",
              "    RcgLaunch b = a;", "    for (int k = 0; k < 4; ++k) { const int s = (k + 2) & 3; b.perm[k] = a.perm[s]; b.nsph[k] = a.nsph[s]; b.lcan[k] = a.lcan[s]; }",
              "    return %s(b);" % inner, "}"]
        meta["warp_fock_launcher"] = "rcg_launch_fock_warp_%s_swapped" % tag
    return text + "\n".join(w) + "\n", "rcg_launch_warp_%s_swapped" % tag, meta
