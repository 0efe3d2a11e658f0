"""Emit the global-scratch tier (RCG_TIER_GLOBAL) tables of one class.

The paper's Tier 2 keeps intermediates in an interleaved global buffer, slot-major and
thread-minor, so that a warp's accesses coalesce.  Here that tier is a
table-driven kernel (csrc/tier_global.cu): the generator writes the recurrence graph as data --
one record per vertex FAMILY (a,c) covering its contiguous range of Boys orders m -- instead of
unrolled code, because unrolled (gg|gg) does not compile.

VRR family record, 5 x uint32 (vertex [a|c]^(m) lives in slot off_dst + m):
  w0 off_dst   w1 off1 (parents p1 = off1+m, p2 = off1+m+1)   w2 off3 (p3 = off3+m, p4 = off3+m+1)
  w3 off5 (cross parent p5 = off5+m+1)
  w4 mlo | nm<<5 | side<<10 (0 bra, 1 ket) | axis<<11 | n2<<13 | ncross<<17
Phase-2 node record (dst <- sum_k coef_k * src_k), level-sorted: w0 dst | nterms<<16, then per term
  src | coefsel<<16; coefsel 0: 1.0; 1..3: displacement X_x,X_y,X_z; >=4: consts[coefsel-4].
"""
from .graph import VrrGraph, hrr_c2s_program, class_flops, peak_live, dsa_order, slot_allocation


def vrr_families(g):
    fam = {}
    for k in g.order:
        a, c, m = k
        fam.setdefault((a, c), []).append(m)
    # topological order of families: a family depends on families with smaller |a|+|c|.
    keys = sorted(fam.keys(), key=lambda ac: (sum(ac[0]) + sum(ac[1]), sum(ac[1]), ac))
    # slot allocation by lifetime (the paper's slot packing, in its simplest exact form):
    # a vertex of level l=|a|+|c| is read only by levels l+1 and l+2 (and, if it is a target, by the
    # contraction right after its own level), so three rotating level buffers suffice.
    base = {}
    recs = []
    lev_of = lambda ac: sum(ac[0]) + sum(ac[1])      # noqa: E731
    lev_size = {}
    for ac in keys:
        lev_size[lev_of(ac)] = lev_size.get(lev_of(ac), 0) + len(fam[ac])
    bufsz = max(lev_size.values())
    fill = {}
    for ac in keys:
        ms = sorted(fam[ac])
        assert ms == list(range(ms[0], ms[-1] + 1)), "non-contiguous Boys orders in a family"
        lv = lev_of(ac)
        start = (lv % 3) * bufsz + fill.get(lv, 0)
        fill[lv] = fill.get(lv, 0) + len(ms)
        base[ac] = (start - ms[0], ms[0], len(ms))       # off, mlo, nm
    nslots = 3 * bufsz
    unpacked = sum(lev_size.values())
    assert keys[0] == ((0, 0, 0), (0, 0, 0)) and base[keys[0]][0] == 0
    for ac in keys[1:]:
        off, mlo, nm = base[ac]
        n = g.nodes[(ac[0], ac[1], mlo)]
        for m in range(mlo, mlo + nm):     # same structure for every m of the family
            nn = g.nodes[(ac[0], ac[1], m)]
            assert (nn.side, nn.axis, nn.n2, nn.ncross) == (n.side, n.axis, n.n2, n.ncross)
        off1 = base[(n.p1[0], n.p1[1])][0]
        off3 = base[(n.p3[0], n.p3[1])][0] if n.p3 is not None else 0
        off5 = base[(n.p5[0], n.p5[1])][0] if n.p5 is not None else 0
        # parents must exist for every m of the range
        for m in range(mlo, mlo + nm):
            for (pac, pm) in (((n.p1[0], n.p1[1]), m), ((n.p1[0], n.p1[1]), m + 1)):
                o, lo, cnt = base[pac]
                assert lo <= pm < lo + cnt
        off_w = off & 0xffffffff                        # may be negative when mlo > start; stored as two's complement
        meta = mlo | (nm << 5) | ((1 if n.side == "ket" else 0) << 10) | (n.axis << 11) | (n.n2 << 13) | (n.ncross << 17)
        recs.append((off_w, off1 & 0xffffffff, off3 & 0xffffffff, off5 & 0xffffffff, meta))
    # families of one level |a|+|c| are independent of each other: [start index of level l] for the
    # warp-parallel kernel (parents lie one or two levels below)
    lvl_off = [0]
    lv = [sum(ac[0]) + sum(ac[1]) for ac in keys[1:]]
    for i in range(1, len(lv)):
        if lv[i] != lv[i - 1]:
            lvl_off.append(i)
    lvl_off.append(len(lv))
    # targets grouped by level: contracted right after their level is complete
    tg = sorted(((lev_of((a, c)), t, base[(a, c)][0]) for t, (a, c, _) in enumerate(g.targets())))
    for (a, c, _) in g.targets():
        assert base[(a, c)][1] == 0
    maxlev = max(lev_size)
    tgt_off = [0]
    for lv in range(0, maxlev + 1):
        tgt_off.append(tgt_off[-1] + sum(1 for x in tg if x[0] == lv))
    while len(tgt_off) < len(lvl_off) + 1:
        tgt_off.append(tgt_off[-1])
    tslots = [x[2] for x in tg]
    tindex = [x[1] for x in tg]
    assert len(lvl_off) - 1 == maxlev or len(keys) == 1
    return recs, (tslots, tindex, tgt_off), nslots, lvl_off, unpacked


def pack_nodes(prog, consts):
    """Phase-2 program as level-sorted NODES for the warp-parallel kernel: node = dst <- sum_k coef_k * src_k.
    Returns (words, node_off, lvl_off): words = per node [dst | nterms<<16, then src | coefsel<<16 per term];
    node_off[n] = first word of node n; nodes [lvl_off[l], lvl_off[l+1]) are independent (inputs = level 0)."""
    nodes = []
    for (dst, src, coef, init) in prog.ops:
        if coef[0] == "one":
            sel = 0
        elif coef[0] == "x":
            sel = 1 + coef[1]
        else:
            v = coef[1]
            if v not in consts:
                consts[v] = len(consts)
            sel = 4 + consts[v]
        if init:
            nodes.append([dst, [(src, sel)]])
        else:
            assert nodes[-1][0] == dst
            nodes[-1][1].append((src, sel))
    level = {k: 0 for k in range(prog.nin)}
    for dst, terms in nodes:
        level[dst] = 1 + max(level[s_] for s_, _ in terms)
    nodes.sort(key=lambda n: level[n[0]])
    words, node_off, lvl_off = [], [], [0]
    for i, (dst, terms) in enumerate(nodes):
        if i and level[dst] != level[nodes[i - 1][0]]:
            lvl_off.append(i)
        node_off.append(len(words))
        assert dst < 65536 and len(terms) < 65536
        words.append(dst | (len(terms) << 16))
        for (src, sel) in terms:
            assert src < 65536 and sel < 65536
            words.append(src | (sel << 16))
    lvl_off.append(len(nodes))
    return words, node_off, lvl_off


def pack_program(prog, consts):
    words = []
    for (dst, src, coef, init) in prog.ops:
        if coef[0] == "one":
            sel = 0
        elif coef[0] == "x":
            sel = 1 + coef[1]
        else:
            v = coef[1]
            if v not in consts:
                consts[v] = len(consts)
            sel = 4 + consts[v]
        assert dst < 65536 and src < 65536 and sel < 65536
        words.append(((dst << 16) | src, sel | ((1 if init else 0) << 16)))
    return words


def _arr(name, ctype, vals, per_line=8, fmt="%s"):
    lines = ["static const %s %s[] = {" % (ctype, name)]
    vals = list(vals) or [0]
    for i in range(0, len(vals), per_line):
        lines.append("  " + ",".join(fmt % v for v in vals[i:i + per_line]) + ",")
    lines.append("};")
    return "\n".join(lines)


def class_tag(cls):
    return "%d%d%d%d" % cls


def emit_class(cls, tier, launch_symbol=None, extra_decl="", ws_quartet_doubles=0, fock_symbol=None):
    la, lb, lc, ld = cls
    g = VrrGraph(la, lb, lc, ld)
    recs, (tslots, tindex, tgt_off), nv, lvl_off, unpacked = vrr_families(g)
    bra = hrr_c2s_program(la, lb)
    ket = hrr_c2s_program(lc, ld)
    consts = {}
    bw, bno, blo = pack_nodes(bra, consts)
    kw, kno, klo = pack_nodes(ket, consts)
    fp, fq = class_flops(la, lb, lc, ld, g)
    pl_default = peak_live(g, g.order)
    pl_dsa = peak_live(g, dsa_order(g)) if g.num_nodes() <= 20000 else -1
    tag = class_tag(cls)
    src = []
    src.append("// GENERATED by paper_2605_10312_b200/gen/generate.py -- do not edit.")
    src.append("// class (%d %d|%d %d): %d VRR vertices in %d families, %d targets, PeakLive(post-order)=%d, PeakLive(DSA)=%d"
               % (la, lb, lc, ld, g.num_nodes(), len(recs), len(tslots), pl_default, pl_dsa))
    src.append('#include "rcg_internal.h"')
    src.append("namespace {")
    src.append(_arr("vrr_fam", "uint32_t", [w for r in recs for w in r], 10, "0x%xu"))
    src.append(_arr("tslots", "int32_t", tslots, 16, "%d"))
    src.append(_arr("tindex", "int32_t", tindex, 16, "%d"))
    src.append(_arr("tgt_off", "int32_t", tgt_off, 16, "%d"))
    src.append(_arr("lvl_off", "int32_t", lvl_off, 16, "%d"))
    src.append(_arr("bra_ops", "uint32_t", bw, 10, "0x%xu"))
    src.append(_arr("bra_noff", "int32_t", bno, 16, "%d"))
    src.append(_arr("bra_loff", "int32_t", blo, 16, "%d"))
    src.append(_arr("ket_ops", "uint32_t", kw, 10, "0x%xu"))
    src.append(_arr("ket_noff", "int32_t", kno, 16, "%d"))
    src.append(_arr("ket_loff", "int32_t", klo, 16, "%d"))
    src.append(_arr("bra_out", "uint16_t", bra.outputs, 16, "%d"))
    src.append(_arr("ket_out", "uint16_t", ket.outputs, 16, "%d"))
    cvals = [v for v, _ in sorted(consts.items(), key=lambda kv: kv[1])]
    src.append(_arr("consts", "double", cvals, 4, "%.17g"))
    src.append("}  // namespace")
    if extra_decl:
        src.append(extra_decl)
    src.append("extern const RcgClassDesc rcg_class_%s = {" % tag)
    src.append("  {%d,%d,%d,%d}, %d, %dLL, %dLL, %d, %d," % (la, lb, lc, ld, tier, fp, fq, g.num_nodes(), min(p for p in (pl_default, pl_dsa) if p > 0)))
    src.append("  { vrr_fam, %d, lvl_off, %d, tslots, tindex, tgt_off, %d, %d, %d, %d," % (len(recs), len(lvl_off) - 1, len(tslots), len(g.target_a), len(g.target_c), nv))
    src.append("    bra_ops, %d, bra_noff, %d, bra_loff, %d, %d, %d, bra_out, %d," % (len(bw), len(bno), len(blo) - 1, bra.nin, bra.nslots, len(bra.outputs)))
    src.append("    ket_ops, %d, ket_noff, %d, ket_loff, %d, %d, %d, ket_out, %d," % (len(kw), len(kno), len(klo) - 1, ket.nin, ket.nslots, len(ket.outputs)))
    src.append("    consts, %d }," % len(cvals))
    src.append("  %s, %s, %d, %dLL" % (launch_symbol or "nullptr", fock_symbol or "nullptr",
                                       0 if not fock_symbol else (1 if "fock_reg" in fock_symbol else 2), ws_quartet_doubles))
    src.append("};")
    meta = dict(cls=list(cls), tier=tier, vrr_vertices=g.num_nodes(), families=len(recs), targets=len(tslots),
                peaklive_postorder=pl_default, peaklive_dsa=pl_dsa, flops_per_prim_quartet=fp, flops_per_quartet=fq,
                vrr_slots=nv, vrr_slots_unpacked=unpacked, vrr_slots_serial_postorder=slot_allocation(g, g.order)[1],
                bra_nodes=len(bno), ket_nodes=len(kno))
    return "\n".join(src) + "\n", meta
