"""Host-side generator: graph builder, schedules, Phase-2 programs, tier choice, emitters.
CPU only.  What is checked is what the paper and the mathematics fix: counting facts (PAPER.md:189-191,
:253-255, :299), parent counts, the fusion identity Eq. (16) == Eq. (17)
(PAPER.md:231-235), the solid-harmonic rows of SURVEY 8(c) (the generator builds them by recursion, the
oracle by the closed form: two routes, compared here), and that every emitter variant is the same linear map."""
import json
import math
import os
import random

import numpy as np
import pytest

import oracle
from paper_2605_10312_b200.gen import emit_block, emit_register, tiers
from paper_2605_10312_b200.gen.emit_warp import Prog
from paper_2605_10312_b200.gen.graph import (VrrGraph, canonical_classes, dsa_order, hrr_c2s_program, peak_live,
                                              reduction_axis, sub1)
from paper_2605_10312_b200.gen.solid import c2s_rows, cart_comps, ncart

GEN = os.path.join(os.path.dirname(emit_block.__file__), "..", "csrc", "gen")


def test_counting_facts():
    # ncart(l) = (l+1)(l+2)/2, nsph = 2l+1; l = 4: 15 -> 9; 15^4 / 9^4 = 7.7
    assert [ncart(l) for l in range(5)] == [1, 3, 6, 10, 15]
    assert [len(c2s_rows(l)) for l in range(5)] == [1, 3, 5, 7, 9]
    assert round(15 ** 4 / 9 ** 4, 1) == 7.7
    # N_acc = prod(2 l_i + 1): (2,2,1,1) -> 225, (2,2,2,1) -> 375
    nacc = lambda cls: int(np.prod([2 * l + 1 for l in cls]))      # noqa: E731
    assert nacc((2, 2, 1, 1)) == 225 and nacc((2, 2, 2, 1)) == 375
    # 120 pair-canonical classes for lmax = 4 (reading R-CLASSN); this round generates l <= 3 + (gg|gg)
    assert len(canonical_classes(4, extra=())) == 120
    assert len(canonical_classes()) == 120 and (4, 4, 4, 4) in canonical_classes() and len(canonical_classes(3)) == 55
    # true Cartesian accumulator count (R-NACC): (sum_e ncart(e)) (sum_f ncart(f)); (dd|dd): 961, not 625
    g = VrrGraph(2, 2, 2, 2)
    assert len(g.target_a) * len(g.target_c) == 961


@pytest.mark.parametrize("cls", [(1, 1, 1, 1), (2, 2, 2, 2), (3, 1, 2, 0), (3, 3, 2, 1)])
def test_vrr_graph_invariants(cls):
    g = VrrGraph(*cls)
    pos = {k: i for i, k in enumerate(g.order)}
    for k in g.order:
        n = g.nodes[k]
        ps = g.parents(k)
        if n.side is None:
            assert not ps and n.a == (0, 0, 0) and n.c == (0, 0, 0)
            continue
        assert 2 <= len(ps) <= 5                       # "2-5 parents per node"
        assert all(pos[p] < pos[k] for p in ps)        # g.order is topological
        # axis rule as the TEXT states it: ket wholly before bra, z -> y -> x
        if sum(n.c) > 0:
            assert n.side == "ket" and n.axis == reduction_axis(n.c)
        else:
            assert n.side == "bra" and n.axis == reduction_axis(n.a)
        # Eq. (2): the first two parents differ by one Boys order; every parent sits on a lower level
        assert n.p1[:2] == n.p2[:2] and n.p2[2] == n.p1[2] + 1 == n.m + 1
        assert all(sum(p[0]) + sum(p[1]) < sum(n.a) + sum(n.c) for p in ps)
    for t in g.targets():
        assert t in g.nodes
    # both schedules are topological orders of the same vertex set; PeakLive (Eq. (4)) is at least the base values
    for order in (g.order, dsa_order(g)):
        assert sorted(order) == sorted(g.order)
        seen = set()
        for k in order:
            assert all(p in seen for p in g.parents(k))
            seen.add(k)
        assert peak_live(g, order) >= g.L + 1


def test_dddd_graph_size():
    # SURVEY 7.1 / 8(a) a3, from an independent probe during the survey: pruned ket-first graph of (dd|dd) has
    # 2,330 vertices incl. the 9 Boys values and 13,923 flops per primitive quartet; (pp|pp): 146 and 663
    g = VrrGraph(2, 2, 2, 2)
    assert g.num_nodes() + g.L + 1 == 2330 and g.flops()[0] == 13923
    g = VrrGraph(1, 1, 1, 1)
    assert g.num_nodes() + g.L + 1 == 146 and g.flops()[0] == 663
    g = VrrGraph(3, 3, 3, 3)
    assert g.num_nodes() + g.L + 1 == 16682 and g.flops()[0] == 111269


def _run_prog(prog, xin, X):
    val = dict(enumerate(xin))
    for (dst, src, coef, init) in prog.ops:
        c = 1.0 if coef[0] == "one" else (X[coef[1]] if coef[0] == "x" else coef[1])
        val[dst] = c * val[src] if init else val[dst] + c * val[src]
    return np.array([val[o] for o in prog.outputs])


def _dense_side(l1, l2, xin, X, T1, T2):
    """Eq. (17) side: materialise the full Cartesian (a b| block by the HRR of Eq. (3), THEN transform."""
    vals = {}
    k = 0
    for e in range(l1, l1 + l2 + 1):
        for a in cart_comps(e):
            vals[(a, (0, 0, 0))] = xin[k]
            k += 1

    def hrr(a, b):
        if (a, b) not in vals:
            i = max(j for j in range(3) if b[j] > 0)        # any axis is legal; deliberately not the generator's choice
            b1 = sub1(b, i)
            a1 = tuple(v + (1 if j == i else 0) for j, v in enumerate(a))
            vals[(a, b)] = hrr(a1, b1) + X[i] * hrr(a, b1)
        return vals[(a, b)]

    cart = np.array([[hrr(a, b) for b in cart_comps(l2)] for a in cart_comps(l1)])
    return (T1 @ cart @ T2.T).reshape(-1)


@pytest.mark.parametrize("l1,l2", [(0, 0), (1, 0), (1, 1), (2, 1), (2, 2), (3, 1), (3, 2), (3, 3), (4, 4)])
def test_phase2_programs_equal_materialise_then_transform(l1, l2):
    """stepwise program (Eqs. (11)-(12): HRR, T^(l1), T^(l2)) == Eq. (17)'s dense form with the ORACLE's c2s
    matrices (closed-form route), for the table program, the depth-first program of the block tier and both
    HRR axis choices; every HRR node has exactly two parents."""
    prog = hrr_c2s_program(l1, l2)
    rng = random.Random(10 * l1 + l2)
    xin = [rng.uniform(-1, 1) for _ in range(prog.nin)]
    X = [0.3, -0.7, 1.1]
    ref = _dense_side(l1, l2, xin, X, oracle.c2s_matrix(l1), oracle.c2s_matrix(l2))
    got = _run_prog(prog, xin, X)
    assert np.abs(got - ref).max() <= 1e-13 * max(1.0, np.abs(ref).max())
    terms = {}
    for (dst, src, coef, init) in prog.ops:
        terms.setdefault(dst, []).append(coef[0])
    hrr_nodes = [t for t in terms.values() if "x" in t]
    assert all(sorted(t) == ["one", "x"] for t in hrr_nodes)
    # depth-first straight-line program (emit_block.emit_side_dfs), executed by translating it to Python
    P = Prog()
    P.ind = 0
    emit_block.emit_side_dfs(P, l1, l2, lambda k: "IN[%d]" % k, ["X[0]", "X[1]", "X[2]"], lambda i: "SC[%d]" % i,
                             lambda r, e: P.w("OUT[%d] = %s;" % (r, e)), "h")
    py = [ln.strip().replace("const double ", "").rstrip(";") for ln in P.text().split("\n") if ln.strip() not in ("", "{", "}")]
    env = dict(IN=xin, X=X, SC=[0.0] * 2000, OUT=[0.0] * len(ref), fma=lambda a, b, c: a * b + c)
    exec("\n".join(py), env)
    assert np.abs(np.array(env["OUT"]) - ref).max() <= 1e-13 * max(1.0, np.abs(ref).max())


def test_solid_harmonics_two_routes_and_printed_rows():
    """generator (three-term recursion) vs oracle (closed-form triple sum) vs the rows printed in SURVEY 8(c)."""
    for l in range(5):
        T = np.zeros((2 * l + 1, ncart(l)))
        for m, row in enumerate(c2s_rows(l)):
            for (k, v) in row:
                T[m, k] = v
        assert np.abs(T - oracle.c2s_matrix(l)).max() < 1e-14
        assert int((np.abs(T) > 0).sum()) == [1, 3, 8, 16, 28][l]       # non-zero counts used in the flop model
    comps = cart_comps(2)
    T2 = {m - 2: {comps[k]: v for k, v in row} for m, row in enumerate(c2s_rows(2))}
    r3 = math.sqrt(3.0)
    assert T2[-2] == pytest.approx({(1, 1, 0): r3}) and T2[1] == pytest.approx({(1, 0, 1): r3})
    assert T2[0] == pytest.approx({(0, 0, 2): 1.0, (2, 0, 0): -0.5, (0, 2, 0): -0.5})
    assert T2[2] == pytest.approx({(2, 0, 0): r3 / 2, (0, 2, 0): -r3 / 2})
    assert [cart_comps(1)[row[0][0]] for row in c2s_rows(1)] == [(0, 1, 0), (0, 0, 1), (1, 0, 0)]    # p = (y, z, x)


@pytest.mark.parametrize("cls", [(3, 2, 3, 2), (3, 3, 0, 0), (3, 3, 2, 1), (3, 3, 3, 3)])
def test_block_layout(cls):
    """block tier: depth closure (a vertex of level k, order m needs order m+1 of level k-1), three rotating
    level buffers never alias a level with the two it reads, every thread's needed table lies inside the uniform one."""
    lay = emit_block.block_layout(cls)
    D, base, ctop, g = lay["D"], lay["base"], lay["ctop"], lay["g"]
    for k in range(1, ctop + 1):
        assert D[k - 1] >= D[k] + 1
        if k >= 2:
            assert D[k - 2] >= D[k] + 1
    size = [lay["L"] + 1] + [ncart(k) * D[k] for k in range(1, ctop + 1)]
    ranges = [(base[k % 3], base[k % 3] + size[k]) for k in range(ctop)]            # stored levels
    for k in range(len(ranges)):
        for j in (k - 1, k - 2):
            if j >= 0:
                assert ranges[k][1] <= ranges[j][0] or ranges[j][1] <= ranges[k][0]
    assert max(r[1] for r in ranges) <= lay["nslot"] if ranges else True
    for (a, c, m) in g.nodes:
        assert m < D[sum(c)] or sum(c) == 0
        if sum(c) == 0:
            assert m <= lay["L"] - sum(a)          # a level-e thread needs L+1-e orders of its pure-bra row
    assert lay["NB"] == sum(ncart(e) for e in range(lay["nst"] + 1)) and lay["NTH"] % 32 == 0


def test_tiers_and_committed_sources():
    """tier choice is a pure function of the class and matches classes.json; every class has a committed source;
    the register tier's order is the lower-PeakLive one."""
    meta = {tuple(m["cls"]): m for m in json.load(open(os.path.join(GEN, "classes.json")))}
    classes = canonical_classes()
    assert sorted(meta) == sorted(classes)
    count = {}
    for cls in classes:
        t = tiers.choose_tier(cls)
        assert meta[cls]["tier"] == t, cls
        count[t] = count.get(t, 0) + 1
        assert os.path.exists(os.path.join(GEN, "eri_%d%d%d%d.cu" % cls))
        if t == tiers.TIER_REGISTER:
            g = VrrGraph(*cls)
            from paper_2605_10312_b200.gen.emit_register import REG_EXTRA
            assert len(g.target_a) * len(g.target_c) <= 100 or cls in REG_EXTRA
            pl = {"postorder": meta[cls]["reg_peaklive_postorder"], "dsa": meta[cls]["reg_peaklive_dsa"]}
            from paper_2605_10312_b200.gen.emit_register import REG_ORDER_OF
            assert cls in REG_ORDER_OF or pl[meta[cls]["reg_order"]] == min(pl.values())      # (one class takes the DSA order for its 0 spill bytes)
    assert tiers.TIER_GLOBAL not in count and tiers.choose_tier((4, 4, 4, 4)) == tiers.TIER_BLOCK      # no class is left to the interpreter
    assert count[tiers.TIER_BLOCK] == 11 + 65 + 3 and count[tiers.TIER_REGISTER] == 25 and count[tiers.TIER_WARP] == 16
    # bra sides up to la + lb = 6 run the slab variant (x-slabs in warps, y- and z-chains in registers), (gf| and (gg| the z-column one
    assert sum(1 for c in classes if "slab_passes" in meta[c]) == 50 and sum(1 for c in classes if "heavy_passes" in meta[c]) == 29
    assert len(meta[(4, 4, 4, 4)]["heavy_passes"]) >= 2
    assert tiers.choose_tier((2, 2, 2, 2)) == tiers.TIER_WARP and tiers.choose_tier((3, 3, 3, 3)) == tiers.TIER_BLOCK


def test_lifetime_slot_allocator():
    """PAPER.md:265 slot packing for a serial order: no two vertices whose lifetimes overlap share a slot, every consumer finds its
    parents' slots intact, and the slot count equals PeakLive (Eq. (4)) -- the optimum for interval lifetimes."""
    from paper_2605_10312_b200.gen.graph import slot_allocation
    for cls in [(1, 1, 1, 1), (2, 1, 1, 0), (2, 2, 2, 2), (3, 1, 2, 0)]:
        g = VrrGraph(*cls)
        for order in (list(g.order), dsa_order(g)):
            slot, n = slot_allocation(g, order)
            assert n == peak_live(g, order) and set(slot) == set(order) and max(slot.values()) == n - 1
            owner = {}          # replay: slot -> vertex currently stored there
            for k in order:
                if g.nodes[k].side is None:
                    owner[slot[k]] = k
            for k in order:
                if g.nodes[k].side is None:
                    continue
                for p_ in g.parents(k):
                    assert owner[slot[p_]] == p_, (cls, k, p_)      # the parent's value has not been overwritten
                owner[slot[k]] = k
    g = VrrGraph(2, 2, 2, 2)
    assert slot_allocation(g, g.order)[1] == 443 and g.num_nodes() == 2321


def test_warp_record_stride_spreads_the_setup_lanes():
    """Warp tier, one quartet per warp: lane p of the set-up pass writes primitive record p, so the record stride
    PRS decides the bank conflicts of those stores.  8-byte banks, 16 of them per half-warp: PRS must be even
    (16-byte broadcast loads of the record) and PRS/2 odd, which puts the 16 set-up lanes on 8 distinct banks
    (2 wavefronts per store; PRS = 40 at (dd|dd) gave 8)."""
    import glob
    import re
    seen = 0
    for path in sorted(glob.glob(os.path.join(GEN, "eri_*.cu"))):
        for m in re.finditer(r"constexpr int Q = (\d+), G = \d+;.*\nconstexpr int WARPS = \d+, WSM = (\d+), PRS = (\d+), PBS = (\d+),", open(path).read()):
            q, wsm, prs, pbs = (int(x) for x in m.groups())
            if q != 1:
                assert prs % 2 == 1                    # packed kernels: odd stride spreads the groups' records
                continue
            seen += 1
            assert prs % 2 == 0 and wsm % 2 == 0, path
            banks = {}
            for lane in range(min(pbs, 16)):
                banks.setdefault((lane * prs) % 16, set()).add(lane * prs)
            assert max(len(v) for v in banks.values()) <= 2, (path, prs)
    assert seen >= 30


def test_no_spill_bytes_in_class_kernels():
    """ptxas of the committed class sources (the logs build.py keeps beside the objects): no kernel of a class source keeps a stack
    frame or spills a byte -- where registers run out the emitters stage values in shared memory explicitly.  The
    table-driven cross-check interpreter and the buffered digest (csrc/*.cu, not generated) are not covered."""
    import glob
    import re
    from paper_2605_10312_b200 import build
    build.build_library()
    logs = sorted(glob.glob(os.path.join(build.OBJ, "gen_eri_*.o.log")))
    assert len(logs) == 120
    pat = re.compile(r"Compiling entry function '(\S+)' for 'sm_100a'.*?\n.*?(\d+) bytes stack frame, (\d+) bytes spill stores, (\d+) bytes spill loads\n.*?Used (\d+) registers", re.S)
    seen = 0
    for f in logs:
        for name, stack, st, ld, regs in pat.findall(open(f).read()):
            seen += 1
            assert (int(stack), int(st), int(ld)) == (0, 0, 0), (os.path.basename(f), name, stack, st, ld)
            assert int(regs) <= 255
    assert seen >= 240      # one to four kernels per class source (plain, packed, Fock, primitive-split, side kernels apart)
