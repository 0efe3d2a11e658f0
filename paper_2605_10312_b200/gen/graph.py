"""Recurrence graphs for one angular class (la lb|lc ld): the generator's data model.

Phase 1 = VRR graph of Eq. (2) and its ket mirror (reading R-KET), built with
the axis-priority rule of Alg. 1 as the TEXT states it (reading R-AXIS):
consumer side first (ket before bra), z -> y -> x inside a side.  Vertex = one FP64
intermediate [a0|c0]^(m).  Only vertices reachable from the targets
[e0|f0]^(0), e in [la,la+lb], f in [lc,lc+ld] are kept.
Phase 2 = HRR of Eq. (3) with the stepwise Cartesian->spherical transform of
Eqs. (11)-(16): bra HRR, Ta, Tb, ket HRR, Tc, Td (mask 0000->..->1111).
Schedules: PeakLive of Eq. (4) and the DSA greedy order of Eq. (7)
(reading R-REACH).
"""
from .solid import cart_comps, ncart, c2s_rows


def sub1(t, i):
    return tuple(v - (1 if k == i else 0) for k, v in enumerate(t))


def reduction_axis(t):
    """z -> y -> x priority."""
    return 2 if t[2] > 0 else (1 if t[1] > 0 else 0)


class VrrNode:
    __slots__ = ("a", "c", "m", "side", "axis", "n2", "ncross", "p1", "p2", "p3", "p4", "p5")


class VrrGraph:
    """nodes: dict (a,c,m) -> VrrNode (base nodes (0,0,m) have side None); order: topological."""

    def __init__(self, la, lb, lc, ld, axis_rule="side"):
        self.l = (la, lb, lc, ld)
        self.L = la + lb + lc + ld
        self.axis_rule = axis_rule
        self.nodes = {}
        self.order = []
        self.bra_levels = list(range(la, la + lb + 1))
        self.ket_levels = list(range(lc, lc + ld + 1))
        self.target_a = [a for e in self.bra_levels for a in cart_comps(e)]
        self.target_c = [c for f in self.ket_levels for c in cart_comps(f)]
        for a in self.target_a:
            for c in self.target_c:
                self._need(a, c, 0)

    def _pick(self, a, c):
        """which (side, axis) Eq. (2) is applied on to produce [a|c]."""
        if self.axis_rule == "side":            # text reading: ket wholly before bra
            if sum(c) > 0:
                return "ket", reduction_axis(c)
            return "bra", reduction_axis(a)
        # literal Alg. 1 (no break -> last hit wins): c_z, a_z, c_y, a_y, c_x, a_x
        for i in (2, 1, 0):
            if c[i] > 0:
                return "ket", i
            if a[i] > 0:
                return "bra", i
        raise AssertionError

    def _need(self, a, c, m):
        key = (a, c, m)
        if key in self.nodes:
            return key
        n = VrrNode()
        n.a, n.c, n.m = a, c, m
        n.p1 = n.p2 = n.p3 = n.p4 = n.p5 = None
        n.n2 = n.ncross = 0
        if sum(a) == 0 and sum(c) == 0:
            n.side, n.axis = None, -1
            self.nodes[key] = n
            self.order.append(key)
            return key
        self.nodes[key] = n            # placeholder (graph is acyclic; safe)
        side, i = self._pick(a, c)
        n.side, n.axis = side, i
        if side == "ket":
            c1 = sub1(c, i)
            n.p1 = self._need(a, c1, m)
            n.p2 = self._need(a, c1, m + 1)
            if c1[i] > 0:
                n.n2 = c1[i]
                c2 = sub1(c1, i)
                n.p3 = self._need(a, c2, m)
                n.p4 = self._need(a, c2, m + 1)
            if a[i] > 0:
                n.ncross = a[i]
                n.p5 = self._need(sub1(a, i), c1, m + 1)
        else:
            a1 = sub1(a, i)
            n.p1 = self._need(a1, c, m)
            n.p2 = self._need(a1, c, m + 1)
            if a1[i] > 0:
                n.n2 = a1[i]
                a2 = sub1(a1, i)
                n.p3 = self._need(a2, c, m)
                n.p4 = self._need(a2, c, m + 1)
            if c[i] > 0:
                n.ncross = c[i]
                n.p5 = self._need(a1, sub1(c, i), m + 1)
        self.order.append(key)          # post-order => topological
        return key

    def parents(self, key):
        n = self.nodes[key]
        return [p for p in (n.p1, n.p2, n.p3, n.p4, n.p5) if p is not None]

    def num_nodes(self):
        """recurrence vertices, base values [00|00]^(m) excluded."""
        return sum(1 for k in self.order if self.nodes[k].side is not None)

    def flops(self):
        """(flops, dp_instructions) per primitive quartet for the VRR vertices alone.
        vertex = c1*p1 (MUL) + c2*p2 (FMA) [+ t=p3-r*p4 (FMA), += k*t (FMA)] [+ k5*p5 (FMA)]."""
        fl = ins = 0
        for k in self.order:
            n = self.nodes[k]
            if n.side is None:
                continue
            fl += 1 + 2
            ins += 2
            if n.p3 is not None:
                fl += 4
                ins += 2
            if n.p5 is not None:
                fl += 2
                ins += 1
        return fl, ins

    def targets(self):
        return [(a, c, 0) for a in self.target_a for c in self.target_c]


def peak_live(g, order):
    """Eq. (4): max number of simultaneously live vertices under `order` (reading R-LIVE:
    a target dies when produced, it is accumulated at once; base values are live from the start)."""
    pos = {k: i for i, k in enumerate(order)}
    last = {}
    for k in order:
        for p in g.parents(k):
            last[p] = max(last.get(p, -1), pos[k])
    events = [0] * (len(order) + 2)
    for k in order:
        birth = 0 if g.nodes[k].side is None else pos[k]
        death = last.get(k, pos[k])
        events[birth] += 1
        events[death + 1] -= 1
    live = peak = 0
    for e in events:
        live += e
        peak = max(peak, live)
    return peak


def slot_allocation(g, order):
    """The paper's two-pass lifetime slot allocator for a SERIAL order (forward dry run for births and deaths, then
    packing): vertices whose lifetimes do not overlap share a buffer slot.  Lifetimes as in peak_live (reading R-LIVE): a vertex is
    born at its position (base values at 0), dies at its last consumer, a target at its own position.  Interval graphs are coloured
    optimally by handing every vertex, in order of birth, the lowest slot that is free again, so the slot count EQUALS PeakLive of
    Eq. (4) -- (dd|dd): 2,330 vertices in 443 slots in post-order (5.3x; the paper quotes 1.9x for its count of 3,545) -- against
    3 x the widest level (1,680) for the level-synchronous execution of the table-driven tier, the only kernel here that keeps a slot
    buffer.  -> (dict vertex -> slot, number of slots)."""
    import heapq
    pos = {k: i for i, k in enumerate(order)}
    last = {}
    for k in order:
        for p in g.parents(k):
            last[p] = max(last.get(p, -1), pos[k])
    birth = {k: (0 if g.nodes[k].side is None else pos[k]) for k in order}
    death = {k: last.get(k, pos[k]) for k in order}
    by_birth = sorted(order, key=lambda k: (birth[k], pos[k]))
    free, busy, slot, nslots = [], [], {}, 0        # free slots (min-heap), (death, slot) of live vertices
    for k in by_birth:
        while busy and busy[0][0] < birth[k]:
            heapq.heappush(free, heapq.heappop(busy)[1])
        if free:
            s_ = heapq.heappop(free)
        else:
            s_, nslots = nslots, nslots + 1
        slot[k] = s_
        heapq.heappush(busy, (death[k], s_))
    return slot, nslots


def dsa_order(g):
    """Greedy dependency scheduling, Eq. (7): among ready vertices pick the one
    maximising sum_{w in Reach(v)} (out(w) - in(w)); Reach = v and its transitive consumers
    (R-REACH) -- approximated by v and its direct consumers for graphs above 4000 vertices to stay
    O(|V|^2).  Ties: higher Boys order first, then creation order."""
    keys = list(g.order)
    idx = {k: i for i, k in enumerate(keys)}
    cons = [[] for _ in keys]
    npar = [0] * len(keys)
    for k in keys:
        ps = g.parents(k)
        npar[idx[k]] = len(ps)
        for p in ps:
            cons[idx[p]].append(idx[k])
    score_node = [len(cons[i]) - npar[i] for i in range(len(keys))]
    big = len(keys) > 4000
    reach_score = [0] * len(keys)
    for i in range(len(keys) - 1, -1, -1):
        if big:
            reach_score[i] = score_node[i] + sum(score_node[j] for j in cons[i])
        else:
            seen = set()
            stack = [i]
            while stack:
                j = stack.pop()
                if j in seen:
                    continue
                seen.add(j)
                stack.extend(cons[j])
            reach_score[i] = sum(score_node[j] for j in seen)
    remaining = list(npar)
    ready = [i for i in range(len(keys)) if remaining[i] == 0]
    out = []
    import heapq
    heap = [(-reach_score[i], -g.nodes[keys[i]].m, i) for i in ready]
    heapq.heapify(heap)
    while heap:
        _, _, i = heapq.heappop(heap)
        out.append(keys[i])
        for j in cons[i]:
            remaining[j] -= 1
            if remaining[j] == 0:
                heapq.heappush(heap, (-reach_score[j], -g.nodes[keys[j]].m, j))
    assert len(out) == len(keys)
    return out


# ----------------------------------------------------------------------------- Phase 2
class LinProgram:
    """Straight-line program of ops  dst (=|+=) coef * src  over a private slot space.
    coef: ("one",) | ("x", axis) [HRR displacement A-B or C-D] | ("const", value).
    inputs: slots 0..nin-1; outputs: list of slots."""

    def __init__(self, nin):
        self.nin = nin
        self.nslots = nin
        self.ops = []
        self.outputs = []

    def new(self):
        self.nslots += 1
        return self.nslots - 1

    def op(self, dst, src, coef, init):
        self.ops.append((dst, src, coef, init))

    def flops(self):
        fl = 0
        for (_, _, coef, init) in self.ops:
            if init:
                fl += 0 if coef[0] == "one" else 1
            else:
                fl += 1 if coef[0] == "one" else 2
        return fl


def hrr_c2s_program(l1, l2, c2s=True):
    """One side of Phase 2 for a fixed index of the other side: inputs = (e0| for e=l1..l1+l2 in
    cart_comps order (level-major); HRR Eq. (3) (a,b+1i| = (a+1i,b| + X_i (a,b|, X=A-B (or C-D,
    R-HRRK); then T^(l1) on the first index (mask step), then T^(l2) on the second (Eqs. (11)-(12),
    (15)-(16)).  Outputs: [nsph(l1)][nsph(l2)] row-major."""
    levels = list(range(l1, l1 + l2 + 1))
    idx = {}
    n = 0
    for e in levels:
        for a in cart_comps(e):
            idx[(a, (0, 0, 0))] = n
            n += 1
    prog = LinProgram(n)

    def get(a, b):
        key = (a, b)
        if key in idx:
            return idx[key]
        i = 0 if b[0] > 0 else (1 if b[1] > 0 else 2)
        b1 = sub1(b, i)
        a1 = tuple(v + (1 if k == i else 0) for k, v in enumerate(a))
        hi = get(a1, b1)
        lo = get(a, b1)
        s = prog.new()
        prog.op(s, hi, ("one",), True)
        prog.op(s, lo, ("x", i), False)
        idx[key] = s
        return s

    A, B = cart_comps(l1), cart_comps(l2)
    cart = [[get(a, b) for b in B] for a in A]
    if not c2s:          # ablation "no spherical fusion": the Cartesian pair block, transformed later
        prog.outputs = [cart[ia][jb] for ia in range(len(A)) for jb in range(len(B))]
        return prog
    T1, T2 = c2s_rows(l1), c2s_rows(l2)
    # first index: [nsph1][ncart2]
    if l1 >= 2:
        half = []
        for row in T1:
            r = []
            for jb in range(len(B)):
                s = prog.new()
                for t, (ia, coef) in enumerate(row):
                    prog.op(s, cart[ia][jb], ("const", coef), t == 0)
                r.append(s)
            half.append(r)
    else:   # l<=1: pure permutation (s: identity, p: y,z,x) -- no arithmetic
        half = [[cart[row[0][0]][jb] for jb in range(len(B))] for row in T1]
    if l2 >= 2:
        outs = []
        for ia in range(len(half)):
            for row in T2:
                s = prog.new()
                for t, (jb, coef) in enumerate(row):
                    prog.op(s, half[ia][jb], ("const", coef), t == 0)
                outs.append(s)
    else:
        outs = [half[ia][row[0][0]] for ia in range(len(half)) for row in T2]
    prog.outputs = outs
    return prog


def c2s_pair_program(l1, l2):
    """T^(l1) (x) T^(l2) applied to a Cartesian pair block [ncart(l1)][ncart(l2)] -> [nsph(l1)][nsph(l2)] (Eq. (8)):
    the deferred transform of the "materialise then transform" order, Eq. (17)."""
    n1, n2 = ncart(l1), ncart(l2)
    prog = LinProgram(n1 * n2)
    T1, T2 = c2s_rows(l1), c2s_rows(l2)
    half = []
    for row in T1:
        r = []
        for jb in range(n2):
            if len(row) == 1 and row[0][1] == 1.0:
                r.append(row[0][0] * n2 + jb)
                continue
            s = prog.new()
            for t, (ia, coef) in enumerate(row):
                prog.op(s, ia * n2 + jb, ("const", coef), t == 0)
            r.append(s)
        half.append(r)
    outs = []
    for ia in range(len(half)):
        for row in T2:
            if len(row) == 1 and row[0][1] == 1.0:
                outs.append(half[ia][row[0][0]])
                continue
            s = prog.new()
            for t, (jb, coef) in enumerate(row):
                prog.op(s, half[ia][jb], ("const", coef), t == 0)
            outs.append(s)
    prog.outputs = outs
    return prog


def class_flops(la, lb, lc, ld, g=None):
    """Algorithmic FP64 flop model, FMA=2, MUL/ADD=1.
    per primitive quartet: VRR vertices + contraction adds (one per target) + a fixed 70 (pair/
    quartet setup) + Boys (9-term Taylor 17 + exp/rsqrt counted 1 each + 3 per downward step);
    per contracted quartet: Phase 2 = nC * bra program + nAB_sph * ket program."""
    g = g or VrrGraph(la, lb, lc, ld)
    vfl, _ = g.flops()
    L = la + lb + lc + ld
    ntarget = len(g.target_a) * len(g.target_c)
    per_prim = vfl + ntarget + 70 + (19 + 3 * L)
    bra = hrr_c2s_program(la, lb)
    ket = hrr_c2s_program(lc, ld)
    per_q = len(g.target_c) * bra.flops() + (2 * la + 1) * (2 * lb + 1) * ket.flops()
    return per_prim, per_q


def canonical_classes(lmax=4, extra=()):
    """the pair-canonical classes la >= lb, lc >= ld, (la,lb) >= (lc,ld): 120 for lmax = 4 (reading R-CLASSN)."""
    pairs = [(a, b) for a in range(lmax + 1) for b in range(a + 1)]
    out = [(p[0], p[1], q[0], q[1]) for p in pairs for q in pairs if p >= q]
    return out + [e for e in extra if e not in out]
