"""Tier selection and specialised-kernel emission (PAPER.md:251-257 tiers, re-derived for sm_100a;
DESIGN.md 'Tiers').  Every class also carries the table-driven global tier.

Warp tier (emit_warp.py) is generated where one warp can hold a quartet: at most 32 bra target
components (bra pair up to (dd| or (fp|) and a ket side whose accumulators (nC per lane) and table
fit the register file (ket pair up to |dd) or |fp)).  The paper's rule (Sigma l <= 6 -> Tier 1,
PAPER.md:253-257) came from 255 registers per THREAD-per-quartet on A100 and does not carry over.
"""
import os

from . import options
from .solid import ncart

TIER_REGISTER, TIER_WARP, TIER_GLOBAL, TIER_BLOCK = 1, 2, 3, 4
WARP_PAIRS = {(0, 0), (1, 0), (1, 1), (2, 0), (2, 1), (2, 2), (3, 0), (3, 1)}
WARP_KETS = WARP_PAIRS | {(0, 0)}


def warp_eligible(cls):
    la, lb, lc, ld = cls
    nT = sum(ncart(e) for e in range(la, la + lb + 1))
    return (la, lb) in WARP_PAIRS and (lc, ld) in WARP_KETS and nT <= 32


def swapped_eligible(cls):
    """bra too wide for one warp ((fd|: 46 target components) but ket light: generate the kernel for the
    bra<->ket swapped quartet (cd|ab) = (ab|cd) -- lanes = components of the light side, the (fd| side
    becomes the per-lane table with 46 accumulators -- and permute indices in the launcher."""
    la, lb, lc, ld = cls
    nTk = sum(ncart(e) for e in range(lc, lc + ld + 1))
    return (la, lb) == (3, 2) and (lc, ld) in WARP_PAIRS and nTk <= 32 and not options.flag("GEN_NO_SWAP")


def block_eligible(cls):
    """bra side wider than a warp, ket table too large for registers: one thread block per quartet, thread =
    bra component (all levels), ket table in shared memory, accumulators in registers (emit_block.py).
    (gg|gg) stays in the global tier: 145 accumulators per thread and a 373 KB table do not fit an SM."""
    la, lb, lc, ld = cls
    if options.flag("GEN_NO_BLOCK") or (la, lb) not in ((3, 2), (3, 3)):
        return False
    nC = sum(ncart(f) for f in range(lc, lc + ld + 1))
    return nC <= 80


def register_eligible(cls):
    """at most 56 Cartesian targets: one thread per quartet (the paper's Tier 1) beats a warp per quartet when
    the list is long and its contraction depths are even; the class keeps its warp-tier kernels for the rest."""
    if options.flag("GEN_NO_REGISTER"):
        return False
    from . import emit_register
    return emit_register.eligible(cls)


def heavy_eligible(cls):
    """classes with a g shell: heavy block tier (emit_heavy.py): z-chains in registers, heads in shared memory, passes over
    ket x-slabs, Phase 2 in the side kernels."""
    if options.flag("GEN_HEAVY_ALL") and block_eligible(cls):       # comparison runs: the (fd|fd), (ff|xx) classes through the heavy emitter
        return True
    return max(cls) == 4 and not options.flag("GEN_NO_HEAVY")


def slab_eligible(cls):
    """bra sides with la + lb <= 6 of the block-tier classes and of the g classes: every x-slab of the bra pyramid fits a
    warp, so y- and z-chains of the ket run in registers with shuffled cross terms (emit_heavy.emit_class_slab)."""
    from . import emit_heavy
    if (options.flag("GEN_SLAB_ALL") or options.get("FORCE_TIER", "") == "block") and not register_eligible(cls) and emit_heavy.slab_eligible(cls):
        return True       # comparison runs: warp-tier classes through the slab kernel
    if warp_eligible(cls):
        return False
    if swapped_eligible(cls):     # (fd|xx) with a light ket: in the cfg5 pass (one K4 per batch, mostly 1) the slab kernel is 1.3-1.8x faster than
        nC = sum(ncart(f) for f in range(cls[2], cls[2] + cls[3] + 1))      # the bra<->ket swapped warp kernel from 16 ket targets up, 1.5-2.3x slower below
        if options.flag("GEN_NO_SLAB_FD") or register_eligible(cls) or nC < 16:
            return False
    return (block_eligible(cls) or max(cls) == 4) and emit_heavy.slab_eligible(cls) and not options.flag("GEN_NO_SLAB")


def choose_tier(cls):
    force = options.get("FORCE_TIER", "")      # ablation: one tier for every class that has its emitter
    if options.flag("GEN_ALL_GLOBAL") or force == "global":
        return TIER_GLOBAL
    if force == "register" and (warp_eligible(cls) or swapped_eligible(cls)):
        from .graph import VrrGraph
        if VrrGraph(*cls).num_nodes() <= 1500:          # the unrolled thread-per-quartet kernel (the paper's Tier 1) up to (dd|dp)
            return TIER_REGISTER
    if force == "warp" and warp_eligible(cls):
        return TIER_WARP
    if heavy_eligible(cls) or slab_eligible(cls):
        return TIER_BLOCK
    if (warp_eligible(cls) or swapped_eligible(cls)) and register_eligible(cls):
        return TIER_REGISTER
    if warp_eligible(cls) or swapped_eligible(cls):
        return TIER_WARP
    return TIER_BLOCK if block_eligible(cls) else TIER_GLOBAL


def emit_specialised(cls, tier):
    """-> (declarations to splice into the class source, launcher symbol or None, metadata)."""
    if tier == TIER_REGISTER:
        from . import emit_warp, emit_register
        # classes whose thread-per-quartet Fock epilogue would spill digest in their warp kernels instead (any list)
        wfock = cls in emit_register.REG_FOCK_EXCLUDED and options.get("SPH_FUSION", "1") != "0"
        wt, wsym, meta = emit_warp.emit_class(cls, fock=wfock) if warp_eligible(cls) else emit_warp.emit_class_swapped(cls, fock=wfock)
        rt, rsym, rmeta = emit_register.emit_class(cls)
        meta.update(rmeta)
        text, sym = emit_register.emit_auto(cls, wt, wsym, rt, rsym)
        return text, sym, meta
    if tier == TIER_WARP:
        from . import emit_warp
        fock = options.get("SPH_FUSION", "1") != "0"       # (the Fock epilogue goes with the default Phase 2)
        if not warp_eligible(cls):
            return emit_warp.emit_class_swapped(cls, fock=fock)
        return emit_warp.emit_class(cls, fock=fock)
    if tier == TIER_BLOCK and slab_eligible(cls):
        from . import emit_heavy
        return emit_heavy.emit_class_slab(cls)
    if tier == TIER_BLOCK and heavy_eligible(cls):
        from . import emit_heavy
        return emit_heavy.emit_class(cls)
    if tier == TIER_BLOCK:
        from . import emit_block
        return emit_block.emit_class(cls)
    return "", None, {}
