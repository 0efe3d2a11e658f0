"""Tier selection and specialised-kernel emission (PAPER.md:251-257 tiers, re-derived for sm_100a;
DESIGN.md 'Tiers').  Every class also carries the table-driven global tier."""
import os

TIER_REGISTER, TIER_WARP, TIER_GLOBAL = 1, 2, 3

WARP_CLASSES = {(1, 1, 1, 1), (2, 2, 2, 2)}


def choose_tier(cls):
    if os.environ.get("RCG_GEN_ALL_GLOBAL"):
        return TIER_GLOBAL
    if cls in WARP_CLASSES:
        return TIER_WARP
    return TIER_GLOBAL


def emit_specialised(cls, tier):
    """-> (declarations to splice into the class source, launcher symbol or None, metadata)."""
    if tier == TIER_WARP:
        from . import emit_warp
        return emit_warp.emit_class(cls)
    return "", None, {}
