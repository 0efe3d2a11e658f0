"""Tier selection and specialised-kernel emission (PAPER.md:251-257 tiers, re-derived for sm_100a;
DESIGN.md 'Tiers').  Every class also carries the table-driven global tier."""

TIER_REGISTER, TIER_WARP, TIER_GLOBAL = 1, 2, 3


def choose_tier(cls):
    return TIER_GLOBAL


def emit_specialised(cls, tier):
    """-> (declarations to splice into the class source, launcher symbol or None, metadata)."""
    return "", None, {}
