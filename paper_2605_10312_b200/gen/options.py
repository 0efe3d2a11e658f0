"""Generator options (ablation and sweep switches).  Defaults are the product; `generate.py --set KEY=VALUE ...` (and its
named flags --axis-rule, --order, --no-spherical-fusion, --force-tier) changes them for ONE run that writes to --out-dir.
Nothing is read from the environment: what a run generates depends on its command line only.

  AXIS_RULE      side | alg1     Phase-1 axis priority: the text's side-major rule or the literal Alg. 1 (reading R-AXIS)
  ORDER          auto | dsa | post   emission order of the register tier (Eq. (7) DSA greedy, post-order, or the lower PeakLive)
  SPH_FUSION     1 | 0           stepwise c2s fused into the HRR (Eqs. (11)-(16)) or "materialise then transform" (Eq. (17))
  FORCE_TIER     0 | register | warp | block | global     tier override where the class has that emitter
  ... and the per-emitter tuning knobs (WARP_*, BLOCK_*, HEAVY_*), documented where they are read.
"""
OPT = {}


def set_options(d):
    OPT.clear()
    OPT.update(d or {})


def get(name, default=""):
    return OPT.get(name, default)


def geti(name, default=0):
    return int(OPT.get(name, default))


def flag(name):
    return str(OPT.get(name, "")) not in ("", "0", "False", "false")
