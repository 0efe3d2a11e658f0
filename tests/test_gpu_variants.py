"""Variant parity (SURVEY section 4 "variant parity"; PAPER.md:311 ablation toggles): every generator variant of the
ablation study -- literal Alg. 1 axis rule, DSA / post-order emission, no spherical fusion, thread-per-quartet Tier 1
forced, table-driven buffered tier forced, level-synchronous block tier -- must give the oracle's integrals on a seeded
sample.  The variant libraries are generated into a temporary directory (never into csrc/gen) and linked there; each runs
in a child process that loads it through RCG_LIB."""
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
CLASSES = [(1, 0, 1, 0), (1, 1, 1, 1), (2, 1, 2, 1), (2, 2, 2, 2), (3, 3, 2, 2)]


@pytest.mark.parametrize("name", ["no_sph_fusion", "tier1_thread", "tier1_thread_alg1_axis", "tier1_thread_dsa",
                                  "tier1_thread_no_sph_fusion", "buffered_global", "block_level_table"])
def test_variant_equals_oracle(name, tmp_path):
    import torch
    assert torch.cuda.is_available()
    from paper_2605_10312_b200 import ablation
    lib, facts = ablation.build_variant(name, classes=CLASSES, workdir=str(tmp_path))
    assert os.path.abspath(lib) != os.path.join(ROOT, "paper_2605_10312_b200", "librcg.so") and facts
    _, tier, _ = ablation.VARIANTS[name]
    tags = ",".join("%d%d%d%d" % c for c in facts)
    p = subprocess.run([sys.executable, os.path.join(ROOT, "tests", "variant_worker.py"), str(tier), tags, "200"],
                       env=dict(os.environ, RCG_LIB=lib), capture_output=True, text=True, cwd=ROOT)
    assert p.returncode == 0, p.stdout[-2000:] + p.stderr[-3000:]
    assert p.stdout.count("ok") == len(facts), p.stdout
    print(name, p.stdout.strip().replace("\n", " | "))
