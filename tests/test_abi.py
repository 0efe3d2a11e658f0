"""CPU-side checks of the boundary: the C-ABI library builds for sm_100a, loads, and exports every
symbol include/rcg.h declares; the binding fails loudly without a GPU (no CPU fallback)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    from paper_2605_10312_b200 import build
    return build.build_library()


def declared_symbols():
    txt = open(os.path.join(ROOT, "include", "rcg.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(rcg_[a-z0-9_]+)\s*\(", txt)))


def test_header_symbols_exported(libpath):
    lib = ctypes.CDLL(libpath)
    syms = declared_symbols()
    assert "rcg_eri_batch" in syms and len(syms) >= 12
    for s in syms:
        assert hasattr(lib, s), "librcg.so does not export %s" % s
    from paper_2605_10312_b200 import rcg
    assert sorted(rcg.EXPORTS) == syms


def test_class_table(libpath):
    from paper_2605_10312_b200 import rcg, workloads
    cls = rcg.classes()
    assert set(workloads.canonical_classes(4)) == set(cls) and len(cls) == 120      # PAPER.md:299, reading R-CLASSN
    info = rcg.class_info((2, 2, 2, 2))
    assert info["flops_per_prim_quartet"] > 13923 and info["tier"] in (1, 2, 3)
    assert rcg.class_info((0, 2, 1, 2)) == rcg.class_info((2, 1, 2, 0))    # canonicalisation
    assert rcg.class_info((4, 3, 0, 0))["tier"] == 4 and rcg.class_info((0, 0, 3, 4)) == rcg.class_info((4, 3, 0, 0))
    with pytest.raises(rcg.RcgError):
        rcg.class_info((5, 0, 0, 0))
    assert rcg.lib().rcg_status_string(-3).decode() == "workspace too small"


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_2605_10312_b200 import rcg, workloads
    basis, q = workloads.cfg1(4)
    with pytest.raises(rcg.RcgError):
        rcg.Basis(basis)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2605_10312_b200")
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dp, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "eri_oracle" not in txt, f


def test_grad_supported_classes_host_logic():
    """rcg_eri_grad_supported is host logic (no CUDA call): every class of s, p, d shells in any order, all 55 pair-canonical classes of
    lmax = 3 and 111 of the 120 of lmax = 4 (the heaviest with their accumulators in a global scratch); a refused class states why
    (more than 227 KB of shared memory for the recurrence buffers alone, or a Boys order beyond 16)."""
    import itertools
    from paper_2605_10312_b200 import rcg, workloads
    assert all(rcg.eri_grad_supported(c)[0] for c in itertools.product(range(3), repeat=4))
    for lmax, want in ((2, 21), (3, 55), (4, 111)):
        res = [rcg.eri_grad_supported(c) for c in workloads.canonical_classes(lmax)]
        assert sum(ok for ok, _ in res) == want
        assert all(ok or smem > 227 * 1024 for ok, smem in res)
    assert rcg.eri_grad_supported((3, 3, 3, 3))[0] and not rcg.eri_grad_supported((4, 4, 4, 4))[0] and not rcg.eri_grad_supported((4, 3, 3, 3))[0]
    with pytest.raises(Exception):
        rcg.eri_grad_supported((5, 0, 0, 0))
