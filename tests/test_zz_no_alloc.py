"""rcg_eri_batch_static (include/rcg.h): the allocation-free entry point -- scratch in the library's 32 MiB static device array --
against the existing path (rcg_eri_batch with a caller-allocated workspace) on the same lists, two calls in a row per class (the
second with a different list and size, so stale scratch contents of the first would show), within the gates of the parity tests
(tests/parity_util.py: 1e-12 + 1e-10 relative per component, 1e-10 of the quartet's scale).  Collected last on purpose (the suite
runs with pytest -x); it passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest

from parity_util import gates
from paper_2605_10312_b200 import workloads

pytestmark = pytest.mark.gpu


def test_static_scratch_entry_equals_existing_path():
    import torch
    from paper_2605_10312_b200 import rcg
    assert torch.cuda.is_available()
    bg = workloads.water_cluster((2, 2, 1), 6, with_g=True)
    b4, _, qg = workloads.cfg4(1, 120)
    Bg, B4 = rcg.Basis(bg), rcg.Basis(b4)
    cases = [(Bg, bg, (4, 0, 0, 0), 3000, 1777), (Bg, bg, (4, 3, 1, 0), 700, 333), (Bg, bg, (3, 3, 1, 0), 2000, 901),
             (Bg, bg, (0, 1, 3, 4), 500, 77), (B4, b4, (4, 4, 4, 4), 100, 37)]
    free_marks = []
    for ci, (B, basis, cls, n1, n2) in enumerate(cases):
        nmax = rcg.eri_batch_static_max_quartets(B, cls)
        assert nmax >= max(n1, n2) and rcg.eri_workspace_bytes(B, cls, nmax) <= rcg.STATIC_SCRATCH_BYTES < rcg.eri_workspace_bytes(B, cls, nmax + 1)
        for k, n in enumerate((n1, n2)):                    # two calls in a row, different lists
            q = qg[k * 50:k * 50 + n] if cls == (4, 4, 4, 4) else workloads.sample_class_quartets(basis, cls, n, seed=4000 + 10 * ci + k)
            qd = torch.tensor(np.ascontiguousarray(q), device="cuda")
            ref = rcg.eri_batch(B, cls, qd)                 # existing path: workspace allocated by the binding
            out = torch.full(ref.shape, float("nan"), dtype=torch.float64, device="cuda")
            torch.cuda.synchronize()
            free0 = torch.cuda.mem_get_info()[0]
            rcg.eri_batch_static(B, cls, qd, out)
            torch.cuda.synchronize()
            free_marks.append((ci, k, free0 - torch.cuda.mem_get_info()[0]))
            g1, g2, err, scale = gates(out.cpu().numpy(), ref.cpu().numpy())
            assert g1.all() and g2.all(), (cls, k, float(err.max()))
    # no device memory is taken by a call once the class's kernels are loaded (second call of each class)
    assert all(d == 0 for (_, k, d) in free_marks if k == 1), free_marks


def test_static_scratch_entry_limits():
    import torch
    from paper_2605_10312_b200 import rcg
    b4, _, qg = workloads.cfg4(1, 200)
    B4 = rcg.Basis(b4)
    nmax = rcg.eri_batch_static_max_quartets(B4, (4, 4, 4, 4))
    assert nmax == rcg.STATIC_SCRATCH_BYTES // (32770 * 8) == 127
    qd = torch.tensor(qg[:nmax + 1], device="cuda")
    out = torch.zeros((nmax + 1, 9, 9, 9, 9), dtype=torch.float64, device="cuda")
    with pytest.raises(rcg.RcgError, match="static scratch"):
        rcg.eri_batch_static(B4, (4, 4, 4, 4), qd, out)
    torch.cuda.synchronize()
    assert float(out.abs().sum()) == 0.0                    # nothing was launched
    b2, q2 = workloads.cfg2(16)
    with pytest.raises(rcg.RcgError, match="unsupported"):  # (dd|dd) uses no scratch: rcg_eri_batch with no workspace is the call
        rcg.eri_batch_static(rcg.Basis(b2), (2, 2, 2, 2), torch.tensor(q2, device="cuda"),
                             torch.zeros((16, 5, 5, 5, 5), dtype=torch.float64, device="cuda"))
    rcg.eri_batch_static(B4, (4, 4, 4, 4), qd[:0].contiguous(), out[:0].contiguous())      # empty batch: no-op
