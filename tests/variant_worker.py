"""child process of tests/test_gpu_variants.py: the library RCG_LIB names (a generator variant) against the oracle.
argv: tier classes(comma-separated tags) n"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))


def main():
    import torch
    import oracle
    from parity_util import assert_parity
    from paper_2605_10312_b200 import ablation, rcg, workloads
    tier, n = int(sys.argv[1]), int(sys.argv[3])
    assert os.path.abspath(rcg.LIB_PATH) == os.path.abspath(os.environ["RCG_LIB"])
    basis = ablation.make_basis()
    B = rcg.Basis(basis)
    for ci, t in enumerate(sys.argv[2].split(",")):
        cls = tuple(int(ch) for ch in t)
        q = workloads.sample_class_quartets(basis, cls, n, seed=31 + ci)
        tr = tier if (tier in (0, 3) or rcg.class_info(cls)["tier"] == tier) else 0
        got = rcg.eri_batch(B, cls, torch.tensor(q, device="cuda"), tier=tr).cpu().numpy()
        ref = oracle.eri_batch(basis, q)
        r = assert_parity(got, ref, lambda i: oracle.eri_batch_long_double(basis, q[i]), what="variant %s" % (cls,),
                          allow_adjudication=sum(cls) > 8)
        print("ok", cls, "tier", tr or rcg.class_info(cls)["tier"], "max scaled err %.2e" % r["max_scaled"], "adjudicated", r["adjudicated"])


if __name__ == "__main__":
    main()
