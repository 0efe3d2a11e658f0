"""CPU oracle (TEST INFRASTRUCTURE, not the product).  See oracle/eri_oracle.c and
oracle/eri_grad_oracle.c (first derivatives).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this package.  It imports nothing from paper_2605_10312_b200.
"""
from .oracle import (bf_offsets, eri_tensor, jk_dense, build, boys, boys_quadrature, c2s_matrix, eri_batch, num_threads,
                     build_long_double, eri_batch_long_double, build_grad, eri_grad_batch,
                     build_grad_long_double, eri_grad_batch_long_double)  # noqa: F401
