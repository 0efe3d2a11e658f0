"""Multi-GPU host logic.  The integral path shards over independent quartets (disjoint output rows, basis
replicated per GPU): contiguous slices of a class's quartet list, no data-path collective.
A Fock build has the paper's one cross-GPU step ("final J/K-matrix reduction"): every rank digests its share of
each unit of the screened pass into its own Jt, Kt, and ONE all-reduce (sum) of the two matrices follows (
NCCL over NVLink for CUDA tensors, gloo in the CPU tests)."""


def shard_slice(n, rank, world):
    """contiguous [lo, hi) of n items for `rank`; sizes differ by at most one, slices tile [0, n)."""
    base, rem = divmod(int(n), int(world))
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def max_over_ranks(value, device="cpu"):
    """max of a python float over all ranks (identity when torch.distributed is not initialised)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def shard_rows(offs, rank, world):
    """bra rows [lo, hi) of one unit of a screened pass for `rank`: offs = exclusive prefix sum (length n + 1) of the surviving quartets per
    bra row; boundary r is the first row whose prefix reaches r/world of the total, so the ranks' ranges tile [0, n) and carry
    about the same number of quartets (a row is never split)."""
    import numpy as np
    offs = np.asarray(offs)
    n, total = len(offs) - 1, int(offs[-1])

    def bound(r):
        return n if r >= world else int(np.searchsorted(offs[:-1], (total * r + world - 1) // world, side="left"))

    return bound(rank), bound(rank + 1)


def allreduce_sum_(tensors):
    """in-place sum over all ranks of every tensor in the list (identity when torch.distributed is not initialised or world = 1)."""
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return tensors
    for t in tensors:
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return tensors
