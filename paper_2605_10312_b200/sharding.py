"""Multi-GPU host logic.  The path shards over independent quartets (disjoint output rows, basis
replicated per GPU): contiguous slices of a class's quartet list, no data-path collective
(the paper's only cross-GPU step is the J/K reduction, out of scope).
torch.distributed is used for the timing reduction only."""


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
