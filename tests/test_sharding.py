"""N > 1 host logic on CPU: world_size-2 gloo processes (no GPU): slices tile the list, the timing
reduction is a max over ranks, and the union of per-rank oracle results equals the single-process one."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2605_10312_b200 import sharding, workloads


def test_shard_slices_tile():
    for n in (0, 1, 7, 100, 100003):
        for world in (1, 2, 3, 8):
            sl = [sharding.shard_slice(n, r, world) for r in range(world)]
            assert sl[0][0] == 0 and sl[-1][1] == n
            assert all(sl[i][1] == sl[i + 1][0] for i in range(world - 1))
            sizes = [b - a for a, b in sl]
            assert max(sizes) - min(sizes) <= 1


def test_shard_rows_tile_and_balance():
    """units of a screened pass are cut by bra rows at equal shares of the surviving quartets: the ranks' ranges tile the rows, no row
    is split, and the quartet counts differ by less than the largest row."""
    rng = np.random.default_rng(3)
    for n in (1, 2, 17, 1000):
        cnt = rng.integers(0, 500, n)
        cnt[rng.integers(0, n)] = 0
        offs = np.concatenate([[0], np.cumsum(cnt)])
        for world in (1, 2, 3, 8):
            rng_ = [sharding.shard_rows(offs, r, world) for r in range(world)]
            assert rng_[0][0] == 0 and rng_[-1][1] == n
            assert all(rng_[i][1] == rng_[i + 1][0] for i in range(world - 1))
            share = [int(offs[hi] - offs[lo]) for lo, hi in rng_]
            assert sum(share) == int(offs[-1])
            assert max(share) - min(share) <= 2 * int(cnt.max()) + 1
    assert sharding.shard_rows(np.array([0, 0, 0]), 1, 2)[1] == 2          # a unit with no survivors


def _worker(rank, world, port, ret):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import oracle
    basis, q = workloads.cfg1(41)
    lo, hi = sharding.shard_slice(len(q), rank, world)
    part = oracle.eri_batch(basis, q[lo:hi], nthreads=1)
    tmax = sharding.max_over_ranks(1.0 + rank)
    # the collective of a multi-GPU Fock build: every rank's partial Jt, Kt summed in place
    Jt = torch.full((5, 5), float(rank + 1), dtype=torch.float64)
    Kt = torch.arange(25, dtype=torch.float64).reshape(5, 5) * (rank + 1)
    sharding.allreduce_sum_([Jt, Kt])
    assert float(Jt[0, 0]) == 3.0 and torch.equal(Kt, torch.arange(25, dtype=torch.float64).reshape(5, 5) * 3)
    gathered = [None] * world
    dist.all_gather_object(gathered, (lo, hi, part))
    if rank == 0:
        ret["tmax"] = tmax
        ret["parts"] = gathered
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_gloo():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    mgr = mp.Manager()
    ret = mgr.dict()
    mp.spawn(_worker, args=(2, port, ret), nprocs=2, join=True)
    assert ret["tmax"] == 2.0
    import oracle
    basis, q = workloads.cfg1(41)
    full = oracle.eri_batch(basis, q, nthreads=1)
    got = np.concatenate([p for (_, _, p) in sorted(ret["parts"], key=lambda t: t[0])])
    assert got.shape == full.shape and np.array_equal(got, full)
