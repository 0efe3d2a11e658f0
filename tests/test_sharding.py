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


def _worker(rank, world, port, ret):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import oracle
    basis, q = workloads.cfg1(41)
    lo, hi = sharding.shard_slice(len(q), rank, world)
    part = oracle.eri_batch(basis, q[lo:hi], nthreads=1)
    tmax = sharding.max_over_ranks(1.0 + rank)
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
