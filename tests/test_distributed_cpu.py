"""World-size-2 gloo test (CPU) of the multi-GPU host logic: molecules are sharded across ranks, each rank forms
its local normal equations, and one all-reduce gives the full ones.  The per-rank
products here are plain numpy stand-ins for the device results; what is under test is the sharding + reduction."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2206_01580_b200.distributed import shard_range, allreduce_normal_equations, max_over_ranks


def test_shard_range_partitions():
    for n in (0, 1, 7, 1000):
        for world in (1, 2, 3, 8):
            got = [shard_range(n, r, world) for r in range(world)]
            assert got[0][0] == 0 and got[-1][1] == n
            assert all(got[i][1] == got[i + 1][0] for i in range(world - 1))
            sizes = [b - a for a, b in got]
            assert max(sizes) - min(sizes) <= 1


def _worker(rank, world, port, ret):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    rng = np.random.default_rng(3)
    A = rng.standard_normal((37, 16)).astype(np.float32)      # 37 "molecules" (rows), D = 16
    y = rng.standard_normal(37).astype(np.float32)
    lo, hi = shard_range(37, rank, world)
    ZtZ = torch.from_numpy(A[lo:hi].T @ A[lo:hi])
    Zty = torch.from_numpy(A[lo:hi].T @ y[lo:hi])
    allreduce_normal_equations(ZtZ, Zty)
    t = max_over_ranks(float(rank + 1), "cpu")
    ok = (np.allclose(ZtZ.numpy(), A.T @ A, rtol=1e-5, atol=1e-5) and np.allclose(Zty.numpy(), A.T @ y, rtol=1e-5, atol=1e-5)
          and t == float(world))
    ret[rank] = bool(ok)
    dist.destroy_process_group()


def test_allreduce_normal_equations_gloo_world2():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    mgr = mp.Manager()
    ret = mgr.dict()
    mp.spawn(_worker, args=(2, port, ret), nprocs=2, join=True)
    assert ret[0] and ret[1]
