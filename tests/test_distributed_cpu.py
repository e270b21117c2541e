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

from paper_2206_01580_b200.distributed import (shard_range, allreduce_normal_equations, max_over_ranks,
                                                NormalEquationsReducer, pack_lower_reference, unpack_lower_reference,
                                                allreduce_forces)


def test_shard_range_partitions():
    for n in (0, 1, 7, 1000):
        for world in (1, 2, 3, 8):
            got = [shard_range(n, r, world) for r in range(world)]
            assert got[0][0] == 0 and got[-1][1] == n
            assert all(got[i][1] == got[i + 1][0] for i in range(world - 1))
            sizes = [b - a for a, b in got]
            assert max(sizes) - min(sizes) <= 1


def test_pack_lower_roundtrip():
    rng = np.random.default_rng(0)
    for D in (1, 2, 7, 33):
        A = rng.standard_normal((D + 3, D)).astype(np.float32)
        S = torch.from_numpy(A.T @ A)
        p = pack_lower_reference(S)
        assert p.numel() == D * (D + 1) // 2
        for i in range(D):                       # row i holds i + 1 entries at offset i (i + 1) / 2
            assert torch.equal(p[i * (i + 1) // 2: i * (i + 1) // 2 + i + 1], S[i, : i + 1])
        assert torch.equal(unpack_lower_reference(p, D), S)


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
          and t == float(world) and np.array_equal(ZtZ.numpy(), ZtZ.numpy().T))
    # persistent reducer, ZtZ only, twice in a row (buffer reuse)
    red = NormalEquationsReducer(16, "cpu")
    for _ in range(2):
        Z2 = torch.from_numpy(A[lo:hi].T @ A[lo:hi])
        red.allreduce(Z2, None)
        ok = ok and np.allclose(Z2.numpy(), A.T @ A, rtol=1e-5, atol=1e-5)
    # inference sharded over atoms: forces scattered by every rank are summed
    F = torch.zeros((37, 3)); F[lo:hi] = 1.0; F[(lo + 5) % 37] += 2.0
    allreduce_forces(F)
    ok = ok and abs(float(F.sum()) - (37 * 3 + 2.0 * 3 * world)) < 1e-4
    ret[rank] = bool(ok)
    dist.destroy_process_group()


def test_allreduce_normal_equations_gloo_world2():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    mgr = mp.Manager()
    ret = mgr.dict()
    mp.spawn(_worker, args=(2, port, ret), nprocs=2, join=True)
    assert ret[0] and ret[1]
