"""Multi-GPU plumbing (one process per GPU, torch.distributed).  The path shards over molecules: every rank
builds its own rows of Z / G and its local normal equations with no data-path collective; the only exchange
step is the sum of the [D, D] + [D] normal equations, one all-reduce over NCCL.
Host-side logic only; covered on CPU with gloo (tests/test_distributed_cpu.py)."""
from __future__ import annotations

import torch
import torch.distributed as dist


def shard_range(n_units: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous, balanced [lo, hi) slice of n_units for `rank` (sizes differ by at most one)."""
    base, extra = divmod(n_units, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def allreduce_normal_equations(ZtZ: torch.Tensor, Zty: torch.Tensor | None) -> None:
    """In-place sum over ranks of the local normal equations (eq. 16-17 are sums over rows)."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return
    dist.all_reduce(ZtZ, op=dist.ReduceOp.SUM)
    if Zty is not None:
        dist.all_reduce(Zty, op=dist.ReduceOp.SUM)


def max_over_ranks(value: float, device) -> float:
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return value
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
