"""Multi-GPU plumbing (one process per GPU, torch.distributed).  The path shards over molecules: every rank builds its
own rows of Z / G and its local normal equations with no data-path collective; the only exchange step of training is
the sum of the normal equations over ranks.  ZtZ is symmetric, so the exchange moves the
row-packed lower triangle (D (D + 1) / 2 floats, packed / unpacked by the library's kernels) plus Zty in ONE NCCL
all-reduce.  Inference shards over molecules too (energies and forces of a molecule depend on that molecule only);
a single huge cell (config 5) shards over atoms with the neighbour-scattered forces all-reduced (`allreduce_forces`).
Host-side logic only; covered on CPU with gloo (tests/test_distributed_cpu.py)."""
from __future__ import annotations

import torch
import torch.distributed as dist


def shard_range(n_units: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous, balanced [lo, hi) slice of n_units for `rank` (sizes differ by at most one)."""
    base, extra = divmod(n_units, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def _active() -> bool:
    return dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1


def pack_lower_reference(ZtZ: torch.Tensor) -> torch.Tensor:
    """Row-packed lower triangle with torch ops (small D only: CPU tests and a cross-check of the CUDA kernels)."""
    D = ZtZ.shape[0]
    i, j = torch.tril_indices(D, D, device=ZtZ.device)
    return ZtZ[i, j].contiguous()


def unpack_lower_reference(packed: torch.Tensor, D: int) -> torch.Tensor:
    out = torch.zeros((D, D), dtype=packed.dtype, device=packed.device)
    i, j = torch.tril_indices(D, D, device=packed.device)
    out[i, j] = packed
    out[j, i] = packed
    return out


class NormalEquationsReducer:
    """Sums (ZtZ, Zty) over ranks in place: pack the lower triangle + Zty into one persistent buffer, one all-reduce,
    unpack (both triangles).  On CUDA tensors the library's pack / unpack kernels are used; on CPU tensors (gloo
    tests) the torch reference above."""

    def __init__(self, D: int, device):
        self.D = D
        self.n_tri = D * (D + 1) // 2
        self.buf = torch.empty((self.n_tri + D,), dtype=torch.float32, device=device)

    def allreduce(self, ZtZ: torch.Tensor, Zty: torch.Tensor | None) -> None:
        if not _active():
            return
        tri, tail = self.buf[: self.n_tri], self.buf[self.n_tri:]
        if ZtZ.is_cuda:
            from . import qmll_pack_lower, qmll_unpack_lower
            qmll_pack_lower(ZtZ, tri)
        else:
            tri.copy_(pack_lower_reference(ZtZ))
        if Zty is not None:
            tail.copy_(Zty)
        else:
            tail.zero_()
        dist.all_reduce(self.buf, op=dist.ReduceOp.SUM)
        if ZtZ.is_cuda:
            qmll_unpack_lower(tri, ZtZ)
        else:
            ZtZ.copy_(unpack_lower_reference(tri, self.D))
        if Zty is not None:
            Zty.copy_(tail)


def allreduce_normal_equations(ZtZ: torch.Tensor, Zty: torch.Tensor | None) -> None:
    """One-shot form of NormalEquationsReducer (allocates the exchange buffer on every call)."""
    if _active():
        NormalEquationsReducer(ZtZ.shape[0], ZtZ.device).allreduce(ZtZ, Zty)


def allreduce_forces(forces: torch.Tensor) -> None:
    """Inference on one cell sharded over atoms (config 5): every rank scatters force contributions of ITS atoms'
    neighbour blocks to any atom of the cell, so the [n_atoms, 3] forces are summed over ranks."""
    if _active():
        dist.all_reduce(forces, op=dist.ReduceOp.SUM)


def max_over_ranks(value: float, device) -> float:
    if not _active():
        return value
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
