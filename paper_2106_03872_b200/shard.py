"""State sharding for multi-GPU runs (Fig. 7).

Each state's H psi and each Taylor chain is independent of every other state, so a block is split into contiguous
state ranges, one per rank, with V and the projector tables replicated.  There is no collective on the path of H|psi> and
of the Taylor steps; torch.distributed supplies the barrier and the max-over-ranks timing in bench.py, and the one real
exchange step of a self-consistent propagation: the sum of the per-shard densities (Eq. 1, "requires a parallel reduction
over states") -- one all-reduce of N_p doubles per step (NCCL over NVLink on GPUs, gloo in the CPU tests).
"""
from __future__ import annotations

from typing import Tuple


def state_range(rank: int, world: int, nst: int) -> Tuple[int, int]:
    """Contiguous [s0, s1) of rank `rank`; sizes differ by at most one, lower ranks get the larger shards."""
    if not (0 <= rank < world) or nst < 0:
        raise ValueError("bad rank / world / nst")
    base, rem = divmod(nst, world)
    s0 = rank * base + min(rank, rem)
    return s0, s0 + base + (1 if rank < rem else 0)


def max_over_ranks(seconds: float) -> float:
    """Max over ranks of a timing (the job is as slow as its slowest rank).  No-op without a process group."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(seconds)
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([seconds], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def allreduce_density(dens):
    """Sum the per-rank partial densities (tdh_density of each rank's states) in place; no-op without a process group.

    `dens` is a float64 tensor of the grid's shape, on the GPU under NCCL, on the CPU under gloo.
    """
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(dens, op=dist.ReduceOp.SUM)
    return dens
