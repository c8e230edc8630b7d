"""Multi-GPU = independent replicas: one process per GPU, each with its own plan, frames
dealt round-robin, NO data-path collective (the solve is a latency-bound ~10 MB working set).
Only the bench bookkeeping crosses ranks: a barrier and a max over ranks of the measured time."""
from __future__ import annotations

from typing import List


def frames_of_rank(n_frames: int, rank: int, world: int) -> List[int]:
    """Round-robin deal of frame indices: rank r gets r, r + world, r + 2 world, ..."""
    if world < 1 or not (0 <= rank < world):
        raise ValueError("bad rank / world size")
    return list(range(rank, n_frames, world))


def barrier(world: int) -> None:
    if world > 1:
        import torch.distributed as dist
        dist.barrier()


def max_over_ranks(value: float, world: int) -> float:
    """Max of a host scalar over all ranks (device-timed milliseconds in bench.py)."""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([float(value)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, world: int) -> float:
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([float(value)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())
