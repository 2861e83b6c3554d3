"""Multi-GPU plumbing: "replicas only".

Cells are independent and the path has no exchange step, so N GPUs run N
independent replicas of the workload, one process per GPU; the only cross-rank operation is the
MAX of the measured time.  Works on any torch.distributed backend (nccl on GPUs, gloo in the CPU
tests)."""
from __future__ import annotations


def replica_seed(base_seed: int, rank: int) -> int:
    """Seed of rank's replica of the synthetic disc (rank 0 = the single-GPU workload)."""
    return int(base_seed) + 1000 * int(rank)


def max_over_ranks(seconds: float, world: int, device=None) -> float:
    """MAX over ranks of a per-rank duration (the slowest replica sets the job's time)."""
    if world <= 1:
        return float(seconds)
    import torch
    import torch.distributed as dist
    on_gpu = dist.get_backend() == "nccl"
    t = torch.tensor([float(seconds)], dtype=torch.float64, device=device if on_gpu else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_throughput(units_per_rank: int, steps: int, seconds: float, world: int, device=None) -> float:
    """Whole-job units/s: every rank processed units_per_rank * steps units; time = max over ranks."""
    return world * units_per_rank * steps / max_over_ranks(seconds, world, device)
