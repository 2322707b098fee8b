"""Whole-job throughput of N independent replicas (the path is scoped to one GPU, so
``bench.py --gpus N`` runs N replicas of the same block and no data-path collective exists).

The only exchange between ranks is the clock: every rank times its own replica on its own device, the job
time is the maximum over ranks, and the job's value is the work of all ranks divided by that time.  Kept
apart from bench.py so that the world_size > 1 logic is covered by a gloo test on CPU.
"""
from __future__ import annotations


def job_time(local_seconds: float, device=None) -> float:
    """Maximum over ranks of a locally measured duration; the local value when no process group is up."""
    import torch
    import torch.distributed as dist

    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(local_seconds)
    if device is None:
        device = torch.device("cuda", torch.cuda.current_device()) if dist.get_backend() == "nccl" else torch.device("cpu")
    t = torch.tensor([float(local_seconds)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_value(cells_per_replica: int, steps: int, local_seconds: float, device=None):
    """(cell-updates/s of the whole job, job seconds): all replicas' work over the slowest replica's time."""
    import torch.distributed as dist

    world = dist.get_world_size() if (dist.is_available() and dist.is_initialized()) else 1
    seconds = job_time(local_seconds, device)
    return cells_per_replica * world * steps / seconds, seconds
