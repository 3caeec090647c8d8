"""Multi-GPU plumbing of bench.py: replicas only.

The path does not shard in this build (north_star: one GPU, no collectives), so N ranks run N independent
replicas of the same two-site problem.  The only cross-rank traffic is the timing protocol: a barrier around the
timed region and a MAX reduction of the per-rank step time; the job's value is N x (work of one replica) / that
time.  Backend "nccl" on GPUs, "gloo" in the CPU tests (tests/test_replicas_gloo.py).
"""
from __future__ import annotations


def init(backend: str, device=None):
    """Initialise torch.distributed from the torchrun environment; returns (rank, world)."""
    import os
    import torch.distributed as dist
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    if world > 1 and not dist.is_initialized():
        if device is not None:
            dist.init_process_group(backend, device_id=device)
        else:
            dist.init_process_group(backend)
    return rank, world


def barrier(world: int):
    if world > 1:
        import torch.distributed as dist
        dist.barrier()


def max_over_ranks(value: float, world: int, device=None) -> float:
    """MAX over ranks of a per-rank scalar (the step time in ms)."""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_throughput(units_per_replica: float, ms_local: float, world: int, device=None):
    """(ms_max, whole-job units per second) for `world` replicas that each processed `units_per_replica`."""
    ms_max = max_over_ranks(ms_local, world, device)
    return ms_max, world * units_per_replica / (ms_max * 1e-3)
