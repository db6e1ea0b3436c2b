"""Host logic of the multi-GPU mode: replicas only.  The path does not shard a matrix and has no data-path
collective; N ranks run N independent replicas (seed = rank) and only the TIMES are reduced: max over ranks, because the job is
finished when its slowest replica is.  Works with any torch.distributed backend (nccl on GPUs, gloo in the CPU tests)."""
from __future__ import annotations

import torch


def replica_seed(rank: int, base_seed: int = 0) -> int:
    """Seed of the synthetic problem a rank solves: distinct per rank, reproducible."""
    return base_seed + rank


def max_over_ranks(values, dist=None, device="cpu"):
    """Element-wise maximum of a list of per-rank floats over all ranks (identity without a process group)."""
    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t.tolist()]


def job_value(seconds_per_step_max: float) -> float:
    """The bench metric is a time per step (lower is better): the whole job's value is the slowest replica's time."""
    return seconds_per_step_max
