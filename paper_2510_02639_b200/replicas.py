"""Multi-GPU plumbing of bench.py: the hot path has no exchange step (every source point is independent,
PAPER.md P:101; DESIGN.md 9 "replicas only"), so N GPUs run N independent replicas and the only
communication is the timing reduction: a barrier and the MAX over ranks of the device-measured times.
Works on any torch.distributed backend (NCCL on the GPU box, gloo in the CPU tests)."""
from __future__ import annotations


def max_over_ranks(values, device=None):
    """Element-wise maximum over all ranks of a short list of floats (identity when not distributed)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t.cpu()]


def aggregate_throughput(units_per_rank: int, world: int, ms_per_step_max: float) -> float:
    """Whole-job units/s of `world` replicas that each processed units_per_rank per step; the step time is the
    slowest rank's ("weak" scaling: per-GPU work is fixed as N grows)."""
    return world * units_per_rank / (ms_per_step_max * 1e-3)
