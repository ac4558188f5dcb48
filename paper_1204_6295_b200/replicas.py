"""Multi-GPU plumbing: replicas only.

The DISC hot path does not shard (north_star: one GPU; a z-slab split would need halo exchanges of ~20 slices
several times inside a 200 us iteration).  N GPUs therefore run N independent registrations -- one process per
GPU, no data-path collective.  What is left for `torch.distributed` is the bookkeeping below: which registrations
a rank owns, and the max-over-ranks reduction of the device-timed duration (whole-job throughput = total units
/ slowest rank).  Nothing here touches the method's arithmetic; the tests run it on CPU with the gloo backend.
"""
from __future__ import annotations


def shard_cases(n_cases: int, rank: int, world: int) -> list[int]:
    """indices of the independent registrations rank `rank` of `world` owns (round robin; disjoint, covering)"""
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    return list(range(rank, n_cases, world))


def max_over_ranks(value: float, dist=None, device="cpu") -> float:
    """MAX all-reduce of a per-rank scalar (the elapsed time); identity without a process group"""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    t = torch.tensor([value], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, dist=None, device="cpu") -> float:
    """SUM all-reduce of a per-rank scalar (units processed)"""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    t = torch.tensor([value], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def whole_job_throughput(units_this_rank: float, ms_this_rank: float, dist=None, device="cpu") -> tuple[float, float]:
    """(units of all ranks / max-over-ranks time [units/s], that time [ms])"""
    ms = max_over_ranks(ms_this_rank, dist, device)
    units = sum_over_ranks(units_this_rank, dist, device)
    return units / (ms * 1e-3), ms
