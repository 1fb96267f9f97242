"""Multi-GPU plumbing: independent replicas, no data-path collective.

The spectral Ewald path of one plan runs on one GPU (BASELINE.json north_star); N GPUs run N
independent evaluations (different force vectors / time steps).  The only cross-rank traffic
is the timing reduction of the benchmark: max over ranks of the device time, sum of the units.
Works on any torch.distributed backend (nccl on the GPU box, gloo in the CPU tests).
"""
from __future__ import annotations

SEED_STRIDE = 1000


def replica_seed(base_seed: int, rank: int) -> int:
    """Seed of rank `rank`'s synthetic batch: rank 0 is the BASELINE config's own seed."""
    return int(base_seed) + SEED_STRIDE * int(rank)


def aggregate(units: float, ms: float, device="cpu"):
    """(sum over ranks of units, max over ranks of ms).  No-op without an initialised process group."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(units), float(ms)
    t_sum = torch.tensor([float(units)], dtype=torch.float64, device=device)
    t_max = torch.tensor([float(ms)], dtype=torch.float64, device=device)
    dist.all_reduce(t_sum, op=dist.ReduceOp.SUM)
    dist.all_reduce(t_max, op=dist.ReduceOp.MAX)
    return float(t_sum.item()), float(t_max.item())


def throughput(units: float, ms: float, device="cpu") -> float:
    """Whole-job units per second: all ranks' units / the slowest rank's time."""
    u, m = aggregate(units, ms, device)
    return u / (m * 1e-3)
