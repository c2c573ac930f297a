"""Host-side logic of the multi-GPU path: orbits are independent, so ranks own
contiguous orbit-index ranges and no collective touches the data path.  The only communication is the
max-over-ranks of each rank's device time (one scalar), which bench.py needs for the job throughput.

Backend-agnostic (nccl on GPUs, gloo in the CPU tests): tensors are created on the device passed in.
"""
import numpy as np

from .workloads import Workload, shard_range


def rank_rows(n_rows_per_rank: int, rank: int, world_size: int):
    """Row range [lo, hi) of a grid widened to n_rows_per_rank * world_size rows (weak scaling)."""
    return shard_range(n_rows_per_rank * world_size, rank, world_size)


def rank_shard(w: Workload, n_rows_per_rank: int, n_cols: int, rank: int, world_size: int) -> Workload:
    """The slice of a row-major (rows x n_cols) grid workload that `rank` integrates."""
    lo, hi = rank_rows(n_rows_per_rank, rank, world_size)
    return w.subset(np.arange(lo * n_cols, hi * n_cols))


def max_over_ranks(value: float, device=None) -> float:
    """all_reduce(MAX) of one float64 scalar; identity when torch.distributed is not initialised."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, device=None) -> float:
    """all_reduce(SUM) of one float64 scalar; identity when torch.distributed is not initialised."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def job_throughput(units_per_rank: float, world_size: int, n_timed: int, local_ms: float, device=None) -> float:
    """Whole-job units/s: all ranks' units over the slowest rank's device time (bench.py contract)."""
    return units_per_rank * world_size * n_timed / (max_over_ranks(local_ms, device) * 1e-3)
