"""Host-side logic of the multi-GPU path: orbits are independent, so every rank owns a
fixed subset of the grid rows and no collective touches the data path.  Rows are dealt round-robin (global row i
belongs to rank i mod N): the strong-field rows (small r0: dropped and chaotic cells, more Gauss-Newton steps) and
the calm ones are then spread evenly, and since the job time is the maximum over ranks a contiguous split would
measure the imbalance between the first and the last r0 band instead of the machine.  The only communication is
the max-over-ranks of each rank's device time (one scalar), which bench.py needs for the job throughput.

Backend-agnostic (nccl on GPUs, gloo in the CPU tests): tensors are created on the device passed in.
"""
import numpy as np

from .workloads import Workload


def rank_rows(n_rows_per_rank: int, rank: int, world_size: int) -> np.ndarray:
    """Global row indices of `rank` in a grid widened to n_rows_per_rank * world_size rows (weak scaling):
    rank, rank + N, rank + 2N, ... (round-robin)."""
    return np.arange(rank, n_rows_per_rank * world_size, world_size)


def rank_orbits(n_rows_per_rank: int, n_cols: int, rank: int, world_size: int) -> np.ndarray:
    """Global orbit indices (row-major, index = row * n_cols + col) of `rank`, in the order it integrates them."""
    rows = rank_rows(n_rows_per_rank, rank, world_size)
    return (rows[:, None] * n_cols + np.arange(n_cols)[None, :]).ravel()


def rank_shard(w: Workload, n_rows_per_rank: int, n_cols: int, rank: int, world_size: int) -> Workload:
    """The part of a row-major (rows x n_cols) grid workload that `rank` integrates."""
    return w.subset(rank_orbits(n_rows_per_rank, n_cols, rank, world_size))


def strong_orbits(n_rows: int, n_cols: int, rank: int, world_size: int) -> np.ndarray:
    """Strong scaling: the SAME (n_rows x n_cols) grid dealt over the ranks, row i to rank i mod N.  Ranks hold
    ceil(n_rows / N) or floor(n_rows / N) rows (314 rows over 8 ranks: 40, 40, 39, ...: 12 560 or 12 246 orbits)."""
    rows = np.arange(rank, n_rows, world_size)
    return (rows[:, None] * n_cols + np.arange(n_cols)[None, :]).ravel()


def strong_shard(w: Workload, n_rows: int, n_cols: int, rank: int, world_size: int) -> Workload:
    return w.subset(strong_orbits(n_rows, n_cols, rank, world_size))


def scatter_back(parts, n_rows_per_rank: int, n_cols: int, world_size: int) -> np.ndarray:
    """Inverse of the split for an output array: parts[r] has the rank-local orbit axis last; returns the global
    array (outputs of different ranks are disjoint slices, so this is a permutation, not a reduction)."""
    n = n_rows_per_rank * world_size * n_cols
    first = np.asarray(parts[0])
    out = np.empty(first.shape[:-1] + (n,), dtype=first.dtype)
    for r, part in enumerate(parts):
        out[..., rank_orbits(n_rows_per_rank, n_cols, r, world_size)] = np.asarray(part)
    return out


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
