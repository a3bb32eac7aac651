"""Multi-GPU plumbing of the npFEM hot path: one process per GPU, cells sharded, NO collective on
the data path (cells are independent given their forces; the paper
itself hands whole cells to cores / GPUs).  torch.distributed is used only to line
the ranks up around a timed region and to take the max of a per-rank time.

Nothing here touches CUDA by itself: the helpers run under the `gloo` backend on CPU (tests) and
under `nccl` on GPUs (bench.py).
"""
from __future__ import annotations

from typing import Tuple

import torch
import torch.distributed as dist


def cell_range(n_cells: int, rank: int, world: int) -> Tuple[int, int]:
    """Contiguous range [lo, hi) of cell indices owned by `rank` when n_cells cells are spread
    over `world` ranks (strong scaling of one suspension): sizes differ by at most one cell and
    the ranges tile [0, n_cells) in rank order."""
    if world <= 0 or not (0 <= rank < world) or n_cells < 0:
        raise ValueError("need 0 <= rank < world and n_cells >= 0")
    base, extra = divmod(n_cells, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def rank_seed(seed: int, rank: int) -> list:
    """Seed material for the rank's own cells under weak scaling (every rank its own suspension):
    distinct per rank, reproducible, independent of the world size."""
    return [int(seed), 0xCE11, int(rank)]


def max_over_ranks(value: float, device="cpu") -> float:
    """Max of a per-rank scalar (a device-timed duration) over all ranks; the value itself when
    torch.distributed is not initialised (single process)."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, device="cpu") -> float:
    """Sum of a per-rank scalar (units processed) over all ranks."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def aggregate_throughput(units_this_rank: float, ms_this_rank: float, device="cpu") -> float:
    """Whole-job throughput in units per second: all ranks' units over the slowest rank's time."""
    return sum_over_ranks(units_this_rank, device) / (max_over_ranks(ms_this_rank, device) * 1e-3)
