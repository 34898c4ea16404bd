"""Multi-GPU = replicas only (BASELINE.json:north_star: "nothing here is sharded or uses
collectives between GPUs").  Each rank solves its own copy of the workload on its own GPU; the
only cross-rank traffic is the timing protocol below (a barrier and a MAX reduction of the
per-rank elapsed time).  Kept free of CUDA so that the N>1 logic is testable with gloo on CPU.
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def world():
    if dist.is_available() and dist.is_initialized():
        return dist.get_world_size(), dist.get_rank()
    return 1, 0


def barrier():
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def max_over_ranks(ms_local: float, device="cpu") -> float:
    """Slowest rank's time: the job is done when the last replica is."""
    n, _ = world()
    if n == 1:
        return float(ms_local)
    t = torch.tensor([float(ms_local)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def ns_per_cell(ms_step: float, cells_per_rank: int, n_ranks: int) -> float:
    """Whole-job metric: every rank processed `cells_per_rank` cells in `ms_step` (weak scaling)."""
    return ms_step * 1e6 / (cells_per_rank * n_ranks)
