"""Multi-GPU plumbing of the bench: the path shards over independent problems -- one
inverse-design problem per rank, no data-path collective.  This module holds the only host logic the N > 1
run adds: which problem a rank works on and how the per-rank times combine into the whole-job figure.
It has none of the method's arithmetic."""
from __future__ import annotations

import torch
import torch.distributed as dist


def problem_seed(base_seed: int, rank: int) -> int:
    """Every rank draws its own design (rho) from its own seed; rank 0 is the single-GPU problem."""
    return base_seed + rank


def max_over_ranks(ms_local: float, device=None) -> float:
    """Device time of the slowest rank (the job is as slow as its slowest problem)."""
    t = torch.tensor([ms_local], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(cells_steps_per_rank: int, reps: int, ms_max: float, world: int) -> float:
    """Mcells/s summed over ranks: every rank processed cells_steps_per_rank * reps cell updates in ms_max."""
    return world * cells_steps_per_rank * reps / (ms_max * 1e-3) / 1e6
