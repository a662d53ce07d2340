"""Host-side logic of the multi-GPU mode (replicas only).

The path has no exchange step on one GPU and north_star keeps everything on one GPU, so N ranks advance N sets of
independent simulations; nothing here touches the data path. torch.distributed is used for two things only: the
barrier around the timed region and the max-over-ranks of the device time. Works with the `nccl` backend on GPUs
and with `gloo` on CPU (tests/test_replicas_gloo.py, world_size 2).
"""
from __future__ import annotations

import numpy as np


def replica_seed(base_seed: int, rank: int, replica: int, replicas_per_rank: int) -> int:
    """Distinct seed for every (rank, replica): no two simulations of a job share their initial noise."""
    return int(base_seed) + int(rank) * int(replicas_per_rank) + int(replica)


def perturb(c: np.ndarray, rank: int, replica: int, replicas_per_rank: int, amp: float = 1e-4) -> np.ndarray:
    """Deterministic per-replica offset of the conserved field (keeps every replica's state distinct in memory)."""
    return c + amp * (rank * replicas_per_rank + replica)


def max_over_ranks(value: float, device=None) -> float:
    """Max of a host scalar over all ranks (identity when torch.distributed is not initialised)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_throughput(units_per_rank: float, elapsed_ms_max: float, world_size: int) -> float:
    """Whole-job units/s: every rank processed `units_per_rank` units within the slowest rank's time."""
    return world_size * units_per_rank / (elapsed_ms_max * 1e-3)
