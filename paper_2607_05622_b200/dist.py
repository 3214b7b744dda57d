"""Multi-GPU plumbing for bench.py: the path shards over independent
problems -- every rank runs whole sweeps on its own batch of amplitude sets for the same molecule; there is no
data-path collective, only the max-over-ranks of the device time.  Backend-agnostic so that the logic is covered by
world_size-2 gloo tests on CPU."""
from __future__ import annotations

import numpy as np


def rank_amplitudes(workload, rank: int) -> np.ndarray:
    """Amplitude batch of one rank: rank 0 keeps the workload's seeded T; other ranks draw their own (same shape,
    same distribution), seeded by the rank."""
    if rank == 0:
        return workload.T
    rng = np.random.default_rng(1000 + rank)
    return 1e-2 * rng.standard_normal(workload.T.shape)


def max_over_ranks(value: float, device=None) -> float:
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_builds_per_s(n_builds_per_rank: int, world: int, ms_per_step_max: float) -> float:
    """weak scaling: every rank does n_builds_per_rank builds per step; the job's rate uses the slowest rank's time"""
    return world * n_builds_per_rank / (ms_per_step_max * 1e-3)
