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


# ---------------------------------------------------------------------------------------------------------------
# Sharding ONE sweep over ranks (second alternative): the n_D = n_tau x n_T densities of a sweep are
# independent builds, so rank r takes densities r, r + world, r + 2 world, ... and recomputes the integrals for its
# share; there is no data-path collective.  Results are gathered only when the caller wants the whole batch on one
# rank (tests, checks), never inside a timed step.
def density_shard(n_densities: int, rank: int, world: int) -> np.ndarray:
    """Indices (into the sweep's density batch) owned by `rank`: round-robin, so Laplace points and amplitude sets
    are spread evenly and every rank gets the same count up to one."""
    if not (0 <= rank < world):
        raise ValueError("rank outside the world")
    return np.arange(rank, n_densities, world)


def shard_sizes(n_densities: int, world: int) -> list:
    return [len(range(r, n_densities, world)) for r in range(world)]


def gather_sharded(local, n_densities: int):
    """Inverse of density_shard for a result tensor: every rank passes its [n_local, ...] block (torch tensor on the
    backend's device) and gets the full [n_densities, ...] batch in sweep order.  Uses all_gather on blocks padded to
    the largest shard (the only collective, outside any timed region)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return local
    world, rank = dist.get_world_size(), dist.get_rank()
    sizes = shard_sizes(n_densities, world)
    if local.shape[0] != sizes[rank]:
        raise ValueError("local block does not match this rank's shard")
    nmax = max(sizes)
    pad = torch.zeros((nmax,) + tuple(local.shape[1:]), dtype=local.dtype, device=local.device)
    pad[:local.shape[0]] = local
    parts = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(parts, pad)
    full = torch.empty((n_densities,) + tuple(local.shape[1:]), dtype=local.dtype, device=local.device)
    for r in range(world):
        full[r::world] = parts[r][:sizes[r]]
    return full


def sharded_sweep_builds_per_s(n_densities: int, ms_per_step_max: float) -> float:
    """strong scaling: the job is ONE sweep of n_densities builds split over the ranks"""
    return n_densities / (ms_per_step_max * 1e-3)


# ---------------------------------------------------------------------------------------------------------------
# Sharding one build in the space of shell quartets (first alternative; 8(f) N5): every rank calls
# ctx.set_quartet_shard(rank, world), builds its partial J, K for ALL densities, and the partials are summed by ONE
# all-reduce of 2 nD N^2 doubles (NCCL over NVLink/NVSwitch on GPUs; gloo in the CPU test).  This is the path's only
# data-plane collective.
def allreduce_jk(J, K=None):
    """In-place SUM over ranks of the partial results (torch tensors on the backend's device)."""
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return
    dist.all_reduce(J, op=dist.ReduceOp.SUM)
    if K is not None:
        dist.all_reduce(K, op=dist.ReduceOp.SUM)
