"""Multi-GPU plumbing: every (design, direction) pair is independent, so ranks take
disjoint direction slices of a replicated design batch and there is NO data-path collective.  The only
communication is bookkeeping through torch.distributed (NCCL on GPUs, gloo in the CPU tests): the max
of the per-rank step times, the sum of the per-rank unit counts, and an optional gather of the
per-rank force slices.
"""
import numpy as np
import torch
import torch.distributed as dist


def direction_slice(S_total, rank, world_size):
    """Interleaved slice rank::world_size of the global direction list (keeps every rank's directions
    spread over the whole sphere, so per-rank hit fractions -- and work -- match)."""
    if not (0 <= rank < world_size):
        raise ValueError("bad rank")
    return np.arange(rank, S_total, world_size)


def weak_scaling_directions(S_per_rank, rank, world_size, front_hemisphere=False):
    """Weak scaling: the job has S_per_rank * world_size Fibonacci directions; this rank's share."""
    from .workloads import fibonacci_sphere
    allv = fibonacci_sphere(S_per_rank * world_size, front_hemisphere)
    return allv[direction_slice(len(allv), rank, world_size)]


def combine_timing(step_seconds, units, device=None):
    """(max over ranks of the step time, sum over ranks of the units processed)."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(step_seconds), float(units)
    t = torch.tensor([float(step_seconds)], dtype=torch.float64, device=device)
    u = torch.tensor([float(units)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def gather_forces(local_forces, S_total):
    """local_forces [D, S_local, 3] of every rank -> [D, S_total, 3] in global direction order."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return local_forces
    world = dist.get_world_size()
    D = local_forces.shape[0]
    counts = [len(direction_slice(S_total, r, world)) for r in range(world)]
    pad = max(counts)
    buf = torch.zeros((D, pad, 3), dtype=local_forces.dtype, device=local_forces.device)
    buf[:, :local_forces.shape[1]] = local_forces
    parts = [torch.empty_like(buf) for _ in range(world)]
    dist.all_gather(parts, buf)
    out = torch.empty((D, S_total, 3), dtype=local_forces.dtype, device=local_forces.device)
    for r in range(world):
        out[:, direction_slice(S_total, r, world)] = parts[r][:, :counts[r]]
    return out
