"""Energy sharding of the sweep across GPUs — host logic only.

The march, the specular boundary condition and the boundary stores never couple different energies, so rank r
of W owns a contiguous slice of the Matsubara table for all angles and trajectories; the un-finalised accumulator
fields (Re, Im of every order-parameter component's numerator, Jx, Jy, I: five for one component) are summed with ONE all-reduce per sweep (`sc_set_allreduce_hook`), after which every rank
applies Eq. 22 / Eq. 8 / Eq. 19 to the same summed accumulators.  The denominator of
Eq. 22 is a property of the whole table, so it is passed to every shard explicitly.
"""
from __future__ import annotations

import numpy as np


def energy_slice(n_energies: int, world: int, rank: int) -> slice:
    """Contiguous balanced slice of range(n_energies) owned by `rank`; slices are rounded to whole warps of
    32 energies when n_energies allows it (the march processes energies 32 lanes at a time)."""
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    unit = 32 if n_energies % 32 == 0 and n_energies // 32 >= world else 1
    blocks = n_energies // unit
    lo = (blocks * rank) // world * unit
    hi = (blocks * (rank + 1)) // world * unit
    return slice(lo, hi)


def matsubara_shard(t: float, n_energies: int, world: int, rank: int):
    """(z, w, denominator_sum) of this rank: z_n = i t (n + 1/2) for its slice, unit weights, and
    sum_{n < n_energies} 1/(n + 1/2) of the WHOLE table (reading R-A5)."""
    sl = energy_slice(n_energies, world, rank)
    n = np.arange(n_energies, dtype=np.float64)
    z = 1j * t * (n[sl] + 0.5)
    return z, np.ones(len(z)), float(np.sum(1.0 / (n + 0.5)))


def attach(ctx, t: float, n_energies: int, group=None):
    """Shard `ctx` (a ScContext created with the full n_matsubara) over torch.distributed: sets this rank's
    energy slice and an all-reduce hook on the five accumulator fields.  Returns the accumulator tensor."""
    import torch
    import torch.distributed as dist
    world, rank = dist.get_world_size(group), dist.get_rank(group)
    z, w, dsum = matsubara_shard(t, n_energies, world, rank)
    if len(z) == 0:
        raise ValueError("more ranks than energies")
    ctx.sc_set_energies(z, w, dsum)
    acc = torch.zeros((2 * ctx.n_components + 3, ctx.ny, ctx.nx), dtype=torch.float64, device=ctx.device)
    ctx.sc_set_allreduce_hook(acc, lambda: dist.all_reduce(acc, group=group))
    return acc
