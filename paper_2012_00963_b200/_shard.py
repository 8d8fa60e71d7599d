"""Multi-GPU plumbing of the photon path: histories are independent and keyed by photon id, so
a run shards by id range with NO data-path collective; the only exchange is one sum of the additive tallies
(histograms, sums of squared weights, counters) at the end of a run.  One process per GPU; `torch.distributed`
(NCCL on GPUs, gloo in the CPU tests) carries that sum.  No method arithmetic lives here.
"""
from __future__ import annotations

import numpy as np


def shard_photons(n_total: int, rank: int, world: int, first_photon_id: int = 0) -> tuple[int, int]:
    """Contiguous id range of `rank`: (first id, count).  The ranges of all ranks tile
    [first_photon_id, first_photon_id + n_total) exactly; the first n_total % world ranks get one more."""
    if world < 1 or not (0 <= rank < world) or n_total < 0:
        raise ValueError("need world >= 1, 0 <= rank < world, n_total >= 0")
    base, rem = divmod(int(n_total), world)
    count = base + (1 if rank < rem else 0)
    start = int(first_photon_id) + rank * base + min(rank, rem)
    return start, count


def shard_units(n_units: int, rank: int, world: int) -> range:
    """Whole (cloud, snapshot) units per rank (configs 3 and 4): unit u goes to rank u % world."""
    if world < 1 or not (0 <= rank < world) or n_units < 0:
        raise ValueError("need world >= 1, 0 <= rank < world, n_units >= 0")
    return range(rank, n_units, world)


ADDITIVE_STATS = ("detected", "underflow", "overflow", "escaped", "absorbed_particles", "absorbed_surface",
                  "roulette_killed", "roulette_gained", "truncated", "histories", "particle_events",
                  "surface_reflections")


def allreduce_tallies(hist, hist2=None, group=None):
    """In-place sum over ranks of the additive tallies (torch tensors, CPU for gloo / CUDA for NCCL).
    Tallies are integer multiples of 2^-31 below 2^53 * 2^-31, so the float64 sums are exact and the result
    does not depend on the reduction order (bit-identical to a one-GPU run over the union of the id ranges)."""
    import torch.distributed as dist
    if not dist.is_initialized() or dist.get_world_size(group) == 1:
        return
    dist.all_reduce(hist, op=dist.ReduceOp.SUM, group=group)
    if hist2 is not None:
        dist.all_reduce(hist2, op=dist.ReduceOp.SUM, group=group)


def merge_stats(stats_list):
    """Merges per-rank structured stats arrays (STATS_DTYPE) of the same units: additive fields are summed,
    max_events_in_history is the maximum."""
    out = np.array(stats_list[0], copy=True)
    for s in stats_list[1:]:
        for k in ADDITIVE_STATS:
            out[k] = out[k] + s[k]
        out["max_events_in_history"] = np.maximum(out["max_events_in_history"], s["max_events_in_history"])
    return out
