"""Multi-GPU sharding of the path: photons and navigation queries are independent units,
and photon i depends only on (seed, global id i), so contiguous id ranges per rank give a result that does
not depend on the partition.  Geometry is replicated.  The one exchange step of transport is the sum of
the per-volume tallies (and of the run statistics) at the end of a run -- an all-reduce over NCCL on GPUs,
gloo in the CPU tests.  Navigation queries are a pure map: no collective."""
from __future__ import annotations


def shard_range(n_total: int, rank: int, world: int):
    """Contiguous [first, first + count) range of rank `rank` out of `world`; remainders go to the low ranks."""
    if world <= 0 or not (0 <= rank < world) or n_total < 0:
        raise ValueError("bad shard arguments")
    base, rem = divmod(n_total, world)
    first = rank * base + min(rank, rem)
    return first, base + (1 if rank < rem else 0)


STAT_KEYS = ("n_steps", "n_compton", "n_pe", "n_pair", "n_cut", "n_escaped", "n_stuck", "n_photons", "n_rayleigh",
             "e_escaped", "e_stuck", "e_source", "e_deposited")


def allreduce_tally(edep, stats: dict, group=None):
    """Sum the per-volume edep tensor (in place) and the additive run statistics over all ranks."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return edep, dict(stats)
    dist.all_reduce(edep, op=dist.ReduceOp.SUM, group=group)
    vec = torch.tensor([float(stats.get(k, 0)) for k in STAT_KEYS], dtype=torch.float64, device=edep.device)
    dist.all_reduce(vec, op=dist.ReduceOp.SUM, group=group)
    out = dict(stats)
    for k, v in zip(STAT_KEYS, vec.tolist()):
        out[k] = int(round(v)) if k.startswith("n_") else v
    return edep, out
