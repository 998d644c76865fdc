"""Multi-GPU plumbing (one process per GPU, torch.distributed): which maps a rank convolves and how
the timings of the ranks combine.

The path shards over INDEPENDENT maps (BASELINE.json north_star "Batch support for B maps sharing one
kernel"): every rank builds the same plan and convolves its own maps, so there is no data-path
collective; the only communication is the reduction of the timings.  The
functions here are backend agnostic (nccl on GPUs, gloo in the CPU tests) and hold no method
arithmetic.
"""
import numpy as np


def map_shard(n_maps, rank, world):
    """Indices of the maps rank `rank` of `world` convolves: contiguous, sizes differ by at most 1."""
    if not (0 <= rank < world) or n_maps < 0:
        raise ValueError("bad rank/world/n_maps")
    base, extra = divmod(n_maps, world)
    lo = rank * base + min(rank, extra)
    return list(range(lo, lo + base + (1 if rank < extra else 0)))


def rank_seeds(seeds, rank):
    """Seeds of the synthetic maps of one rank in the weak-scaling benchmark (distinct per rank)."""
    return [int(s) + 1000 * int(rank) for s in seeds]


def combine_timing(local_ms, local_units, group=None):
    """Whole-job throughput: (max over ranks of local_ms, sum over ranks of local_units).

    local_ms: sequence of times measured on this rank (each reduced with MAX);
    local_units: work this rank did in those times (pairs), reduced with SUM.  Without an
    initialised process group the local values are returned."""
    import torch
    import torch.distributed as dist
    ms = torch.tensor([float(x) for x in local_ms], dtype=torch.float64)
    units = torch.tensor([float(local_units)], dtype=torch.float64)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        if dist.get_backend(group) == "nccl":
            ms, units = ms.cuda(), units.cuda()
        dist.all_reduce(ms, op=dist.ReduceOp.MAX, group=group)
        dist.all_reduce(units, op=dist.ReduceOp.SUM, group=group)
    return [float(x) for x in ms.cpu()], float(units.cpu()[0])


def gather_outputs(local_out, n_maps, group=None):
    """All ranks' output maps in map order (list of numpy arrays); local_out follows map_shard()."""
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return [np.asarray(o) for o in local_out]
    world = dist.get_world_size(group)
    parts = [None] * world
    dist.all_gather_object(parts, [np.asarray(o) for o in local_out], group=group)
    out = [None] * n_maps
    for r in range(world):
        for i, o in zip(map_shard(n_maps, r, world), parts[r]):
            out[i] = o
    return out
