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


# ---------------------------------------------------------------------------------------------------
# One map over several ranks: latitude bands with overlap.  Rank r owns the input and
# output rows `out_rows` of band r (sc_band_partition); before the convolution it needs the overlap
# rows in_rows - out_rows from the ranks that own them (halo exchange, point to point), afterwards
# the bands are independent.  Maps are full-size N_pix tensors on every rank so that rows land at
# their global positions; only the band's rows are ever valid / touched.
# ---------------------------------------------------------------------------------------------------

def _ranges(rows):
    """(a, b, c, d) -> list of non-empty half-open pixel ranges."""
    a, b, c, d = (int(x) for x in rows)
    return [(lo, hi) for lo, hi in ((a, b), (c, d)) if hi > lo]


def _intersect(xs, ys):
    out = []
    for a, b in xs:
        for c, d in ys:
            lo, hi = max(a, c), min(b, d)
            if hi > lo:
                out.append((lo, hi))
    return sorted(out)


def _subtract(xs, ys):
    out = []
    for a, b in xs:
        cur = [(a, b)]
        for c, d in ys:
            nxt = []
            for lo, hi in cur:
                if d <= lo or c >= hi:
                    nxt.append((lo, hi))
                else:
                    if c > lo:
                        nxt.append((lo, c))
                    if d < hi:
                        nxt.append((d, hi))
            cur = nxt
        out += cur
    return sorted(out)


def halo_plan(bands, rank):
    """bands: per rank dict(out_rows=(..4), in_rows=(..4)).  -> (sends, recvs): lists of (peer, lo, hi)
    pixel ranges this rank must send to / receive from each peer, in a deterministic order."""
    own = [_ranges(b["out_rows"]) for b in bands]
    need = [_subtract(_ranges(b["in_rows"]), own[r]) for r, b in enumerate(bands)]
    sends, recvs = [], []
    for peer in range(len(bands)):
        if peer == rank:
            continue
        sends += [(peer, lo, hi) for lo, hi in _intersect(need[peer], own[rank])]
        recvs += [(peer, lo, hi) for lo, hi in _intersect(need[rank], own[peer])]
    return sends, recvs


def _global_rank(group, r):
    """Rank r of `group` as a global rank (P2POp / broadcast take global ranks)."""
    import torch.distributed as dist
    return r if group is None else dist.get_global_rank(group, r)


def exchange_halos(maps, bands, rank, group=None):
    """Fill the overlap rows of the full-size tensors `maps` (valid in this rank's out_rows) from their
    owners.  Point to point, ONE packed message per peer and direction (all ranges of all maps, in the order
    maps outer / halo_plan ranges inner, which both sides derive identically); bytes = the overlap only.
    `rank` and the band index are ranks within `group`.  Returns the number of elements received."""
    import torch
    import torch.distributed as dist
    sends, recvs = halo_plan(bands, rank)
    if not sends and not recvs:
        return 0
    ops, unpack = [], []
    for peer in sorted({p for p, _, _ in recvs}):
        rng = [(lo, hi) for p, lo, hi in recvs if p == peer]
        buf = torch.empty(sum(hi - lo for lo, hi in rng) * len(maps), dtype=maps[0].dtype, device=maps[0].device)
        unpack.append((buf, rng))
        ops.append(dist.P2POp(dist.irecv, buf, _global_rank(group, peer), group))
    keep = []
    for peer in sorted({p for p, _, _ in sends}):
        rng = [(lo, hi) for p, lo, hi in sends if p == peer]
        buf = torch.cat([m[lo:hi] for m in maps for lo, hi in rng])
        keep.append(buf)
        ops.append(dist.P2POp(dist.isend, buf, _global_rank(group, peer), group))
    for req in dist.batch_isend_irecv(ops):
        req.wait()
    for buf, rng in unpack:
        off = 0
        for m in maps:
            for lo, hi in rng:
                m[lo:hi] = buf[off:off + hi - lo]
                off += hi - lo
    return sum(hi - lo for _, lo, hi in recvs) * len(maps)


def gather_bands(maps, bands, group=None):
    """Make every rank's full-size tensors complete: each band's rows are broadcast by their owner."""
    import torch.distributed as dist
    for m in maps:
        for owner, b in enumerate(bands):
            for lo, hi in _ranges(b["out_rows"]):
                dist.broadcast(m[lo:hi], src=_global_rank(group, owner), group=group)


def convolve_banded(plan, maps_in, maps_out, group=None, gather=False):
    """Convolve maps sharded by latitude bands over the ranks of `group` with `plan` (a Plan built on
    every rank): halo exchange, then the rank's band through sc_convolve_band.  maps_in: full-size CUDA
    tensors valid in this rank's band rows; maps_out: full-size CUDA tensors, band rows written."""
    import torch.distributed as dist
    world, rank = dist.get_world_size(group), dist.get_rank(group)
    bands = [plan.band(world, r) for r in range(world)]
    exchange_halos(maps_in, bands, rank, group)
    plan.convolve_band(bands[rank]["ring_lo"], bands[rank]["ring_hi"], maps_in, maps_out)
    if gather:
        gather_bands(maps_out, bands, group)
    return bands[rank]
