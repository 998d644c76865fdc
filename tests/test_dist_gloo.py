"""The N > 1 path on CPU: two gloo processes shard independent maps (no data-path collective), run
the per-rank convolution -- here the oracle stands in for the GPU kernels, which a CPU box cannot
run -- and combine outputs and timings exactly as bench.py --gpus N does."""
import os
import sys

import numpy as np
import pytest
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, n_maps, q):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    import oracle as O
    from paper_1409_4441_b200 import dist as D
    from workloads import gen
    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        nside, theta = 16, 13.6 * gen.DEG
        _, th = gen.table_nodes(theta, 257)
        T = np.exp(-0.5 * (th / (0.3 * theta)) ** 2)
        mine = D.map_shard(n_maps, rank, world)
        maps = [gen.noise_map(12 * nside * nside, 900 + i) for i in mine]
        out, cnt, _ = O.convolve(nside, T, theta, maps, nthreads=1) if maps else ([], np.zeros(1), None)
        pairs = int(cnt.astype(np.int64).sum()) * len(maps)
        ms, units = D.combine_timing([10.0 + rank, 3.0 - rank], pairs)
        allout = D.gather_outputs(list(out), n_maps)
        if rank == 0:
            q.put((ms, units, [np.asarray(o) for o in allout], int(cnt.astype(np.int64).sum())))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("n_maps", [3, 4])
def test_two_ranks_shard_independent_maps(n_maps):
    import oracle as O
    from paper_1409_4441_b200 import dist as D
    from workloads import gen
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + (os.getpid() + n_maps) % 2000
    procs = [ctx.Process(target=_worker, args=(r, world, port, n_maps, q)) for r in range(world)]
    for p in procs:
        p.start()
    ms, units, allout, pairs_per_map = q.get(timeout=180)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert ms == [11.0, 3.0]                                  # max over ranks, per entry
    assert units == pairs_per_map * n_maps                    # sum over ranks = whole job
    nside, theta = 16, 13.6 * gen.DEG
    _, th = gen.table_nodes(theta, 257)
    T = np.exp(-0.5 * (th / (0.3 * theta)) ** 2)
    maps = [gen.noise_map(12 * nside * nside, 900 + i) for i in range(n_maps)]
    ref, _, _ = O.convolve(nside, T, theta, maps, nthreads=1)
    assert len(allout) == n_maps
    for i in range(n_maps):
        np.testing.assert_array_equal(allout[i], ref[i])      # same code, same inputs: bit-identical


def test_map_shard_partitions():
    from paper_1409_4441_b200 import dist as D
    for n in range(0, 20):
        for world in (1, 2, 3, 8):
            parts = [D.map_shard(n, r, world) for r in range(world)]
            assert sorted(sum(parts, [])) == list(range(n))
            assert max(map(len, parts)) - min(map(len, parts)) <= 1
    with pytest.raises(ValueError):
        D.map_shard(3, 2, 2)
    assert D.rank_seeds([3, 4], 2) == [2003, 2004]
    ms, units = D.combine_timing([1.5], 7)                     # no process group: local values
    assert ms == [1.5] and units == 7.0


# ---------------------------------------------------------------------------------------------------
# latitude bands with halo exchange over two / three gloo ranks
# ---------------------------------------------------------------------------------------------------
def _cpu_bands(nside, theta, world):
    """Band layout like sc_band_partition's, from the oracle's ring table: equal ring counts, overlap =
    every ring whose colatitude is within theta (+ one ring) of the band."""
    import oracle as O
    t = O.ring_table(nside)
    start, npr, z = t["start"], t["npr"], t["z"]
    npix, N4 = 12 * nside * nside, 4 * nside
    row = lambda r: int(start[r - 1]) if r <= N4 - 1 else npix
    th = np.arccos(np.asarray(z, dtype=np.float64))
    bands = []
    for k in range(world):
        lo, hi = 1 + (2 * nside * k) // world, (2 * nside * (k + 1)) // world
        a = lo
        while a > 1 and th[lo - 1] - th[a - 2] <= theta:
            a -= 1
        a = max(1, a - 1)
        b = hi
        while b < N4 - 1 and th[b] - th[hi - 1] <= theta:
            b += 1
        b = min(N4 - 1, b + 1)
        o = (row(lo), row(hi + 1), row(2 * nside + 1) if hi >= 2 * nside else row(N4 - hi), row(N4 - lo + 1))
        i = [row(a), row(b + 1), row(N4 - b), row(N4 - a + 1)]
        if i[2] <= i[1]:
            i[1] = i[2] = i[3]
        bands.append(dict(ring_lo=lo, ring_hi=hi, out_rows=o, in_rows=tuple(i)))
    return bands


def _band_worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    import torch
    import torch.distributed as dist
    import oracle as O
    from paper_1409_4441_b200 import dist as D
    from workloads import gen
    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        nside, theta = 16, 9.0 * gen.DEG
        npix = 12 * nside * nside
        _, th = gen.table_nodes(theta, 129)
        T = np.exp(-0.5 * (th / (0.4 * theta)) ** 2)
        full = gen.noise_map(npix, 4242)
        bands = _cpu_bands(nside, theta, world)
        mine = bands[rank]
        # this rank starts with its own rows only; everything else is NaN until the halo exchange
        local = torch.full((npix,), float("nan"), dtype=torch.float32)
        for lo, hi in D._ranges(mine["out_rows"]):
            local[lo:hi] = torch.from_numpy(full[lo:hi])
        got = D.exchange_halos([local], bands, rank)
        sel = np.concatenate([np.arange(lo, hi) for lo, hi in D._ranges(mine["out_rows"])])
        out, _, _ = O.convolve(nside, T, theta, [local.numpy()], sel=sel, nthreads=1)   # the oracle stands in for the kernels
        res = torch.full((npix,), float("nan"), dtype=torch.float64)
        res[torch.from_numpy(sel)] = torch.from_numpy(np.asarray(out[0]))
        D.gather_bands([res], bands)
        needed = sum(hi - lo for lo, hi in D._subtract(D._ranges(mine["in_rows"]), D._ranges(mine["out_rows"])))
        q.put((rank, res.numpy(), int(got), int(needed)))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_latitude_bands_halo_exchange(world):
    import oracle as O
    from workloads import gen
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 31500 + (os.getpid() + world) % 2000
    procs = [ctx.Process(target=_band_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    results = [q.get(timeout=240) for _ in range(world)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    nside, theta = 16, 9.0 * gen.DEG
    _, th = gen.table_nodes(theta, 129)
    T = np.exp(-0.5 * (th / (0.4 * theta)) ** 2)
    ref, _, _ = O.convolve(nside, T, theta, [gen.noise_map(12 * nside * nside, 4242)], nthreads=1)
    for rank, res, got, needed in results:
        assert got == needed                       # exactly the overlap rows were received
        assert not np.isnan(res).any()             # a missing overlap row would have poisoned the band
        np.testing.assert_array_equal(res, ref[0])


def test_halo_plan_is_consistent():
    from paper_1409_4441_b200 import dist as D
    bands = _cpu_bands(32, 0.2, 5)
    covered = np.zeros(12 * 32 * 32, int)
    for b in bands:
        for lo, hi in D._ranges(b["out_rows"]):
            covered[lo:hi] += 1
    assert covered.min() == 1 and covered.max() == 1
    for r in range(5):
        sends, _ = D.halo_plan(bands, r)
        for peer, lo, hi in sends:                 # what r sends to peer is what peer expects from r
            assert (r, lo, hi) in D.halo_plan(bands, peer)[1]
    assert D._subtract([(0, 10)], [(2, 4), (6, 20)]) == [(0, 2), (4, 6)]
    assert D._intersect([(0, 10), (20, 30)], [(5, 25)]) == [(5, 10), (20, 25)]


def _subgroup_worker(rank, world, port, q):
    """Ranks 0 and 2 of a 3-rank job form a group and share TWO maps in two latitude bands: exercises the mapping of
    group ranks to global ranks in exchange_halos / gather_bands and the packed one-message-per-peer layout."""
    sys.path.insert(0, ROOT)
    import torch
    import torch.distributed as dist
    from paper_1409_4441_b200 import dist as D
    from workloads import gen
    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        grp = dist.new_group([0, 2])
        if rank in (0, 2):
            nside, theta = 8, 20.0 * gen.DEG
            npix = 12 * nside * nside
            grank = dist.get_rank(grp)
            bands = _cpu_bands(nside, theta, 2)
            full = [gen.noise_map(npix, 77), gen.noise_map(npix, 78)]
            local = []
            for f in full:
                t = torch.full((npix,), float("nan"), dtype=torch.float32)
                for lo, hi in D._ranges(bands[grank]["out_rows"]):
                    t[lo:hi] = torch.from_numpy(f[lo:hi])
                local.append(t)
            D.exchange_halos(local, bands, grank, grp)
            ok = True
            for t, f in zip(local, full):
                for lo, hi in D._ranges(bands[grank]["in_rows"]):
                    ok = ok and bool(np.array_equal(t[lo:hi].numpy(), f[lo:hi]))
            D.gather_bands(local, bands, grp)           # own rows are valid everywhere -> complete maps on both ranks
            ok = ok and all(np.array_equal(t.numpy(), f) for t, f in zip(local, full))
            q.put((rank, ok))
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_halo_exchange_in_a_subgroup_with_two_maps():
    world = 3
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 33500 + os.getpid() % 2000
    procs = [ctx.Process(target=_subgroup_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    results = [q.get(timeout=240) for _ in range(2)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert sorted(r for r, _ in results) == [0, 2] and all(ok for _, ok in results)
