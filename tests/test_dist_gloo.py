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
