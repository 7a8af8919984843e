"""N > 1 host logic on CPU: world_size-2 `gloo` processes run the sharding and the max-over-ranks / sum-over-ranks
aggregation bench.py uses (paper_2401_14564_b200/shard.py).  The data path has no collective (pixels, grid points and
batch systems are independent: PAPER.md:266, 280, 248), so this is all the multi-rank logic there is."""
import os
import socket

import numpy as np
import pytest
import torch.multiprocessing as mp

from paper_2401_14564_b200 import shard
from paper_2401_14564_b200 import workloads as W


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        assert shard.env_rank_world() == (rank, world, rank)
        # weak scaling: every rank draws its own system of the same config
        w = W.get(0, seed=shard.rank_seed(1000, rank))
        lo, hi = shard.split_batch(64, rank, world)
        shard.barrier(dist)
        units, t = shard.aggregate([w.pixel_steps, w.pairs, hi - lo], 0.010 * (rank + 1), dist)
        shard.barrier(dist)
        q.put((rank, units, t, float(w.xyzq.sum()), (lo, hi)))
    finally:
        dist.destroy_process_group()


def test_world2_gloo_aggregation_and_independent_shards():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    w = W.get(0)
    for rank, units, t, chk, sl in res:
        assert units == [2.0 * w.pixel_steps, 2.0 * w.pairs, 64.0]      # SUM over ranks, batch fully covered
        assert t == pytest.approx(0.020)                                 # MAX over ranks
    assert res[0][3] != res[1][3]                                        # different seeds -> different systems
    assert res[0][4] == (0, 32) and res[1][4] == (32, 64)


def test_split_batch_covers_everything_once():
    for n in (0, 1, 7, 64, 65):
        for world in (1, 2, 3, 8):
            parts = [shard.split_batch(n, r, world) for r in range(world)]
            assert parts[0][0] == 0 and parts[-1][1] == n
            assert all(a[1] == b[0] for a, b in zip(parts[:-1], parts[1:]))
            sizes = [hi - lo for lo, hi in parts]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard.split_batch(4, 2, 2)


def test_slab_split_halo_is_clipped():
    assert shard.slab_split(100, 0, 4, halo=8) == (0, 25, 0, 33)
    assert shard.slab_split(100, 3, 4, halo=8) == (75, 100, 67, 100)
    assert shard.slab_split(100, 1, 4, halo=8) == (25, 50, 17, 58)


def test_single_process_aggregate_is_identity():
    assert shard.aggregate([3, 4.5], 0.25, None) == ([3.0, 4.5], 0.25)
    assert shard.rank_seed(4000, 0) == 4000 and shard.rank_seed(4000, 3) - 4000 > 64


def test_rank_workloads_are_valid_and_same_shape():
    a, b = W.get(1, seed=shard.rank_seed(2000, 0)), W.get(1, seed=shard.rank_seed(2000, 1))
    assert a.pairs == b.pairs and a.pixel_steps == b.pixel_steps
    assert not np.array_equal(a.xyzq, b.xyzq)
    assert abs(float(b.xyzq[:, 3].sum())) < 1e-5
