"""N > 1 host logic on CPU: world_size-2 `gloo` processes run the sharding and the max-over-ranks / sum-over-ranks
aggregation bench.py uses (paper_2401_14564_b200/shard.py).  The data path has no collective (pixels, grid points and
batch systems are independent: PAPER.md:266, 280, 248), so this is all the multi-rank logic there is."""
import os
import socket
import sys

import numpy as np
import pytest
import torch.multiprocessing as mp

from paper_2401_14564_b200 import shard
from paper_2401_14564_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


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


def _strong_worker(rank, world, port, q):
    """Strong scaling (shard.strong_slab): every rank relaxes ITS rows on ITS rows of the grid with the FP64 oracle;
    rank 0 gathers the slabs (gloo all_gather) and returns them for comparison with the undivided scan."""
    import torch
    import torch.distributed as dist

    from oracle import oracle
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = _strong_case()
        ws, (lo, hi), (j_lo, j_hi) = shard.strong_slab(w, rank, world, halo=1.5)
        ff = oracle.forcefield(ws)                                    # this rank's rows of the grid only
        r = oracle.relax_scan(ff, ws.grid, ws.tip, ws.fire, ws.scan, traj=False)
        pos = torch.from_numpy(np.ascontiguousarray(r["pos_fz"].reshape(w.scan.nz, hi - lo, w.scan.npx, 4)))
        sizes = [shard.split_batch(w.scan.npy, k, world) for k in range(world)]
        bufs = [torch.empty((w.scan.nz, b - a, w.scan.npx, 4), dtype=torch.float64) for a, b in sizes]
        dist.all_gather(bufs, pos)
        units, t = shard.aggregate([ws.pixel_steps, ws.npoints], 0.5 * (rank + 1), dist)
        if rank == 0:
            q.put((torch.cat(bufs, dim=1).numpy(), units, t, (j_lo, j_hi)))
        else:
            q.put((None, units, t, (j_lo, j_hi)))
    finally:
        dist.destroy_process_group()


def _strong_case():
    w = W.shrink(W.get(0), scan_np=(12, 14), scan_nz=6)
    return w


def test_world2_gloo_strong_scaling_slabs_reproduce_the_undivided_scan():
    """SURVEY 8(e) strong scaling: two ranks, each with its scan rows and the grid rows under them + halo, no
    exchange.  The slabs partition the scan, each rank's grid is a strict subset, the halo covers the largest lateral
    deflection the oracle reports, and the gathered positions are those of the undivided scan."""
    from oracle import oracle
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_strong_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = [q.get(timeout=300) for _ in range(world)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    w = _strong_case()
    full = oracle.relax_scan(oracle.forcefield(w), w.grid, w.tip, w.fire, w.scan, traj=False)
    ref = full["pos_fz"].reshape(w.scan.nz, w.scan.npy, w.scan.npx, 4)
    got = next(r[0] for r in res if r[0] is not None)
    assert got.shape == ref.shape
    assert np.abs(got - ref).max() < 1e-9
    # pixel-steps add up to the scan; each rank sampled fewer grid points than the whole grid; time = MAX over ranks
    for _, units, t, rows in res:
        assert units[0] == w.pixel_steps and units[1] < 2 * w.npoints and t == pytest.approx(1.0)
        assert rows[1] - rows[0] + 1 < w.grid.n[1]
    # the halo (1.5 Å here) covers the largest lateral excursion of the probe particle from the tip
    tips = oracle.tip_positions(w.scan).reshape(w.scan.nz, w.scan.npy, w.scan.npx, 3)
    lateral = np.abs(ref[..., 1] - tips[..., 1]).max()
    h = w.grid.step[1][1]
    assert lateral + h < 1.5, lateral
    # slabs partition the rows for any world size; on config 4 the halo keeps every slab inside the periodic cell
    w4 = W.get(4)
    for world4 in (2, 3, 8):
        rows = [shard.strong_slab(w4, r, world4) for r in range(world4)]
        assert rows[0][1][0] == 0 and rows[-1][1][1] == w4.scan.npy
        assert all(a[1][1] == b[1][0] for a, b in zip(rows[:-1], rows[1:]))
        for ws, (lo, hi), (j_lo, j_hi) in rows:
            assert ws.grid.periodic[1] == 0 and 0 <= j_lo < j_hi <= w4.grid.n[1] - 1
            y_pix = (ws.scan.p0[1], ws.scan.p0[1] + (ws.scan.npy - 1) * ws.scan.dy[1])
            assert ws.grid.origin[1] <= y_pix[0] - 4.0 and ws.grid.origin[1] + (ws.grid.n[1] - 1) * 0.05 >= y_pix[1] + 4.0
    # a slab that would cross the periodic boundary keeps the whole grid
    wp = W.shrink(W.get(2), scan_np=(8, 8), scan_nz=3)
    from dataclasses import replace
    wp = replace(wp, scan=replace(wp.scan, p0=np.array([5.0, 0.5, 9.0])))
    ws, _, rows = shard.strong_slab(wp, 0, 2)
    assert rows == (0, wp.grid.n[1] - 1) and ws.grid.periodic == wp.grid.periodic


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


def test_bench_gpus_n_starts_n_ranks():
    """`python bench.py --gpus 2` launched plainly must start two ranks itself (one process per GPU through
    torch.distributed.run on 127.0.0.1) and report the REAL world size.  Driven here through the host-only oracle arm
    (`--impl reference`: rank 0 works, rank 1 exits 0), which needs no GPU; the GPU arm of the same launcher refuses
    to start when the node has fewer devices than ranks instead of stacking ranks on one GPU; and a --gpus value that
    disagrees with the launcher's WORLD_SIZE is an error, not a silently wrong n_gpus."""
    import json
    import subprocess
    bench = os.path.join(ROOT, "bench.py")
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, bench, "--gpus", "2", "--impl", "reference", "--steps", "1", "--warmup", "0",
                        "--config", "0"], env=env, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [json.loads(l) for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, r.stdout                       # rank 0 alone prints
    assert lines[0]["impl"] == "reference" and lines[0]["n_gpus"] == 2 and lines[0]["gpu_launches"] == 0
    import torch
    if not torch.cuda.is_available():
        r = subprocess.run([sys.executable, bench, "--gpus", "2", "--steps", "1"], env=env, capture_output=True, text=True,
                           timeout=300, cwd=ROOT)
        assert r.returncode != 0 and "needs 2 CUDA devices" in r.stderr
    r = subprocess.run([sys.executable, bench, "--gpus", "2", "--impl", "reference"], env=dict(env, WORLD_SIZE="3", RANK="0"),
                       capture_output=True, text=True, timeout=300, cwd=ROOT)
    assert r.returncode != 0 and "WORLD_SIZE=3" in r.stderr
