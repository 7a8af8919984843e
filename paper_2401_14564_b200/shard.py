"""Multi-GPU plumbing: how the hot path shards across ranks.

The path partitions with NO exchange step: grid points are independent ("perfectly parallelizable"),
pixels are independent and ML-style batches are independent systems.  One process per
GPU; each rank runs whole systems of its own (weak scaling: rank r gets the config's generator with seed + r, or
its contiguous slice of the config-3 molecule batch).  The only communication is the timing protocol: a barrier
on both sides of the timed region and a MAX / SUM all-reduce of three scalars.  No data-path collective exists,
so none is invented.

Works with any torch.distributed backend ("nccl" on the GPU box, "gloo" in the CPU tests); holds none of the
method's arithmetic.
"""
from __future__ import annotations

import os
from typing import List, Sequence, Tuple


def env_rank_world() -> Tuple[int, int, int]:
    """(rank, world_size, local_rank) from the torchrun environment; (0, 1, 0) when launched plainly."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")),
            int(os.environ.get("LOCAL_RANK", "0")))


def rank_seed(base_seed: int, rank: int) -> int:
    """Weak scaling: rank r simulates an independent system drawn with seed base + 7919 r (7919 is prime and larger
    than any per-config molecule index, so rank streams never collide with config 3's seed + molecule index)."""
    return int(base_seed) + 7919 * int(rank)


def split_batch(n_items: int, rank: int, world: int) -> Tuple[int, int]:
    """Contiguous slice [lo, hi) of a batch of independent systems for this rank (sizes differ by at most one)."""
    if n_items < 0 or world < 1 or not (0 <= rank < world):
        raise ValueError("bad split arguments")
    q, r = divmod(n_items, world)
    lo = rank * q + min(rank, r)
    return lo, lo + q + (1 if rank < r else 0)


def slab_split(n_planes: int, rank: int, world: int, halo: int = 0) -> Tuple[int, int, int, int]:
    """Strong-scaling split of ONE grid / scan along an axis into `world` slabs: returns (lo, hi) owned planes and
    (lo_h, hi_h) including a halo clipped to [0, n_planes).  Used for the xy-tiling with halo of §8(e): the same
    tiling for the force-field grid and the scan means nothing ever crosses GPUs."""
    lo, hi = split_batch(n_planes, rank, world)
    return lo, hi, max(lo - halo, 0), min(hi + halo, n_planes)


def strong_slab(w, rank: int, world: int, halo: float = 4.0):
    """Strong scaling of ONE system (SURVEY 8(e); PAPER.md:266 "perfectly parallelizable", :280 pixels "virtually
    independent"): rank r gets scan rows [lo, hi) of w.scan and the rows of the force-field grid those pixels can
    reach: the tip's y range over the slab, widened by `halo` Å (the probe particle sits within |d0| + a deflection
    of well under an Å of the tip laterally) plus one cell for the interpolation.  The same tiling serves grid and
    scan, so nothing crosses GPUs.  Returns (workload of this rank, (lo, hi), (j_lo, j_hi) grid rows, inclusive).

    The grid rows are split only when grid axis 1 and the scan's dy both run along y, and the widened range lies inside
    the grid (a periodic axis would otherwise need wrapped rows: the sub-grid is a plain clamped grid); if not, the rank
    keeps the whole grid and only the scan is split.  Input bookkeeping only: no method arithmetic."""
    from dataclasses import replace

    import numpy as np
    s, g = w.scan, w.grid
    lo, hi = split_batch(s.npy, rank, world)
    sub_scan = replace(s, p0=np.asarray(s.p0, float) + lo * np.asarray(s.dy, float), npy=hi - lo)
    step = np.asarray(g.step, float)
    dy = np.asarray(s.dy, float)
    dxv = np.asarray(s.dx, float)
    ny = int(g.n[1])
    along_y = (step[1][0] == 0.0 and step[1][2] == 0.0 and step[0][1] == 0.0 and step[2][1] == 0.0 and dy[0] == 0.0 and
               dy[2] == 0.0 and dxv[1] == 0.0 and step[1][1] > 0.0 and hi > lo)
    j_lo, j_hi = 0, ny - 1
    if along_y:
        y0 = float(s.p0[1]) + float(w.tip.d0[1])
        ys = (y0 + lo * dy[1], y0 + (hi - 1) * dy[1])
        t_lo = (min(ys) - halo - float(g.origin[1])) / step[1][1]
        t_hi = (max(ys) + halo - float(g.origin[1])) / step[1][1]
        a, b = int(np.floor(t_lo)), int(np.ceil(t_hi)) + 1
        if g.periodic[1]:
            if a >= 0 and b <= ny - 1:
                j_lo, j_hi = a, b
        else:
            j_lo, j_hi = max(a, 0), min(b, ny - 1)
            if j_hi - j_lo < 1:
                j_lo, j_hi = 0, ny - 1
    sub_grid = g
    if (j_lo, j_hi) != (0, ny - 1):
        per = list(g.periodic)
        per[1] = 0
        sub_grid = replace(g, origin=np.asarray(g.origin, float) + j_lo * step[1], n=(int(g.n[0]), j_hi - j_lo + 1, int(g.n[2])),
                           periodic=tuple(per))
    return replace(w, grid=sub_grid, scan=sub_scan), (lo, hi), (j_lo, j_hi)


def aggregate(local_units: Sequence[float], local_seconds: float, dist=None) -> Tuple[List[float], float]:
    """Whole-job units (SUM over ranks) and the job's time (MAX over ranks).  `dist` = torch.distributed (already
    initialised) or None for a single process."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return [float(u) for u in local_units], float(local_seconds)
    import torch
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    u = torch.tensor([float(x) for x in local_units], dtype=torch.float64, device=dev)
    t = torch.tensor([float(local_seconds)], dtype=torch.float64, device=dev)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in u.cpu()], float(t.cpu()[0])


def barrier(dist=None) -> None:
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        dist.barrier()
