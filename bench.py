#!/usr/bin/env python
"""bench.py — one "step" = one pass of the whole hot path (force-field grid -> FIRE relaxation scan -> df) over one
seeded synthetic workload of BASELINE.json.  Prints ONE JSON line (rank 0).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference]
                  [--no-cpu-baseline] [--no-per-config]

Default workload: configs[4], the largest single-GPU configuration.  The other four configs are measured in the
same process (3 warm-up + 3 timed steps each) and reported as compact numeric records under `roofline.per_config`
(full records under `parts.per_config`), so that one driver run carries the force-field and relaxation fractions of
all five configs.  `--gpus N > 1` launched plainly starts N ranks itself (torch.distributed.run, one process per GPU);
under torchrun it reads the rank environment.  `roofline.traffic` is a STORED ncu measurement (`traffic_source` names
the capture and the commit), not something the run measures.

* `value` (device-resident inputs): relaxed pixel-steps per second over the full scan; CUDA events per step on the
  launching stream, L2 flushed between steps, max over ranks.
* `e2e`: the same scan through the one-call host API ppfm_scan_host[_batch|_sweep] with pinned HOST buffers.
* `roofline`: the step's dominant kernel with the bound that binds it; `roofline_kernels`: ff, relax, df of the
  headline config.  What the fields mean, the algorithmic counts and the peaks are stated in DESIGN.md §6.
* `cpu_baseline`: the FP64 oracle, as it stands, timed on this box's host cores on a bounded sample.
* `--impl reference`: the oracle arm (this tier has no reference implementation to install).
The oracle is imported ONLY by the cpu_baseline leg and the reference arm.
"""
from __future__ import annotations

import argparse
import hashlib
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2401_14564_b200 import shard  # noqa: E402
from paper_2401_14564_b200 import workloads as W  # noqa: E402

METRIC = "relaxed pixel-steps/s over the full scan (FF grid + FIRE relaxation + df)"
UNIT = "pixel-steps/s"
BASE_SEED = {0: 1000, 1: 2000, 2: 3000, 3: 4000, 4: 5000}
WORKLOAD_NAME = {0: "configs[0] tiny 10 atoms, 60x60x40 grid, 30x30x40 scan",
                 1: "configs[1] planar 60-atom molecule, 200x200x100 grid, 150x150x40 scan",
                 2: "configs[2] molecule on 500-atom periodic slab (9 images), 250x250x120 grid, 200x200x40 scan x 3 Q",
                 3: "configs[3] ML batch of 64 molecules (20-50 atoms), 128x128x64 grids, 128x128x20 scans",
                 4: "configs[4] 5000 atoms x 9 images, 800x800x200 grid, 400x400x80 scan"}
# ---- algorithmic counts ------------------------------------------------------------------------------
PAIR_INSTR, PAIR_FLOPS = 19, 28        # canonical per pair interaction: FP32-pipe instructions, flops
# what ff_kernel executes per pair (ff.cu, FP32x2-packed): lane-instructions for an atom with / without a Coulomb factor
PAIR_EXEC = {"charged": 15, "neutral": 13, "charged_split": 20, "neutral_split": 14}
# ffe_kernel (energy-only pass): 8 packed lane-instructions + 1 MUFU per pair; flops: dz add, r2 fma, ir2, 2 x ir6,
# t fma, 2 energy fmas = 1 + 2 + 1 + 2 + 2 + 4 = 12 (+ the rsqrt)
ENERGY_PAIR_INSTR, ENERGY_PAIR_FLOPS = 8, 13
ITER_INSTR, ITER_FLOPS = 70, 114       # relax_kernel per FIRE iteration (cached cell, symmetric tip); + 4 MUFU
TRI_INSTR, TRI_FLOPS = 270, 514        # the tri-cubic instance
SMS, LANES = 148, 128
# relax_kernel time (ms) of the committed kernels on a B200 at 1965 MHz; the run reports relax ms against 1.1 x these
# so that a slower instruction schedule of the same source (DESIGN.md §7 "schedule sensitivity") shows up
PERF_GUARD_RELAX_MS = {0: 0.475, 1: 0.76, 2: 2.3, 3: 7.95, 4: 4.65}


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return {"hbm_gbs": float(d["hbm_gbs"]), "sm_max_mhz": float(d.get("sm_max_mhz", 1965.0)), "source": "measured"}
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "source": "fallback"}


TRAFFIC_CSV = "profiles/r02_traffic.csv"
# the commit whose kernels the captures in TRAFFIC_CSV ran (round 2's final kernels; `git log -- profiles/r02_traffic.csv`).
# ff.cu's kernels have not changed since; the number is a stored ncu measurement, NOT something this run measured.
TRAFFIC_COMMIT = "1427f50"


def ncu_traffic(cfg: int, kernel: str, with_source: bool = False):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed `ncu --set full` captures
    (profiles/r02_traffic.csv: cfg,kernel,dram_read_bytes,dram_write_bytes,capture); None where no capture exists.
    with_source: (bytes, "ncu capture profiles/<file>, commit <sha>")."""
    p = os.path.join(ROOT, TRAFFIC_CSV)
    found, src = None, None
    if os.path.exists(p):
        with open(p) as f:
            for line in f:
                c = line.strip().split(",")
                if len(c) >= 4 and c[0] == str(cfg) and c[1] == kernel:
                    found = float(c[2]) + float(c[3])
                    src = (f"stored ncu --set full capture profiles/{c[4].split(' ')[0] if len(c) > 4 else '?'} via "
                           f"{TRAFFIC_CSV}, kernels of commit {TRAFFIC_COMMIT}; not measured in this run")
    return (found, src) if with_source else found


def inputs_sha256(ws) -> str:
    """SHA-256 over the generated inputs of a workload list (atoms, types, and every scalar of grid / scan / tip)."""
    h = hashlib.sha256()
    for w in ws:
        h.update(np.ascontiguousarray(w.xyzq, dtype=np.float32).tobytes())
        h.update(np.ascontiguousarray(w.types, dtype=np.int32).tobytes())
        for arr in (w.elem_R, w.elem_e, w.lattice.a, w.lattice.b, w.lattice.c, w.lattice.nimg, w.grid.origin,
                    w.grid.step, w.grid.n, w.grid.periodic, [w.probe.R, w.probe.e, w.probe.Q], w.tip.k_lat,
                    [w.tip.k_rad], w.tip.d0, w.scan.p0, w.scan.dx, w.scan.dy,
                    [w.scan.npx, w.scan.npy, w.scan.nz, w.scan.dz], [w.df.A, w.df.k0, w.df.f0, w.r_min],
                    w.Q_sweep or []):
            h.update(np.ascontiguousarray(arr, dtype=np.float64).tobytes())
    return h.hexdigest()


# ------------------------------------------------------------------------------------------------- clock sampling
class ClockSampler:
    """Samples SM clock and throttle reasons with NVML while the timed region runs."""

    def __init__(self, index: int):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml as nv
            nv.nvmlInit()
            self.nv = nv
            self.h = nv.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(nv.nvmlDeviceGetMaxClockInfo(self.h, nv.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def _loop(self):
        nv = self.nv
        names = {nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
                 nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap"}
        while not self._stop.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                r = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            self._stop.wait(0.002)

    def start(self):
        if self.nv is not None:
            self._thr = threading.Thread(target=self._loop, daemon=True)
            self._thr.start()

    def stop(self):
        if self._thr is not None:
            self._stop.set()
            self._thr.join()
        return {"sm_mhz": float(np.median(self.samples)) if self.samples else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ------------------------------------------------------------------------------------------------- workloads
def build_workloads(cfg: int, rank: int, world: int, strong: bool = False):
    """This rank's systems.  Weak scaling (default): an independent seeded draw of the same config per rank.  Strong
    scaling (--strong): ONE system; rank r takes its rows of the scan and the grid rows under them + 4 Å halo
    (shard.strong_slab; config 3 splits its 64 molecules instead), no exchange between ranks."""
    if strong:
        if cfg == 3:
            lo, hi = shard.split_batch(64, rank, world)
            return W.config3(64, seed=BASE_SEED[3])[lo:hi]
        return [shard.strong_slab(W.get(cfg, seed=BASE_SEED[cfg]), rank, world)[0]]
    seed = shard.rank_seed(BASE_SEED[cfg], rank)
    if cfg == 3:
        return W.config3(64, seed=seed)
    return [W.get(cfg, seed=seed)]


class DeviceJob:
    """Device-resident buffers of one rank's systems and the step that runs the three entry points on them."""

    def __init__(self, P, torch, cfg, ws):
        import ctypes
        self.P, self.torch, self.cfg, self.ws = P, torch, cfg, ws
        self.batch = len(ws) > 1
        w0 = ws[0]
        self.sweep = w0.Q_sweep if w0.Q_sweep else None
        self.xyzq = torch.from_numpy(np.concatenate([w.xyzq for w in ws]).astype(np.float32)).cuda()
        self.types = torch.from_numpy(np.concatenate([w.types for w in ws]).astype(np.int32)).cuda()
        self.off = np.concatenate([[0], np.cumsum([w.natoms for w in ws])])
        npts = sum(w.npoints for w in ws)
        nps = sum(w.pixel_steps for w in ws)
        s = w0.scan
        nq = len(self.sweep) if self.sweep else 1      # Q sweep: the nq combined grids side by side, the nq scans one batch
        self.npts, self.nps_one = npts, nps
        self.ff = torch.empty((nq * npts, 4), dtype=torch.float32, device="cuda")
        if self.sweep:
            self.ff_lj = torch.empty((npts, 4), dtype=torch.float32, device="cuda")
            self.ff_el = torch.empty_like(self.ff_lj)
        self.pos = torch.empty((nq * nps, 4), dtype=torch.float32, device="cuda")
        self.iters = torch.empty((nq * nps,), dtype=torch.int16, device="cuda")
        self.df = torch.empty((nq * len(ws) * (s.nz - w0.n_df) * s.npy * s.npx,), dtype=torch.float32, device="cuda")
        self.stats = P.new_stats()
        # argument marshalling done once: ready ctypes structs pass straight through the binding
        self.c_lat = P.c_array([w.lattice for w in ws], P.c_lattice)
        self.c_probe = P.c_array([w.probe for w in ws], P.c_probe)
        self.c_grid = P.c_array([w.grid for w in ws], P.c_grid)
        self.c_tip = P.c_array([w.tip for w in ws], P.c_tip)
        self.c_scan = P.c_array([w.scan for w in ws], P.c_scan)
        self.c_fire = P.c_fire(w0.fire)
        if self.sweep:
            self.c_grid_q = P.c_array([w0.grid] * nq, P.c_grid)
            self.c_tip_q = P.c_array([w0.tip] * nq, P.c_tip)
            self.c_scan_q = P.c_array([w0.scan] * nq, P.c_scan)
        self.c_off = (ctypes.c_int32 * (len(ws) + 1))(*[int(v) for v in self.off])
        self.pairs = float(sum(w.pairs for w in ws))
        self.n_runs = len(self.sweep) if self.sweep else 1
        self.pixel_steps = float(nps * self.n_runs)
        self.points = float(npts)
        self.marks = []

    def pair_exec_instr(self):
        """FP32-pipe lane-instructions ff_kernel executes per launch (PAIR_EXEC per pair, by kind of atom record)."""
        tot = 0.0
        for w in self.ws:
            kq_zero = (w.xyzq[:, 3] == 0.0) | (not self.sweep and w.probe.Q == 0.0)
            n_neutral = int(np.count_nonzero(kq_zero))
            n_charged = w.natoms - n_neutral
            per_point = (n_charged * PAIR_EXEC["charged_split" if self.sweep else "charged"] +
                         n_neutral * PAIR_EXEC["neutral_split" if self.sweep else "neutral"])
            tot += float(per_point) * w.nimages * w.npoints
        return tot

    def relax_tricubic(self, E, stats):
        P = self.P
        if self.batch:
            P.relax_scan_tricubic_batch(E, self.c_grid, self.c_tip, self.c_fire, self.c_scan, pos_fz=self.pos,
                                        iters=self.iters, stats=stats)
        else:
            P.relax_scan_tricubic(E, self.c_grid[0], self.c_tip[0], self.c_fire, self.c_scan[0], pos_fz=self.pos,
                                  iters=self.iters, stats=stats)

    def stiffness(self, out):
        P = self.P
        if self.batch:
            P.stiffness_batch(self.ff, self.c_grid, self.c_tip, self.c_scan, self.pos, out=out)
        else:
            P.stiffness(self.ff, self.c_grid[0], self.c_tip[0], self.c_scan[0], self.pos, out=out)

    def relax_stiffness(self, eig, stats):
        """The relaxation scan of step() with the stiffness map folded in (ppfm_relax_scan_stiffness[_batch])."""
        P = self.P
        if self.batch:
            P.relax_scan_stiffness_batch(self.ff, self.c_grid, self.c_tip, self.c_fire, self.c_scan, pos_fz=self.pos,
                                         iters=self.iters, eig=eig, stats=stats)
        else:
            P.relax_scan_stiffness(self.ff, self.c_grid[0], self.c_tip[0], self.c_fire, self.c_scan[0], pos_fz=self.pos,
                                   iters=self.iters, eig=eig, stats=stats)

    def relax_plain(self, stats):
        P = self.P
        if self.batch:
            P.relax_scan_batch(self.ff, self.c_grid, self.c_tip, self.c_fire, self.c_scan, pos_fz=self.pos,
                               iters=self.iters, stats=stats)
        else:
            P.relax_scan(self.ff, self.c_grid[0], self.c_tip[0], self.c_fire, self.c_scan[0], pos_fz=self.pos,
                         iters=self.iters, stats=stats)

    def _mark(self, name):
        ev = self.torch.cuda.Event(enable_timing=True)
        ev.record()
        self.marks.append((name, ev))

    def step(self):
        """Enqueue one full scan (all on torch's current stream); event marks bracket the whole step."""
        P, ws, w0 = self.P, self.ws, self.ws[0]
        s = w0.scan
        self.marks = []
        self._mark("start")
        if self.batch:
            P.forcefield_batch(self.c_off, self.xyzq, self.types, w0.elem_R, w0.elem_e, self.c_lat, self.c_probe,
                               self.c_grid, w0.r_min, out=self.ff)
            P.relax_scan_batch(self.ff, self.c_grid, self.c_tip, self.c_fire, self.c_scan,
                               pos_fz=self.pos, iters=self.iters, stats=self.stats)
            P.df(self.pos, s.npx, s.npy, s.nz, s.dz, w0.df.A, w0.df.k0, w0.df.f0, out=self.df, nsys=len(ws))
        elif self.sweep:
            P.forcefield_split(self.xyzq, self.types, w0.elem_R, w0.elem_e, self.c_lat[0], self.c_probe[0],
                               self.c_grid[0], w0.r_min, out_lj=self.ff_lj, out_el=self.ff_el)
            for i, Q in enumerate(self.sweep):
                P.combine(self.ff_lj, self.ff_el, Q, out=self.ff[i * self.npts:(i + 1) * self.npts])
            # the len(sweep) scans as ONE batch launch: a single 200 x 200 scan cannot fill the GPU, three at once can
            P.relax_scan_batch(self.ff, self.c_grid_q, self.c_tip_q, self.c_fire, self.c_scan_q, pos_fz=self.pos,
                               iters=self.iters, stats=self.stats)
            P.df(self.pos, s.npx, s.npy, s.nz, s.dz, w0.df.A, w0.df.k0, w0.df.f0, out=self.df, nsys=len(self.sweep))
        else:
            P.forcefield(self.xyzq, self.types, w0.elem_R, w0.elem_e, self.c_lat[0], self.c_probe[0], self.c_grid[0],
                         w0.r_min, out=self.ff)
            P.relax_scan(self.ff, self.c_grid[0], self.c_tip[0], self.c_fire, self.c_scan[0], pos_fz=self.pos,
                         iters=self.iters, stats=self.stats)
            P.df(self.pos, s.npx, s.npy, s.nz, s.dz, w0.df.A, w0.df.k0, w0.df.f0, out=self.df)
        self._mark("end")

    def step_ms(self):
        return self.marks[0][1].elapsed_time(self.marks[-1][1])


class HostJob:
    """The same scan through ppfm_scan_host: pinned host buffers in and out, copies inside the timed region."""

    def __init__(self, P, torch, ws):
        from dataclasses import replace as _replace
        ws = [_replace(w, lattice=P.c_lattice(w.lattice), grid=P.c_grid(w.grid), tip=P.c_tip(w.tip),
                       fire=P.c_fire(w.fire), scan=P.c_scan(w.scan)) for w in ws]
        self.P, self.ws = P, ws
        self.bufs = []
        self.h2d = self.d2h = 0
        for w in ws:
            s = w.scan
            hx = torch.from_numpy(w.xyzq.astype(np.float32)).pin_memory()
            ht = torch.from_numpy(w.types.astype(np.int32)).pin_memory()
            nq = len(w.Q_sweep) if w.Q_sweep else 1
            hp = torch.empty((nq, s.nz, s.npy, s.npx, 4), dtype=torch.float32).pin_memory()
            hi = torch.empty((nq, s.nz, s.npy, s.npx), dtype=torch.int16).pin_memory()
            hd = torch.empty((nq, s.nz - w.n_df, s.npy, s.npx), dtype=torch.float32).pin_memory()
            self.bufs.append((hx, ht, hp, hi, hd))
            self.h2d += hx.numel() * 4 + ht.numel() * 4
            self.d2h += hp.numel() * 4 + hi.numel() * 2 + hd.numel() * 4 + 56
        if len(ws) > 1:      # batch: one concatenated set of pinned buffers, one ppfm_scan_host_batch call per step
            hx = torch.cat([b[0] for b in self.bufs]).pin_memory()
            ht = torch.cat([b[1] for b in self.bufs]).pin_memory()
            hp = torch.empty((sum(b[2].numel() // 4 for b in self.bufs), 4), dtype=torch.float32).pin_memory()
            hi = torch.empty((sum(b[3].numel() for b in self.bufs),), dtype=torch.int16).pin_memory()
            hd = torch.empty((sum(b[4].numel() for b in self.bufs),), dtype=torch.float32).pin_memory()
            self.cat = (hx, ht, hp, hi, hd)
            self.bufs = []

    def step(self):
        if len(self.ws) > 1:
            hx, ht, hp, hi, hd = self.cat
            self.P.scan_host_batch(self.ws, hx, ht, hp, hi, hd)
            return
        for w, (hx, ht, hp, hi, hd) in zip(self.ws, self.bufs):
            if w.Q_sweep:
                self.P.scan_host_sweep(w, w.Q_sweep, hx, ht, hp, hi, hd)
            else:
                self.P.scan_host(w, hx, ht, hp, hi, hd)


# ------------------------------------------------------------------------------------------------- oracle legs
def oracle_sample_run(w, n_points: int, n_pixels: int, seed: int = 7):
    """Time the oracle, as it stands, on a bounded sample of workload `w`: `n_points` seeded grid points of the force
    field, then the relaxation scan + df of the central `n_pixels` pixels on the oracle's OWN FP64 force field:
    * where the sub-grid those pixels can reach (lateral margin 4 Å) costs <= 3e9 pair evaluations it is built first
      (not timed) and the scan runs on it;
    * otherwise (configs 2 and 4) the scan evaluates its grid nodes from the atoms on demand (oracle.relax_scan_atoms) and the
      node evaluations (counted) are taken out of the relaxation time at the pair rate measured in the first leg.
    Nothing here comes from the CUDA path.  Returns timings and the rate extrapolated to the full workload."""
    from dataclasses import replace

    from oracle import oracle
    t0 = time.perf_counter()
    idx = W.sample_indices(w.npoints, n_points, seed)
    oracle.forcefield(w, idx=idx)
    t_ff = time.perf_counter() - t0
    ff_pairs = float(len(idx)) * w.natoms * w.nimages
    ff_rate = ff_pairs / t_ff
    s, g = w.scan, w.grid
    side = max(1, int(round(np.sqrt(n_pixels))))
    side_x, side_y = min(side, s.npx), min(side, s.npy)
    ix0, iy0 = (s.npx - side_x) // 2, (s.npy - side_y) // 2
    sub_scan = replace(s, p0=s.p0 + ix0 * s.dx + iy0 * s.dy, npx=side_x, npy=side_y)
    h = np.array([g.step[0][0], g.step[1][1]])
    lo = np.array([sub_scan.p0[0], sub_scan.p0[1]]) - 4.0
    hi = lo + 8.0 + np.array([side_x * s.dx[0], side_y * s.dy[1]])
    i_lo = np.maximum(np.floor((lo - g.origin[:2]) / h).astype(int), 0)
    i_hi = np.minimum(np.ceil((hi - g.origin[:2]) / h).astype(int), np.array(g.n[:2]) - 1)
    sub_n = (int(i_hi[0] - i_lo[0] + 1), int(i_hi[1] - i_lo[1] + 1), g.n[2])
    sub_cost = float(sub_n[0]) * sub_n[1] * sub_n[2] * w.natoms * w.nimages
    if sub_cost <= 3e9:
        grid_kind = f"oracle FP64 sub-grid {list(sub_n)} (built first, not timed)"
        sub_grid = replace(g, origin=g.origin + np.array([i_lo[0] * h[0], i_lo[1] * h[1], 0.0]), n=sub_n,
                           periodic=(0, 0, 0))
        t1 = time.perf_counter()
        ff_sub = oracle.forcefield(replace(w, grid=sub_grid))
        t_grid = time.perf_counter() - t1
        t2 = time.perf_counter()
        r = oracle.relax_scan(ff_sub, sub_grid, w.tip, w.fire, sub_scan, traj=False)
        t_relax = time.perf_counter() - t2
        t_wall = t_relax
    else:
        grid_kind = "oracle FP64 grid nodes evaluated from the atoms on demand (their cost taken out at the oracle's pair rate)"
        t2 = time.perf_counter()
        r = oracle.relax_scan_atoms(w, scan=sub_scan, traj=False)
        t_all = time.perf_counter() - t2
        t_grid = float(r["nodes"].sum()) * w.natoms * w.nimages / ff_rate
        t_relax = max(t_all - t_grid, 0.05 * t_all)
        t_wall = t_all
    t3 = time.perf_counter()
    oracle.df(r["pos_fz"][..., 3], s.dz, w.df.A, w.df.k0, w.df.f0)
    t_df = time.perf_counter() - t3
    nq = len(w.Q_sweep) if w.Q_sweep else 1
    pix_n = side_x * side_y
    relax_rate = pix_n * s.nz / (t_relax + t_df)
    full_s = w.pairs / ff_rate + nq * w.pixel_steps / relax_rate
    return {"t_ff": t_ff, "t_grid": t_grid, "t_relax": t_relax, "t_df": t_df, "ff_pairs_per_s": ff_rate,
            "relax_pixel_steps_per_s": relax_rate, "relax_wall_pixel_steps_per_s": pix_n * s.nz / (t_wall + t_df),
            "s_per_full_scan_extrapolated": full_s,
            "value": nq * w.pixel_steps / full_s, "sample_points": int(len(idx)), "sample_pixels": int(pix_n),
            "grid_kind": grid_kind, "iters_per_pixel_step": float(np.abs(r["iters"]).mean()),
            "cores": oracle.num_threads()}


def sample_sizes(w, target_s: float):
    """Sample sizes for about `target_s` seconds of oracle work, from a quick calibration run."""
    cal = oracle_sample_run(w, 2000, 16)
    n_points = int(min(w.npoints, max(2000, 0.35 * target_s * cal["ff_pairs_per_s"] / (w.natoms * w.nimages))))
    n_pixels = int(min(w.scan.npx * w.scan.npy, max(16, 0.45 * target_s * cal["relax_wall_pixel_steps_per_s"] / w.scan.nz)))
    return n_points, n_pixels


def cpu_baseline(w, target_s: float = 15.0):
    n_points, n_pixels = sample_sizes(w, target_s)
    r = oracle_sample_run(w, n_points, n_pixels)
    return {"value": r["value"], "unit": UNIT, "cores": r["cores"], "kind": "oracle",
            "sample": (f"unoptimised FP64 oracle (gcc -O2, OpenMP), the checker as it stands: force field at "
                       f"{r['sample_points']} seeded grid points ({r['t_ff']:.1f} s); relaxation + df of the central "
                       f"{r['sample_pixels']} pixels x all z-steps on {r['grid_kind']} "
                       f"({r['t_relax'] + r['t_df']:.1f} s); value extrapolated to the full workload"),
            "ff_pairs_per_s": r["ff_pairs_per_s"], "relax_pixel_steps_per_s": r["relax_pixel_steps_per_s"],
            "s_per_full_scan_extrapolated": r["s_per_full_scan_extrapolated"],
            "iters_per_pixel_step": r["iters_per_pixel_step"]}


def run_reference(args):
    """The oracle arm: K timed steps, each a bounded sample of the same workload, on the host cores."""
    rank, world, _ = shard.env_rank_world()
    if rank != 0:
        return
    ws = build_workloads(args.config, 0, 1)
    w = ws[0]
    per_step = max(1.0, min(6.0, 150.0 / max(1, args.steps + args.warmup)))
    n_points, n_pixels = sample_sizes(w, per_step)
    for _ in range(args.warmup):
        oracle_sample_run(w, n_points, n_pixels)
    t0 = time.perf_counter()
    runs = [oracle_sample_run(w, n_points, n_pixels) for _ in range(args.steps)]
    wall = time.perf_counter() - t0
    value = float(np.mean([r["value"] for r in runs]))
    r = runs[-1]
    sample = (f"each step: unoptimised FP64 oracle force field at {r['sample_points']} seeded grid points + relaxation/df "
              f"of the central {r['sample_pixels']} pixels on {r['grid_kind']}; value extrapolated to the full workload")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * wall / max(1, args.steps),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD_NAME[args.config], "seed": BASE_SEED[args.config]},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": r["cores"], "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------- our arm
def measure_config(P, B, torch, cfg, ws, steps, warmup, e2e_steps, flush, env, dist=None, sample_clocks=False):
    """Run `warmup` + `steps` device-resident steps and `e2e_steps` host-API steps of one config; return the numbers."""
    peaks, alu_peak = env["peaks"], env["alu_peak"]
    job = DeviceJob(P, torch, cfg, ws)
    for _ in range(warmup):
        flush.zero_()
        job.stats.zero_()
        job.step()
    torch.cuda.synchronize()
    shard.barrier(dist)
    sampler = ClockSampler(torch.cuda.current_device()) if sample_clocks else None
    if sampler:
        sampler.start()
    n0 = B.launch_count()
    B.timing_enable(True)          # per-kernel CUDA events recorded inside the library, directly around each launch
    tot_ms, iters_total = 0.0, 0
    t_wall0 = time.perf_counter()
    for _ in range(steps):
        flush.zero_()
        job.stats.zero_()
        job.step()
        torch.cuda.synchronize()
        tot_ms += job.step_ms()
        iters_total += P.read_stats(job.stats)["total_iters"]
    torch.cuda.synchronize()
    shard.barrier(dist)
    wall_s = time.perf_counter() - t_wall0
    launches = B.launch_count() - n0
    clocks = sampler.stop() if sampler else None
    kern = B.timing_read()
    B.timing_enable(False)
    K = max(1, steps)
    stats = P.read_stats(job.stats)
    ms = {k: v[0] / K for k, v in kern.items()}
    n_launch = {k: v[1] / K for k, v in kern.items()}
    t_local = tot_ms / K * 1e-3

    # ---- end-to-end arm (host buffers through ppfm_scan_host)
    host = HostJob(P, torch, ws)
    host.step()
    torch.cuda.synchronize()
    shard.barrier(dist)
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        host.step()
    torch.cuda.synchronize()
    e2e_local = (time.perf_counter() - t0) / max(1, e2e_steps)
    shard.barrier(dist)
    h2d, d2h = host.h2d, host.d2h
    del host

    (units_ps, units_pairs), t_step = shard.aggregate([job.pixel_steps, job.pairs], t_local, dist)
    (e2e_units,), e2e_t = shard.aggregate([job.pixel_steps], e2e_local, dist)
    world = env["world"]
    ff_s, relax_s, df_s = ms["ff"] * 1e-3, ms["relax"] * 1e-3, ms["df"] * 1e-3
    iters_per_step = iters_total / K
    exec_instr = job.pair_exec_instr()
    relax_bytes = 128.0 * iters_per_step + 18.0 * job.pixel_steps          # SURVEY 8(d) algorithmic bytes
    gathered = 128.0 * 32.0 * stats["warp_gathers"]                        # bytes the last step really gathered
    df_bytes = job.pixel_steps * 16.0 + job.df.numel() * 4.0
    rec = {
        "cfg": cfg, "steps": steps, "ms_per_step": t_step * 1e3, "pixel_steps_per_s": units_ps / t_step,
        "s_per_full_scan": t_step, "e2e_pixel_steps_per_s": e2e_units / e2e_t, "e2e_ms_per_step": e2e_t * 1e3,
        "kernel_ms": {k: round(v, 5) for k, v in ms.items() if v > 0},
        "ff_pairs_per_s": job.pairs / ff_s, "ff_pipe_frac_canonical": job.pairs / ff_s * PAIR_INSTR / alu_peak,
        "ff_pipe_frac_executed": exec_instr / ff_s / alu_peak,
        "ff_flop_frac": job.pairs / ff_s * PAIR_FLOPS / (2 * alu_peak),
        "relax_pixel_steps_per_s": job.pixel_steps / relax_s, "relax_iters_per_s": iters_per_step / relax_s,
        "relax_iters_per_pixel_step": iters_per_step / job.pixel_steps,
        "relax_alu_pipe_frac": iters_per_step * ITER_INSTR / relax_s / alu_peak,
        "relax_issued_pipe_frac": 32.0 * stats["warp_iters"] * ITER_INSTR / relax_s / alu_peak,
        "relax_lane_utilisation": stats["total_iters"] / max(1, 32 * stats["warp_iters"]),
        "relax_l2_algorithmic_gbs": relax_bytes / relax_s * 1e-9,
        "relax_l2_frac_of_cg_probe": relax_bytes / relax_s * 1e-9 / env["gather_cg"],
        "relax_l2_frac_of_ca_probe": relax_bytes / relax_s * 1e-9 / env["gather_ca"],
        "relax_gathered_gbs": gathered / relax_s * 1e-9,
        "relax_ms_guard": {"ms_per_step": ms["relax"], "limit": 1.1 * PERF_GUARD_RELAX_MS[cfg],
                           "ok": bool(ms["relax"] <= 1.1 * PERF_GUARD_RELAX_MS[cfg])},
        "df_hbm_frac": df_bytes / df_s * 1e-9 / peaks["hbm_gbs"],
        "not_converged": stats["n_not_converged"], "clamped": stats["n_clamped"], "max_iters": stats["max_iters"],
        "inputs_sha256": inputs_sha256(ws),
    }
    if cfg == 3:
        rec["molecules_per_s"] = len(ws) * world / t_step
    extra = {"job": job, "ms": ms, "n_launch": n_launch, "launches": launches, "clocks": clocks, "wall_s": wall_s,
             "stats": stats, "iters_per_step": iters_per_step, "exec_instr": exec_instr, "relax_bytes": relax_bytes,
             "gathered": gathered, "df_bytes": df_bytes, "t_step": t_step, "units_ps": units_ps,
             "units_pairs": units_pairs, "e2e_units": e2e_units, "e2e_t": e2e_t, "h2d": h2d, "d2h": d2h}
    return rec, extra


def next_rows(P, B, torch, job, ws, flush, env):
    """The SURVEY 8(f) rows measured beside the step on the headline config's resident grid and scan: stiffness map
    (N2) and tri-cubic relaxation (N4).  Eq.7 (N3) is measured on the configs[1] grid (see run_ours)."""
    peaks, alu_peak = env["peaks"], env["alu_peak"]
    out = {}
    eig = torch.empty((job.nps_one, 4), dtype=torch.float32, device="cuda")
    for rep in range(2 + 3):
        if rep == 2:
            B.timing_enable(True)
        flush.zero_()
        job.stiffness(eig)
    torch.cuda.synchronize()
    stiff_ms = B.timing_read()["stiffness"][0] / 3.0
    B.timing_enable(False)
    del eig
    n_samples = job.nps_one
    out["stiffness"] = {"kernel": "stiffness_kernel", "bound": "hbm", "unit": "GB/s", "peak": peaks["hbm_gbs"],
                        "achieved": 32.0 * n_samples / (stiff_ms * 1e-3) * 1e-9,
                        "frac": 32.0 * n_samples / (stiff_ms * 1e-3) * 1e-9 / peaks["hbm_gbs"], "ms": stiff_ms,
                        "samples": n_samples, "in_step": False, "traffic": ncu_traffic(job.cfg, "stiffness")}
    # the same map folded into the relaxation: cost = relax_scan_stiffness - relax_scan on the resident grid
    eig = torch.empty((job.nps_one, 4), dtype=torch.float32, device="cuda")
    st2 = P.new_stats()
    t_fused = t_plain = 0.0
    for rep in range(2 + 3):
        flush.zero_()
        B.timing_enable(True)
        job.relax_stiffness(eig, st2)
        torch.cuda.synchronize()
        a = B.timing_read()["relax"][0]
        B.timing_enable(True)
        flush.zero_()
        job.relax_plain(st2)
        torch.cuda.synchronize()
        b = B.timing_read()["relax"][0]
        if rep >= 2:
            t_fused += a / 3.0
            t_plain += b / 3.0
    B.timing_enable(False)
    del eig
    out["stiffness_fused"] = {"kernel": "relax_kernel<.,.,.,0,STIFF>", "relax_with_map_ms": t_fused, "relax_ms": t_plain,
                              "extra_ms": t_fused - t_plain, "extra_frac_of_relax": (t_fused - t_plain) / t_plain,
                              "standalone_kernel_ms": stiff_ms, "samples": n_samples, "in_step": False}
    E_only = P.energy_grid(job.ff[:job.npts])
    tri_stats = P.new_stats()
    for rep in range(1 + 2):
        if rep == 1:
            B.timing_enable(True)
        flush.zero_()
        tri_stats.zero_()
        job.relax_tricubic(E_only, tri_stats)
    torch.cuda.synchronize()
    tri_ms = B.timing_read()["relax_tricubic"][0] / 2.0
    tri = P.read_stats(tri_stats)
    B.timing_enable(False)
    del E_only
    tri_s = tri_ms * 1e-3
    out["relax_tricubic"] = {"kernel": "relax_kernel<.,.,.,TRICUBIC>", "bound": "alu", "unit": "TFLOP/s",
                             "achieved": tri["total_iters"] * TRI_FLOPS / tri_s * 1e-12, "peak": 2 * alu_peak * 1e-12,
                             "frac": tri["total_iters"] * TRI_FLOPS / tri_s / (2 * alu_peak),
                             "pipe_frac": tri["total_iters"] * TRI_INSTR / tri_s / alu_peak,
                             "issued_pipe_frac": 32.0 * tri["warp_iters"] * TRI_INSTR / tri_s / alu_peak,
                             "ms": tri_ms, "pixel_steps_per_s": job.nps_one / tri_s,
                             "iters_per_pixel_step": tri["total_iters"] / job.nps_one,
                             "not_converged": tri["n_not_converged"], "in_step": False, "traffic": None}
    # N4's energy-only force-field pass (ppfm_forcefield_energy) on the headline system, beside the float4 pass
    if len(ws) == 1:
        w = ws[0]
        xyzq, types = P.upload(w)
        E_out = torch.empty((w.grid.n[2], w.grid.n[1], w.grid.n[0]), dtype=torch.float32, device="cuda")
        for rep in range(1 + 2):
            if rep == 1:
                B.timing_enable(True)
            flush.zero_()
            P.forcefield_energy(xyzq, types, w.elem_R, w.elem_e, w.lattice, w.probe, w.grid, w.r_min, out=E_out)
        torch.cuda.synchronize()
        e_ms = B.timing_read()["ff_energy"][0] / 2.0
        B.timing_enable(False)
        del E_out
        e_s = e_ms * 1e-3
        out["ff_energy"] = {"kernel": "ffe_kernel", "bound": "alu", "unit": "TFLOP/s",
                            "achieved": w.pairs / e_s * ENERGY_PAIR_FLOPS * 1e-12, "peak": 2 * alu_peak * 1e-12,
                            "frac": w.pairs / e_s * ENERGY_PAIR_FLOPS / (2 * alu_peak),
                            "pipe_frac_executed": w.pairs / e_s * ENERGY_PAIR_INSTR / alu_peak,
                            "xu_pipe_frac": w.pairs / e_s / (alu_peak / 8.0),      # 1 MUFU.RSQ per pair, 16 XU lanes per SM
                            "pairs_per_s": w.pairs / e_s, "instr_per_pair_executed": ENERGY_PAIR_INSTR,
                            "flops_per_pair": ENERGY_PAIR_FLOPS, "ms": e_ms, "bytes_per_point": 4, "in_step": False,
                            "traffic": None}
    return out


def fft_row(P, B, torch, flush, env):
    """one Eq.7 call on the configs[1] grid (4 M points), CO-like quadrupole tip; V_S = any potential."""
    w = W.get(1)
    peaks = env["peaks"]
    npts = w.npoints
    Vs = torch.linspace(-1.0, 1.0, npts, device="cuda", dtype=torch.float32).reshape(w.grid.n[2], w.grid.n[1], w.grid.n[0])
    ff_fft = torch.empty((npts, 4), dtype=torch.float32, device="cuda")
    P.release_scratch()                      # cold: plans exist after the first call, the tip spectra do not
    P.forcefield_fft(Vs, w.grid, 0.7, -0.03, 0.0, -0.1, out=ff_fft)
    P.forcefield_fft(Vs, w.grid, 0.6, -0.03, 0.0, -0.1, out=ff_fft)
    P.forcefield_fft(Vs, w.grid, 0.5, -0.03, 0.0, -0.1, out=ff_fft)      # evicts the first tip
    torch.cuda.synchronize()
    B.timing_enable(True)
    flush.zero_()
    P.forcefield_fft(Vs, w.grid, 0.7, -0.03, 0.0, -0.1, out=ff_fft)      # tip spectra recomputed (5 + 4 transforms)
    torch.cuda.synchronize()
    miss_ms = B.timing_read()["fft_el"][0]
    B.timing_enable(True)
    for rep in range(3):
        flush.zero_()
        P.forcefield_fft(Vs, w.grid, 0.7, -0.03, 0.0, -0.1, out=ff_fft)  # cached tip spectra (1 + 4 transforms)
    torch.cuda.synchronize()
    fft_ms = B.timing_read()["fft_el"][0] / 3.0
    B.timing_enable(False)
    alg = 20.0 * npts       # algorithmic bytes: 4 B potential read + 16 B float4 written per grid point
    return {"kernel": "ppfm_forcefield_fft (own kernels + cuFFT FP64 transforms)", "bound": "hbm", "unit": "GB/s",
            "peak": peaks["hbm_gbs"], "achieved": alg / (fft_ms * 1e-3) * 1e-9,
            "frac": alg / (fft_ms * 1e-3) * 1e-9 / peaks["hbm_gbs"], "ms": fft_ms, "points": npts,
            "points_per_s": npts / (fft_ms * 1e-3), "ms_tip_spectra_not_cached": miss_ms, "in_step": False,
            "workload": "configs[1] grid, cached tip spectra",
            "traffic": ncu_traffic(1, "fft_el")}


def run_ours(args):
    import torch
    from paper_2401_14564_b200 import ppfm as P
    from paper_2401_14564_b200 import ppfm_bench as B

    rank, world, local_rank = shard.env_rank_world()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device — the ppfm hot path has no CPU fallback")
    P.lib()
    torch.cuda.set_device(local_rank % torch.cuda.device_count())
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", torch.cuda.current_device()))
    peaks = measured_peaks()
    alu_peak = SMS * LANES * peaks["sm_max_mhz"] * 1e6             # FP32 lane-instructions / s
    env = {"peaks": peaks, "alu_peak": alu_peak, "world": world,
           "fma_probe": B.probe_fma(),
           "gather_ca": B.probe_gather(2 << 20, False),     # 32 MiB volume: L2-resident; through L1 (L1-assisted)
           "gather_cg": B.probe_gather(2 << 20, True)}      # L1 bypassed: every request served by L2
    flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")     # > 126 MB L2
    cfg = args.config
    ws = build_workloads(cfg, rank, world, args.strong)
    head, x = measure_config(P, B, torch, cfg, ws, args.steps, args.warmup, max(1, min(args.steps, 5)), flush, env,
                             dist, sample_clocks=True)
    job, ms = x["job"], x["ms"]
    extra_rows = next_rows(P, B, torch, job, ws, flush, env) if rank == 0 or world == 1 else {}
    del job
    x["job"] = None
    P.release_scratch()
    torch.cuda.empty_cache()

    per_config = {}
    if world == 1 and not args.no_per_config:
        for c in (0, 1, 2, 3, 4):
            if c == cfg:
                per_config[str(c)] = head
                continue
            rec, xx = measure_config(P, B, torch, c, build_workloads(c, 0, 1), 3, 3, 2, flush, env)
            xx["job"] = None
            per_config[str(c)] = rec
            P.release_scratch()
            torch.cuda.empty_cache()
        extra_rows["fft_el"] = fft_row(P, B, torch, flush, env)
        P.release_scratch()

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---- rooflines of the headline config (rank 0's kernels; every rank runs the same launch configuration)
    ff_s, relax_s, df_s = ms["ff"] * 1e-3, ms["relax"] * 1e-3, ms["df"] * 1e-3
    pairs = sum(w.pairs for w in ws)
    rl_ff = {"kernel": "ff_kernel", "bound": "alu", "unit": "TFLOP/s", "achieved": pairs / ff_s * PAIR_FLOPS * 1e-12,
             "peak": 2 * alu_peak * 1e-12, "frac": pairs / ff_s * PAIR_FLOPS / (2 * alu_peak),
             "pipe_frac_canonical": head["ff_pipe_frac_canonical"], "pipe_frac_executed": head["ff_pipe_frac_executed"],
             "pipe_frac_canonical_of_fma_probe": pairs / ff_s * PAIR_INSTR / env["fma_probe"],
             "pairs_per_launch": pairs, "flops_per_pair": PAIR_FLOPS, "instr_per_pair_canonical": PAIR_INSTR,
             "instr_per_pair_executed": x["exec_instr"] / pairs, "ms": ms["ff"], "traffic": ncu_traffic(cfg, "ff")}
    ips = x["iters_per_step"]
    n_runs = len(ws[0].Q_sweep) if ws[0].Q_sweep else 1
    rl_relax = {"kernel": "relax_kernel", "bound": "alu", "unit": "TFLOP/s", "achieved": ips * ITER_FLOPS / relax_s * 1e-12,
                "peak": 2 * alu_peak * 1e-12, "frac": ips * ITER_FLOPS / relax_s / (2 * alu_peak),
                "pipe_frac": head["relax_alu_pipe_frac"], "issued_pipe_frac": head["relax_issued_pipe_frac"],
                "lane_utilisation": head["relax_lane_utilisation"], "iters_per_launch": ips / n_runs,
                "flops_per_iter": ITER_FLOPS, "instr_per_iter": ITER_INSTR, "ms": ms["relax"],
                "l2_view": {"bound": "l2", "unit": "GB/s", "algorithmic_bytes_per_step": x["relax_bytes"],
                            "achieved": head["relax_l2_algorithmic_gbs"], "peak_cg_l2_only": env["gather_cg"],
                            "peak_ca_l1_assisted": env["gather_ca"], "frac_of_cg": head["relax_l2_frac_of_cg_probe"],
                            "frac_of_ca": head["relax_l2_frac_of_ca_probe"], "gathered_gbs": head["relax_gathered_gbs"],
                            "gathered_share_of_algorithmic": x["gathered"] / max(1.0, 128.0 * ips)},
                "traffic": ncu_traffic(cfg, "relax")}
    rl_df = {"kernel": "df_kernel", "bound": "hbm", "unit": "GB/s", "achieved": x["df_bytes"] / df_s * 1e-9,
             "peak": peaks["hbm_gbs"], "frac": head["df_hbm_frac"], "bytes_per_step": x["df_bytes"], "ms": ms["df"],
             "traffic": ncu_traffic(cfg, "df")}
    kernels = {"ff": rl_ff, "relax": rl_relax, "df": rl_df}
    kernels.update(extra_rows)
    dominant = max(("ff", "relax", "df"), key=lambda k: ms[k])
    roof = dict(kernels[dominant])
    roof["share_of_step"] = ms[dominant] / (x["t_step"] * 1e3)
    roof["traffic_source"] = ncu_traffic(cfg, dominant, with_source=True)[1]
    compact = ("ms_per_step", "pixel_steps_per_s", "e2e_ms_per_step", "e2e_pixel_steps_per_s", "kernel_ms",
               "ff_pipe_frac_executed", "ff_flop_frac", "relax_alu_pipe_frac", "relax_issued_pipe_frac",
               "relax_lane_utilisation", "df_hbm_frac", "not_converged", "steps")
    roof["per_config"] = {c: {k: r[k] for k in compact if k in r} for c, r in per_config.items()}
    roof["peak_source"] = (f"{SMS} SMs x {LANES} FP32 lanes x {peaks['sm_max_mhz']:.0f} MHz x 2 (DESIGN.md 6.1)"
                           if roof["bound"] == "alu" else f"MEASURED_PEAKS.json hbm_gbs ({peaks['source']})")

    line = {"metric": METRIC, "value": head["pixel_steps_per_s"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": x["t_step"] * 1e3, "higher_is_better": True,
            "scaling": "strong" if args.strong else "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": WORKLOAD_NAME[cfg], "seed": BASE_SEED[cfg], "systems_per_gpu": len(ws),
                       "l2": "flushed between timed steps (512 MiB device write)",
                       "parallelism": ("single GPU" if world == 1 else
                                       f"one system in {world} row slabs (+4 A halo of grid rows), no exchange" if args.strong
                                       else f"replicated x{world}"),
                       "timing": "CUDA events on the launching stream, per step", "inputs_sha256": head["inputs_sha256"]},
            "parts": {"ff_pair_interactions_per_s": x["units_pairs"] / ff_s,
                      "ff_fp32_pipe_frac_canonical": head["ff_pipe_frac_canonical"],
                      "ff_fp32_pipe_frac_executed": head["ff_pipe_frac_executed"],
                      "relax_pixel_steps_per_s": x["units_ps"] / relax_s,
                      "relax_fire_iterations_per_s": ips * world / relax_s, "s_per_full_scan": x["t_step"],
                      "kernel_ms": {k: round(v, 5) for k, v in ms.items() if v > 0},
                      "kernel_launches_per_step": {k: v for k, v in x["n_launch"].items() if v > 0},
                      "wall_s_timed_region": x["wall_s"], "not_converged": head["not_converged"],
                      "clamped": head["clamped"], "max_iters": head["max_iters"],
                      "probes": {"fma_lane_instr_per_s": env["fma_probe"], "gather_cg_gbs": env["gather_cg"],
                                 "gather_ca_gbs": env["gather_ca"]},
                      "per_config": per_config},
            "e2e": {"value": x["e2e_units"] / x["e2e_t"], "unit": UNIT, "h2d_bytes_per_step": x["h2d"],
                    "d2h_bytes_per_step": x["d2h"], "ms_per_step": x["e2e_t"] * 1e3,
                    "api": "ppfm_scan_host[_batch|_sweep], pinned host buffers"},
            "gpu_launches": int(x["launches"]), "clocks": x["clocks"], "roofline": roof, "roofline_kernels": kernels}
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(ws[0])
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def spawn_ranks(n: int) -> int:
    """`python bench.py --gpus N` launched plainly (no torchrun environment): start N ranks of this same command, one
    process per GPU, the way the driver does (torch.distributed.run on 127.0.0.1, a free port), and return its exit
    code.  Rank 0 prints the JSON line; it passes through on the inherited stdout."""
    import socket
    import subprocess
    if args_impl(sys.argv) == "ours":
        import torch
        have = torch.cuda.device_count() if torch.cuda.is_available() else 0
        if have < n:
            raise SystemExit(f"bench.py: --gpus {n} needs {n} CUDA devices on this node, found {have} "
                             "(one process per GPU; ranks are never stacked on one device)")
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}", "--master-addr",
           "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.run(cmd).returncode


def args_impl(argv) -> str:
    for i, a in enumerate(argv):
        if a == "--impl" and i + 1 < len(argv):
            return argv[i + 1]
        if a.startswith("--impl="):
            return a.split("=", 1)[1]
    return "ours"


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4, choices=[0, 1, 2, 3, 4])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-per-config", action="store_true")
    ap.add_argument("--strong", action="store_true",
                    help="with --gpus N > 1: split ONE system across the ranks (row slabs + halo) instead of replicating")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 0)
    if args.gpus < 1:
        raise SystemExit("bench.py: --gpus must be >= 1")
    if "WORLD_SIZE" not in os.environ and args.gpus > 1:
        raise SystemExit(spawn_ranks(args.gpus))
    world = shard.env_rank_world()[1]
    if world != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but the launcher started WORLD_SIZE={world} ranks")
    if args.impl == "reference":
        run_reference(args)
    else:
        if args.warmup < 3:
            args.warmup = 3          # timing rule: at least 3 warm-up steps
        run_ours(args)


if __name__ == "__main__":
    main()
