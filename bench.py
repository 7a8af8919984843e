#!/usr/bin/env python
"""bench.py — one "step" = one pass of the whole hot path (force-field grid -> FIRE relaxation scan -> df) over one
seeded synthetic workload (BASELINE.json configs; default configs[1]).  Prints ONE JSON line (rank 0).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference] [--no-cpu-baseline]

* `value` (device-resident inputs): relaxed pixel-steps per second over the full scan, CUDA-event timed per step on
  the launching stream, L2 flushed between steps, max over ranks.  `parts` carries the other two thirds of
  BASELINE.json's metric (FF pair-interactions/s with its FP32 fraction, seconds per full scan) and the
  relax kernel's own rate.
* `e2e`: the same scan through the one-call host API ppfm_scan_host with pinned HOST buffers (H2D of the atoms and
  D2H of positions, iteration counts and df inside the timed region).
* `roofline`: the step's dominant kernel; `roofline_kernels` all three.  FF is ALU-bound (peak = SMs x 128 FP32
  lanes x max SM clock), relax is bound by the cache gather rate (peak = the in-run gather
  micro-benchmark = "achievable L2 bandwidth"), df streams HBM (peak = MEASURED_PEAKS.json hbm_gbs).
* `cpu_baseline`: the FP64 oracle, as it stands, timed on this box's host cores on a bounded sample.
* `--impl reference`: the oracle arm (this tier has no reference implementation to install).
The oracle is imported ONLY by the cpu_baseline leg and the reference arm.
"""
from __future__ import annotations

import argparse
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
# canonical algorithmic work per pair interaction: 19 FP32-pipe instructions, 28 flops
PAIR_INSTR, PAIR_FLOPS = 19, 28
# what ff_kernel executes per pair and grid point (ff.cu inner loop, FP32x2-packed): 15 FP32-pipe lane-instructions
# + 1 MUFU for an atom with a Coulomb factor, 13 + 1 for an LJ-only atom (split kernel: 20 / 14)
PAIR_EXEC = {"charged": 15, "neutral": 13, "charged_split": 20, "neutral_split": 14}
# what relax_kernel's cached-cell iteration needs (relax.cu, symmetric tip): 44 FFMA + 13 FMUL + 13 FADD = 70
# FP32-pipe lane-instructions = 114 flops, + 4 MUFU
ITER_INSTR, ITER_FLOPS = 70, 114
SMS, LANES = 148, 128
# dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed `ncu --set full` captures (profiles/);
# None where no capture exists for that kernel and config.
NCU_TRAFFIC = {(1, "ff"): 6.59e6, (1, "relax"): 13.59e6, (1, "df"): 14.41e6, (1, "stiffness"): 27.43e6,
               (1, "fft_el"): 2.06e9, (2, "ff"): 188.8e6,
               (3, "ff"): 1.0149e9, (3, "relax"): 513.8e6, (3, "df"): 454.7e6}      # profiles/r01e_full_cfg{1,2,3}*.txt


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return {"hbm_gbs": float(d["hbm_gbs"]), "sm_max_mhz": float(d.get("sm_max_mhz", 1965.0)), "source": "measured"}
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "source": "fallback"}


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
            self._stop.wait(0.002)      # short timed regions (configs 0, 1: ~20 ms) still get several samples

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
def build_workloads(cfg: int, rank: int, world: int):
    """This rank's systems (weak scaling: an independent seeded draw of the same config per rank)."""
    seed = shard.rank_seed(BASE_SEED[cfg], rank)
    if cfg == 3:
        return W.config3(64, seed=seed)
    return [W.get(cfg, seed=seed)]


class DeviceJob:
    """Device-resident buffers of one rank's systems and the step that runs the three entry points on them."""

    def __init__(self, P, torch, cfg, ws):
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
        self.ff = torch.empty((npts, 4), dtype=torch.float32, device="cuda")
        if self.sweep:
            self.ff_lj = torch.empty_like(self.ff)
            self.ff_el = torch.empty_like(self.ff)
        self.pos = torch.empty((nps, 4), dtype=torch.float32, device="cuda")
        self.iters = torch.empty((nps,), dtype=torch.int16, device="cuda")
        self.df = torch.empty((len(ws) * (s.nz - w0.n_df) * s.npy * s.npx,), dtype=torch.float32, device="cuda")
        self.stats = P.new_stats()
        # argument marshalling done once: ready ctypes structs pass straight through the binding
        self.c_lat = P.c_array([w.lattice for w in ws], P.c_lattice)
        self.c_probe = P.c_array([w.probe for w in ws], P.c_probe)
        self.c_grid = P.c_array([w.grid for w in ws], P.c_grid)
        self.c_tip = P.c_array([w.tip for w in ws], P.c_tip)
        self.c_scan = P.c_array([w.scan for w in ws], P.c_scan)
        self.c_fire = P.c_fire(w0.fire)
        import ctypes
        self.c_off = (ctypes.c_int32 * (len(ws) + 1))(*[int(v) for v in self.off])
        self.pairs = float(sum(w.pairs for w in ws))
        self.pixel_steps = float(nps * (len(self.sweep) if self.sweep else 1))
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
        """The scan of step() on the energy-only grid E with tri-cubic interpolation (last Q of a sweep)."""
        P = self.P
        if self.batch:
            P.relax_scan_tricubic_batch(E, self.c_grid, self.c_tip, self.c_fire, self.c_scan, pos_fz=self.pos,
                                        iters=self.iters, stats=stats)
        else:
            P.relax_scan_tricubic(E, self.c_grid[0], self.c_tip[0], self.c_fire, self.c_scan[0], pos_fz=self.pos,
                                  iters=self.iters, stats=stats)

    def stiffness(self, out):
        """Stiffness map of the scan held in self.pos (last Q of a sweep) on the resident grid."""
        P, ws = self.P, self.ws
        if self.batch:
            P.stiffness_batch(self.ff, self.c_grid, self.c_tip, self.c_scan, self.pos, out=out)
        else:
            P.stiffness(self.ff, self.c_grid[0], self.c_tip[0], self.c_scan[0], self.pos, out=out)

    def _mark(self, name):
        ev = self.torch.cuda.Event(enable_timing=True)
        ev.record()
        self.marks.append((name, ev))

    def step(self):
        """Enqueue one full scan; event marks separate the kernels (all on torch's current stream)."""
        P, ws, w0 = self.P, self.ws, self.ws[0]
        s = w0.scan
        self.marks = []
        self._mark("start")
        if self.batch:
            P.forcefield_batch(self.c_off, self.xyzq, self.types, w0.elem_R, w0.elem_e, self.c_lat, self.c_probe,
                               self.c_grid, w0.r_min, out=self.ff)
            self._mark("ff")
            P.relax_scan_batch(self.ff, self.c_grid, self.c_tip, self.c_fire, self.c_scan,
                               pos_fz=self.pos, iters=self.iters, stats=self.stats)
            self._mark("relax")
            P.df(self.pos, s.npx, s.npy, s.nz, s.dz, w0.df.A, w0.df.k0, w0.df.f0, out=self.df, nsys=len(ws))
            self._mark("df")
        elif self.sweep:
            P.forcefield_split(self.xyzq, self.types, w0.elem_R, w0.elem_e, self.c_lat[0], self.c_probe[0],
                               self.c_grid[0], w0.r_min, out_lj=self.ff_lj, out_el=self.ff_el)
            self._mark("ff")
            for Q in self.sweep:
                P.combine(self.ff_lj, self.ff_el, Q, out=self.ff)
                self._mark("combine")
                P.relax_scan(self.ff, self.c_grid[0], self.c_tip[0], self.c_fire, self.c_scan[0], pos_fz=self.pos,
                             iters=self.iters, stats=self.stats)
                self._mark("relax")
                P.df(self.pos, s.npx, s.npy, s.nz, s.dz, w0.df.A, w0.df.k0, w0.df.f0, out=self.df)
                self._mark("df")
        else:
            P.forcefield(self.xyzq, self.types, w0.elem_R, w0.elem_e, self.c_lat[0], self.c_probe[0], self.c_grid[0],
                         w0.r_min, out=self.ff)
            self._mark("ff")
            P.relax_scan(self.ff, self.c_grid[0], self.c_tip[0], self.c_fire, self.c_scan[0], pos_fz=self.pos,
                         iters=self.iters, stats=self.stats)
            self._mark("relax")
            P.df(self.pos, s.npx, s.npy, s.nz, s.dz, w0.df.A, w0.df.k0, w0.df.f0, out=self.df)
            self._mark("df")

    def durations_ms(self):
        """After a synchronise: (total ms, {kernel: ms}) of the last step from its event marks."""
        out = {}
        for (_, e0), (name, e1) in zip(self.marks[:-1], self.marks[1:]):
            out[name] = out.get(name, 0.0) + e0.elapsed_time(e1)
        return self.marks[0][1].elapsed_time(self.marks[-1][1]), out


class HostJob:
    """The same scan through ppfm_scan_host: pinned host buffers in and out, copies inside the timed region."""

    def __init__(self, P, torch, ws):
        from dataclasses import replace as _replace
        # argument marshalling done once (as DeviceJob does): ready ctypes structs pass straight through the binding
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
            self.h2d += nq * (hx.numel() * 4 + ht.numel() * 4)
            self.d2h += nq * (hp.numel() * 4 + hi.numel() * 2 + hd.numel() * 4 + 32)

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
def oracle_sample_run(w, n_points: int, n_pixels: int, seed: int = 7, ff_full=None):
    """Time the oracle, as it stands, on a bounded sample of workload `w`: `n_points` seeded grid points of the force
    field, then the relaxation scan + df of the central `n_pixels` pixels on the oracle's own FP64 grid, built only
    over the sub-volume those pixels can reach (lateral margin 4 A; building it is not timed).  Where that sub-grid
    alone would cost more than ~2e9 pair evaluations (configs 2 and 4) and `ff_full` (a full float32 grid, widened to
    FP64 on access) is given, the relaxation leg runs on it instead — timing only, labelled in `grid_kind`.
    Returns timings and the extrapolated full-scan rate."""
    from dataclasses import replace

    from oracle import oracle
    t0 = time.perf_counter()
    idx = W.sample_indices(w.npoints, n_points, seed)
    oracle.forcefield(w, idx=idx)
    t_ff = time.perf_counter() - t0
    ff_pairs = float(len(idx)) * w.natoms * w.nimages
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
    if sub_cost > 2e9 and ff_full is not None:
        grid_kind = "full float32 grid produced by the CUDA path, widened on access (timing only)"
        iy, ix = np.meshgrid(np.arange(iy0, iy0 + side_y), np.arange(ix0, ix0 + side_x), indexing="ij")
        pix = (iy * s.npx + ix).ravel()
        t_grid = 0.0
        t2 = time.perf_counter()
        r = oracle.relax_scan(ff_full, g, w.tip, w.fire, s, pix=pix, traj=False)
        t_relax = time.perf_counter() - t2
    else:
        if sub_cost > 2e10:
            raise RuntimeError("oracle sub-grid for the relaxation sample is not affordable for this config")
        grid_kind = f"oracle FP64 sub-grid {list(sub_n)}"
        sub_grid = replace(g, origin=g.origin + np.array([i_lo[0] * h[0], i_lo[1] * h[1], 0.0]), n=sub_n,
                           periodic=(0, 0, 0))
        t1 = time.perf_counter()
        ff_sub = oracle.forcefield(replace(w, grid=sub_grid))
        t_grid = time.perf_counter() - t1
        t2 = time.perf_counter()
        r = oracle.relax_scan(ff_sub, sub_grid, w.tip, w.fire, sub_scan, traj=False)
        t_relax = time.perf_counter() - t2
    t3 = time.perf_counter()
    oracle.df(r["pos_fz"][..., 3], s.dz, w.df.A, w.df.k0, w.df.f0)
    t_df = time.perf_counter() - t3
    nq = len(w.Q_sweep) if w.Q_sweep else 1
    pix_n = side_x * side_y
    ff_rate = ff_pairs / t_ff
    relax_rate = pix_n * s.nz / (t_relax + t_df)
    full_s = w.pairs / ff_rate + nq * w.pixel_steps / relax_rate
    return {"t_ff": t_ff, "t_grid": t_grid, "t_relax": t_relax, "t_df": t_df, "ff_pairs_per_s": ff_rate,
            "relax_pixel_steps_per_s": relax_rate, "s_per_full_scan_extrapolated": full_s,
            "value": nq * w.pixel_steps / full_s, "sample_points": int(len(idx)), "sample_pixels": int(pix_n),
            "grid_kind": grid_kind, "iters_per_pixel_step": float(np.abs(r["iters"]).mean()),
            "cores": oracle.num_threads()}


def sample_sizes(w, target_s: float, ff_full=None):
    """Sample sizes for about `target_s` seconds of oracle work, from a quick calibration run."""
    cal = oracle_sample_run(w, 2000, 16, ff_full=ff_full)
    n_points = int(min(w.npoints, max(2000, 0.35 * target_s * cal["ff_pairs_per_s"] / (w.natoms * w.nimages))))
    n_pixels = int(min(w.scan.npx * w.scan.npy, max(16, 0.45 * target_s * cal["relax_pixel_steps_per_s"] / w.scan.nz)))
    return n_points, n_pixels


def cpu_baseline(w, target_s: float = 15.0, ff_full=None):
    n_points, n_pixels = sample_sizes(w, target_s, ff_full)
    r = oracle_sample_run(w, n_points, n_pixels, ff_full=ff_full)
    return {"value": r["value"], "unit": UNIT, "cores": r["cores"], "kind": "oracle",
            "sample": (f"FP64 oracle (gcc -O2, OpenMP): force field at {r['sample_points']} seeded grid points "
                       f"({r['t_ff']:.1f} s), relaxation + df of the central {r['sample_pixels']} pixels x all z-steps "
                       f"on {r['grid_kind']} ({r['t_relax'] + r['t_df']:.1f} s; grid build "
                       f"{r['t_grid']:.1f} s not counted); value = pixel-steps / (pairs / oracle pair rate + "
                       f"pixel-steps / oracle relax rate), extrapolated to the full workload"),
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
    sample = (f"each step: oracle force field at {r['sample_points']} seeded grid points + relaxation/df of the central "
              f"{r['sample_pixels']} pixels on {r['grid_kind']}; value extrapolated to the full workload")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * wall / max(1, args.steps),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD_NAME[args.config], "seed": BASE_SEED[args.config]},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": r["cores"], "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------- our arm
def run_ours(args):
    import torch
    from paper_2401_14564_b200 import ppfm as P

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
    cfg = args.config
    ws = build_workloads(cfg, rank, world)
    job = DeviceJob(P, torch, cfg, ws)
    flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")     # > 126 MB L2

    # ---- device-resident arm
    for _ in range(args.warmup):
        flush.zero_()
        job.stats.zero_()
        job.step()
    torch.cuda.synchronize()
    shard.barrier(dist)
    sampler = ClockSampler(torch.cuda.current_device())
    sampler.start()
    n0 = P.launch_count()
    P.timing_enable(True)          # per-kernel CUDA events recorded inside the library, directly around each launch
    tot_ms, kern_ms, iters_total = 0.0, {}, 0
    t_wall0 = time.perf_counter()
    for _ in range(args.steps):
        flush.zero_()
        job.stats.zero_()
        job.step()
        torch.cuda.synchronize()
        t, k = job.durations_ms()
        tot_ms += t
        for name, v in k.items():
            kern_ms[name] = kern_ms.get(name, 0.0) + v
        iters_total += P.read_stats(job.stats)["total_iters"]
    torch.cuda.synchronize()
    shard.barrier(dist)
    wall_s = time.perf_counter() - t_wall0
    launches = P.launch_count() - n0
    clocks = sampler.stop()
    kern = P.timing_read()
    P.timing_enable(False)
    K = max(1, args.steps)
    stats = P.read_stats(job.stats)

    # ---- stiffness map on the scan just relaxed: measured beside the step, not part of it
    eig = torch.empty_like(job.pos)
    stiff_ms = None
    for rep in range(3 + 5):
        if rep == 3:
            P.timing_enable(True)
        flush.zero_()
        job.stiffness(eig)
    torch.cuda.synchronize()
    stiff_ms = P.timing_read()["stiffness"][0] / 5.0
    P.timing_enable(False)
    del eig

    # ---- tri-cubic relaxation of the same scan on the energy-only grid: beside the step
    E_only = P.energy_grid(job.ff)
    tri_stats = P.new_stats()
    for rep in range(2 + 3):
        if rep == 2:
            P.timing_enable(True)
        flush.zero_()
        tri_stats.zero_()
        job.relax_tricubic(E_only, tri_stats)
    torch.cuda.synchronize()
    tri_ms = P.timing_read()["relax_tricubic"][0] / 3.0
    tri = P.read_stats(tri_stats)
    P.timing_enable(False)
    del E_only

    # ---- Eq.7 electrostatics on the first system's grid: V_S = the .w lane of the resident grid
    # (any potential serves for timing), CO-like quadrupole tip; measured beside the step, not part of it
    w0g = ws[0].grid
    npts0 = ws[0].npoints
    Vs = job.ff[:npts0, 3].contiguous()
    ff_fft = torch.empty((npts0, 4), dtype=torch.float32, device="cuda")
    for rep in range(2 + 3):
        if rep == 2:
            P.timing_enable(True)
        flush.zero_()
        P.forcefield_fft(Vs, w0g, 0.7, -0.03, 0.0, -0.1, out=ff_fft)
    torch.cuda.synchronize()
    fft_ms = P.timing_read()["fft_el"][0] / 3.0
    P.timing_enable(False)
    del Vs, ff_fft
    P.release_scratch()
    (units_ps, units_pairs), t_step = shard.aggregate([job.pixel_steps, job.pairs], tot_ms / K * 1e-3, dist)
    value = units_ps / t_step

    # ---- end-to-end arm (host buffers through ppfm_scan_host)
    host = HostJob(P, torch, ws)
    for _ in range(max(1, min(args.warmup, 3))):
        host.step()
    torch.cuda.synchronize()
    shard.barrier(dist)
    e2e_steps = max(1, min(args.steps, 10))
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        host.step()
    torch.cuda.synchronize()
    e2e_local = (time.perf_counter() - t0) / e2e_steps
    shard.barrier(dist)
    (e2e_units,), e2e_t = shard.aggregate([job.pixel_steps], e2e_local, dist)

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---- rooflines (rank 0's kernels; every rank runs the same launch configuration)
    seg_ms = {k: v / K for k, v in kern_ms.items()}          # event marks around the Python calls (with host gaps)
    ms = {k: v[0] / K for k, v in kern.items()}             # the kernels themselves, per step
    n_launch = {k: v[1] / K for k, v in kern.items()}
    n_relax_launches = len(job.sweep) if job.sweep else 1
    fma_probe = P.probe_fma()
    gather_ca = P.probe_gather(2 << 20, False)       # 32 MiB volume: L2-resident
    gather_cg = P.probe_gather(2 << 20, True)
    alu_peak = SMS * LANES * peaks["sm_max_mhz"] * 1e6             # FP32 lane-instructions / s
    ff_s = ms["ff"] * 1e-3
    ff_pairs_s = job.pairs / ff_s
    exec_instr = job.pair_exec_instr()                            # lane-instructions the kernel really executes
    rl_ff = {"kernel": "ff_kernel", "bound": "alu", "achieved": ff_pairs_s * PAIR_FLOPS * 1e-12,
             "peak": 2 * alu_peak * 1e-12, "unit": "TFLOP/s", "frac": ff_pairs_s * PAIR_FLOPS / (2 * alu_peak),
             "pipe_frac": ff_pairs_s * PAIR_INSTR / alu_peak,
             "pipe_frac_of_probe": ff_pairs_s * PAIR_INSTR / fma_probe,
             "pipe_frac_executed": exec_instr / ff_s / alu_peak,
             "peak_source": f"{SMS} SMs x {LANES} FP32 lanes x {peaks['sm_max_mhz']:.0f} MHz x 2 (FMA); "
                            f"in-run FFMA probe {fma_probe * 1e-12:.2f} T lane-instr/s",
             "algorithmic": f"{PAIR_FLOPS} flops / {PAIR_INSTR} FP32-pipe instructions per pair (SURVEY 8(d) canonical "
                            f"count) x {job.pairs:.4g} pairs per launch; the kernel's own formulation executes "
                            f"{exec_instr / job.pairs:.2f} lane-instructions per pair (pipe_frac_executed, comparable "
                            f"with ncu sm__pipe_fma_cycles_active), so pipe_frac can pass 1",
             "ms": ms["ff"], "traffic": NCU_TRAFFIC.get((cfg, "ff"))}
    relax_s = ms["relax"] * 1e-3
    iters_per_step = iters_total / K
    relax_bytes = 128.0 * iters_per_step + 18.0 * job.pixel_steps
    gather_peak = max(gather_ca, gather_cg)
    gathered = 128.0 * 32.0 * stats["warp_gathers"]                 # bytes the last step's launches really gathered
    rl_relax = {"kernel": "relax_kernel", "bound": "l2", "achieved": relax_bytes / relax_s * 1e-9,
                "peak": gather_peak, "unit": "GB/s", "frac": relax_bytes / relax_s * 1e-9 / gather_peak,
                "peak_source": f"in-run 8-corner float4 gather micro-benchmark over a 32 MiB (L2-resident) volume: "
                               f"ld.global.ca {gather_ca:.0f} GB/s, ld.global.cg {gather_cg:.0f} GB/s",
                "algorithmic": f"SURVEY 8(d): 128 B (8 corners x float4) x {iters_per_step:.4g} FIRE iterations + 18 B x "
                               f"{job.pixel_steps:.4g} pixel-steps per step ({n_relax_launches} launch(es)).  The kernel "
                               f"holds the current cell in registers and gathers only when the probe particle leaves "
                               f"it, so it moves a fraction of these bytes (gathered_share_of_algorithmic) and frac can "
                               f"pass 1 on large scans; what then binds is instruction issue, see alu_view",
                "gathered_gbs": gathered / relax_s * 1e-9,
                "gathered_share_of_algorithmic": gathered / max(1.0, 128.0 * iters_per_step),
                "ms": ms["relax"], "iters_per_pixel_step": iters_per_step / job.pixel_steps,
                "alu_view": {"bound": "alu", "unit": "TFLOP/s",
                             "achieved": iters_per_step * ITER_FLOPS / relax_s * 1e-12, "peak": 2 * alu_peak * 1e-12,
                             "frac": iters_per_step * ITER_FLOPS / relax_s / (2 * alu_peak),
                             "pipe_frac": iters_per_step * ITER_INSTR / relax_s / alu_peak,
                             "issued_pipe_frac": 32.0 * stats["warp_iters"] * ITER_INSTR / relax_s / alu_peak,
                             "algorithmic": f"{ITER_FLOPS} flops / {ITER_INSTR} FP32-pipe lane-instructions (+ 4 MUFU) per "
                                            f"FIRE iteration in the cached-cell formulation; issued_pipe_frac counts the "
                                            f"lanes that idle in a warp until its slowest pixel converges",
                             "peak_source": f"{SMS} SMs x {LANES} FP32 lanes x {peaks['sm_max_mhz']:.0f} MHz x 2 (FMA)"},
                "traffic": NCU_TRAFFIC.get((cfg, "relax"))}
    df_bytes = (job.pixel_steps * 16.0 + job.df.numel() * 4.0 * n_relax_launches)
    rl_df = {"kernel": "df_kernel", "bound": "hbm", "achieved": df_bytes / (ms["df"] * 1e-3) * 1e-9,
             "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": df_bytes / (ms["df"] * 1e-3) * 1e-9 / peaks["hbm_gbs"],
             "peak_source": f"MEASURED_PEAKS.json hbm_gbs ({peaks['source']})",
             "algorithmic": "16 B read per pixel-step (float4 stack, Fz in .w) + 4 B written per df sample",
             "ms": ms["df"], "traffic": NCU_TRAFFIC.get((cfg, "df"))}
    n_samples = job.pos.shape[0]
    rl_stiff = {"kernel": "stiffness_kernel", "bound": "hbm", "achieved": 32.0 * n_samples / (stiff_ms * 1e-3) * 1e-9,
                "peak": peaks["hbm_gbs"], "unit": "GB/s",
                "frac": 32.0 * n_samples / (stiff_ms * 1e-3) * 1e-9 / peaks["hbm_gbs"],
                "peak_source": f"MEASURED_PEAKS.json hbm_gbs ({peaks['source']})",
                "algorithmic": "16 B position read + 16 B eigenvalues written per (pixel, z-step) sample; the 8-corner "
                               "gather (128 B per sample) is served by L1/L2 and the touched grid slab is read from "
                               "HBM once",
                "ms": stiff_ms, "samples": n_samples, "in_step": False, "traffic": NCU_TRAFFIC.get((cfg, "stiffness"))}
    # 5 forward + 4 inverse FP64 3-D transforms; each touches its array (16 B per complex point, N/2 of them) about
    # three times in each direction; plus fill (4 B read, 40 B written), spectral (80 B r/w per complex point on N/2
    # points), pack (32 B read, 16 B written) -> ~ 9 * 3 * 2 * 8 + 44 + 80 + 48 = 604 B per grid point as the model
    fft_model_bytes = 604.0 * npts0
    rl_fft = {"kernel": "ppfm_forcefield_fft (fill + cuFFT D2Z x5 + spectral + cuFFT Z2D x4 + pack)", "bound": "hbm",
              "achieved": fft_model_bytes / (fft_ms * 1e-3) * 1e-9, "peak": peaks["hbm_gbs"], "unit": "GB/s",
              "frac": fft_model_bytes / (fft_ms * 1e-3) * 1e-9 / peaks["hbm_gbs"],
              "peak_source": f"MEASURED_PEAKS.json hbm_gbs ({peaks['source']})",
              "algorithmic": "traffic model 604 B per grid point: nine FP64 3-D FFTs at three read+write passes each "
                             "(8 B per real point per pass) + fill + spectral product + pack; the transforms are "
                             "cuFFT (library), the three kernels around them are this library's",
              "ms": fft_ms, "points": npts0, "points_per_s": npts0 / (fft_ms * 1e-3), "in_step": False,
              "traffic": NCU_TRAFFIC.get((cfg, "fft_el"))}
    # tri-cubic iteration (relax.cu): weights 42 + x pass 128 + y pass 48 + z pass 12 + metric 3 = 233 FP32-pipe
    # lane-instructions for the field (tri-linear: 33), the rest of the iteration as above (37): 270 = 2 * 244 + 26
    TRI_INSTR, TRI_FLOPS = 270, 514
    tri_s = tri_ms * 1e-3
    rl_tri = {"kernel": "relax_kernel<.,.,.,TRICUBIC>", "bound": "alu", "unit": "TFLOP/s",
              "achieved": tri["total_iters"] * TRI_FLOPS / tri_s * 1e-12, "peak": 2 * alu_peak * 1e-12,
              "frac": tri["total_iters"] * TRI_FLOPS / tri_s / (2 * alu_peak),
              "pipe_frac": tri["total_iters"] * TRI_INSTR / tri_s / alu_peak,
              "issued_pipe_frac": 32.0 * tri["warp_iters"] * TRI_INSTR / tri_s / alu_peak,
              "peak_source": f"{SMS} SMs x {LANES} FP32 lanes x {peaks['sm_max_mhz']:.0f} MHz x 2 (FMA)",
              "algorithmic": f"{TRI_FLOPS} flops / {TRI_INSTR} FP32-pipe lane-instructions per FIRE iteration (64-point "
                             f"stencil held in registers) x {tri['total_iters']:.4g} iterations",
              "ms": tri_ms, "pixel_steps_per_s": job.pos.shape[0] / tri_s,
              "iters_per_pixel_step": tri["total_iters"] / job.pos.shape[0], "not_converged": tri["n_not_converged"],
              "grid_bytes_per_point": 4, "in_step": False, "traffic": NCU_TRAFFIC.get((cfg, "relax_tricubic"))}
    kernels = {"ff": rl_ff, "relax": rl_relax, "df": rl_df, "stiffness": rl_stiff, "fft_el": rl_fft,
               "relax_tricubic": rl_tri}
    for k in kernels:
        kernels[k]["timing"] = "CUDA events recorded inside libppfm directly around the launch, mean per step"
    dominant = max(("ff", "relax", "df"), key=lambda k: ms[k])
    roof = dict(kernels[dominant])
    roof["share_of_step"] = ms[dominant] / (tot_ms / K)

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": t_step * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": WORKLOAD_NAME[cfg], "seed": BASE_SEED[cfg], "systems_per_gpu": len(ws),
                       "l2": "flushed between timed steps (512 MiB device write)", "parallelism": f"replicated x{world}"
                       if world > 1 else "single GPU", "timing": "CUDA events on the launching stream, per step"},
            "parts": {"ff_pair_interactions_per_s": units_pairs / (ms["ff"] * 1e-3),
                      "ff_fp32_flop_frac": rl_ff["frac"], "ff_fp32_pipe_frac": rl_ff["pipe_frac"],
                      "relax_pixel_steps_per_s": units_ps / relax_s,
                      "relax_fire_iterations_per_s": iters_per_step * world / relax_s,
                      "s_per_full_scan": t_step, "kernel_ms": ms, "kernel_launches_per_step": n_launch,
                      "call_ms_incl_host_gaps": seg_ms, "wall_s_timed_region": wall_s,
                      "not_converged": stats["n_not_converged"], "clamped": stats["n_clamped"],
                      "max_iters": stats["max_iters"],
                      "relax_warp_loop_trips": stats["warp_iters"],
                      "relax_lane_utilisation": stats["total_iters"] / max(1, 32 * stats["warp_iters"]),
                      "relax_cell_changes_per_iteration": stats["cell_gathers"] / max(1, stats["total_iters"]),
                      "relax_gather_trips_per_loop_trip": stats["warp_gathers"] / max(1, stats["warp_iters"])},
            "e2e": {"value": e2e_units / e2e_t, "unit": UNIT, "h2d_bytes_per_step": host.h2d,
                    "d2h_bytes_per_step": host.d2h, "ms_per_step": e2e_t * 1e3, "steps": e2e_steps,
                    "api": "ppfm_scan_host[_batch|_sweep] (pinned host buffers: inputs copied in, outputs stored by the kernels straight into host memory)"},
            "gpu_launches": int(launches), "clocks": clocks, "roofline": roof, "roofline_kernels": kernels}
    if world == 1 and not args.no_cpu_baseline:
        w0 = ws[0]
        ff_full = None
        if not job.batch and w0.npoints * w0.natoms * w0.nimages > 1e10:      # configs 2 and 4 (see oracle_sample_run)
            ff_full = job.ff.cpu().numpy().reshape(w0.grid.n[2], w0.grid.n[1], w0.grid.n[0], 4)
        line["cpu_baseline"] = cpu_baseline(w0, ff_full=ff_full)
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=1, choices=[0, 1, 2, 3, 4])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 0)
    if args.impl == "reference":
        run_reference(args)
    else:
        if args.warmup < 3:
            args.warmup = 3          # timing rule: at least 3 warm-up steps
        run_ours(args)


if __name__ == "__main__":
    main()
