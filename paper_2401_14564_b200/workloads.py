"""Seeded synthetic workloads (the five BASELINE.json configs) — inputs only.

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none of the method's
arithmetic: no Lennard-Jones, no Coulomb, no interpolation, no FIRE, no Giessibl weights.  It only
draws geometry / charges / parameters with a seeded numpy PCG64 generator and fixes grid and scan
specifications.  Every real-valued *array* input (atom
positions and charges) is rounded to FP32 and widened again, so the FP64 oracle and the FP32 kernels see
bit-identical numbers.

The paper's own inputs (molecular geometries + Mulliken charges) are a Zenodo
data set that is not available here; these generators stand in for it with the shapes, sizes and value
ranges of the paper's workloads.
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace
from typing import List, Optional, Tuple

import numpy as np

# ---- unit constants (SURVEY.md §8 header, S4).  Plain conversions, not method arithmetic. -------------
EVA2_PER_NM = 1.0 / 16.02176634          # 1 N/m in eV/Å^2  (1 eV/Å^2 = 16.02176634 N/m)

# element table (R_i Å, e_i eV) as printed in BASELINE.json config 0 / config 2 (S5)
ELEMENTS = ("H", "C", "N", "O", "X")
ELEM_R = np.array([1.487, 1.908, 1.78, 1.661, 1.7], dtype=np.float64)
ELEM_E = np.array([6.81e-4, 3.73e-3, 3.04e-3, 9.11e-3, 4.0e-3], dtype=np.float64)
T_H, T_C, T_N, T_O, T_X = range(5)


@dataclass
class Lattice:
    a: np.ndarray                      # cell vectors (Å)
    b: np.ndarray
    c: np.ndarray
    nimg: Tuple[int, int, int]         # images -nimg..+nimg per axis


@dataclass
class Grid:
    origin: np.ndarray                 # (3,) Å
    step: np.ndarray                   # (3,3): point(i,j,k) = origin + i*step[0] + j*step[1] + k*step[2]
    n: Tuple[int, int, int]            # (nx, ny, nz); storage [nz][ny][nx][4], x fastest
    periodic: Tuple[int, int, int]


@dataclass
class Probe:
    R: float
    e: float
    Q: float


@dataclass
class Tip:
    k_lat: Tuple[float, float]         # eV/Å^2
    k_rad: float                       # eV/Å^2
    d0: Tuple[float, float, float]     # equilibrium displacement r_PP0 - r_TIP (Å)


@dataclass
class Fire:
    dt: float = 0.5
    dt_max: float = 0.5
    finc: float = 1.1
    fdec: float = 0.5
    alpha0: float = 0.1
    falpha: float = 0.99
    n_min: int = 5
    max_iter: int = 1000
    f_conv: float = 1e-6


@dataclass
class Scan:
    p0: np.ndarray                     # anchor of pixel (0,0) at iz = 0 (Å)
    dx: np.ndarray                     # pixel step vectors (Å)
    dy: np.ndarray
    npx: int
    npy: int
    nz: int
    dz: float                          # tip anchor z(iz) = p0.z - iz*dz  (far -> near)


@dataclass
class DfSpec:
    A: float = 1.0                     # peak-to-peak amplitude (Å)
    k0: float = 1800.0                 # cantilever stiffness (N/m)
    f0: float = 30300.0                # base frequency (Hz)


@dataclass
class Workload:
    name: str
    xyzq: np.ndarray                   # (N,4) float32: x,y,z (Å), q (e)
    types: np.ndarray                  # (N,) int32 index into elem_R/elem_e
    elem_R: np.ndarray
    elem_e: np.ndarray
    lattice: Lattice
    grid: Grid
    probe: Probe
    tip: Tip
    fire: Fire
    scan: Scan
    df: DfSpec
    r_min: float = 0.1
    Q_sweep: Optional[List[float]] = None      # config 2
    seed: int = 0

    # sizes in the metric's units -------------------------------------------------------------------
    @property
    def natoms(self) -> int:
        return int(self.xyzq.shape[0])

    @property
    def nimages(self) -> int:
        na, nb, nc = self.lattice.nimg
        return (2 * na + 1) * (2 * nb + 1) * (2 * nc + 1)

    @property
    def npoints(self) -> int:
        nx, ny, nz = self.grid.n
        return nx * ny * nz

    @property
    def pairs(self) -> int:
        return self.natoms * self.nimages * self.npoints

    @property
    def pixel_steps(self) -> int:
        return self.scan.npx * self.scan.npy * self.scan.nz

    @property
    def n_df(self) -> int:
        return int(round(self.df.A / self.scan.dz))


def _f32(x):
    """Round to FP32 and keep as float32 array."""
    return np.asarray(x, dtype=np.float64).astype(np.float32)


def _ortho_grid(origin, h, n, periodic):
    return Grid(origin=np.asarray(origin, dtype=np.float64), step=np.diag([h, h, h]).astype(np.float64),
                n=tuple(int(v) for v in n), periodic=tuple(int(v) for v in periodic))


def _ortho_lattice(L, nimg):
    return Lattice(a=np.array([L[0], 0, 0.0]), b=np.array([0, L[1], 0.0]), c=np.array([0, 0, L[2]]),
                   nimg=tuple(int(v) for v in nimg))


def _default_probe(Q=-0.05):
    return Probe(R=float(ELEM_R[T_O]), e=float(ELEM_E[T_O]), Q=float(Q))


def _default_tip(k_xy_Nm=0.25):
    k = k_xy_Nm * EVA2_PER_NM
    return Tip(k_lat=(k, k), k_rad=30.0 * EVA2_PER_NM, d0=(0.0, 0.0, -4.0))


def _neutral_charges(rng, n, sigma):
    q = rng.normal(0.0, sigma, n)
    return q - q.mean()


def _honeycomb_sites(centre, bond, nsites):
    """The `nsites` honeycomb-lattice sites nearest `centre`, sorted by distance (ties by index)."""
    a = bond * np.sqrt(3.0)
    a1 = np.array([a, 0.0])
    a2 = np.array([a / 2, a * np.sqrt(3.0) / 2])
    basis = [np.array([0.0, 0.0]), np.array([0.0, bond])]
    m = int(np.ceil(np.sqrt(nsites))) + 6
    pts = []
    for i in range(-m, m + 1):
        for j in range(-m, m + 1):
            for bvec in basis:
                pts.append(i * a1 + j * a2 + bvec)
    pts = np.array(pts)
    pts = pts - np.array([0.0, bond / 2])            # centre of a bond at the origin
    r = np.hypot(pts[:, 0], pts[:, 1])
    order = np.lexsort((np.arange(len(r)), np.round(r, 9)))
    sel = pts[order[:nsites]]
    return sel + np.asarray(centre)[None, :]


def _planar_molecule(rng, centre_xy, sigma_q):
    """Config-1 molecule: 60 honeycomb sites, rim 20 = H, others shuffled 30 C / 6 N / 4 O."""
    sites = _honeycomb_sites(centre_xy, 1.4, 60)      # sorted by distance: last 20 = outermost
    xy = sites + rng.normal(0.0, 0.05, sites.shape)
    inner = np.array([T_C] * 30 + [T_N] * 6 + [T_O] * 4, dtype=np.int32)
    rng.shuffle(inner)
    types = np.concatenate([inner, np.full(20, T_H, dtype=np.int32)])
    q = _neutral_charges(rng, 60, sigma_q)
    xyzq = np.c_[xy, np.zeros(60), q]
    return xyzq, types


def config0(seed: int = 1000) -> Workload:
    rng = np.random.default_rng(seed)
    n = 10
    types = rng.integers(0, 4, n).astype(np.int32)
    x = rng.uniform(3.0, 9.0, n)
    y = rng.uniform(3.0, 9.0, n)
    z = rng.uniform(-0.3, 0.3, n)
    q = _neutral_charges(rng, n, 0.2)
    return Workload(
        name="cfg0_tiny", xyzq=_f32(np.c_[x, y, z, q]), types=types, elem_R=ELEM_R.copy(), elem_e=ELEM_E.copy(),
        lattice=_ortho_lattice((12.0, 12.0, 8.0), (0, 0, 0)),
        grid=_ortho_grid((0.0, 0.0, 1.3), 0.2, (60, 60, 40), (0, 0, 0)),
        probe=_default_probe(), tip=_default_tip(), fire=Fire(),
        scan=Scan(p0=np.array([3.0, 3.0, 10.0]), dx=np.array([0.2, 0, 0.0]), dy=np.array([0, 0.2, 0.0]),
                  npx=30, npy=30, nz=40, dz=0.1),
        df=DfSpec(), seed=seed)


def config1(seed: int = 2000) -> Workload:
    rng = np.random.default_rng(seed)
    xyzq, types = _planar_molecule(rng, (10.0, 10.0), 0.15)
    return Workload(
        name="cfg1_planar60", xyzq=_f32(xyzq), types=types, elem_R=ELEM_R.copy(), elem_e=ELEM_E.copy(),
        lattice=_ortho_lattice((20.0, 20.0, 10.0), (0, 0, 0)),
        grid=_ortho_grid((0.0, 0.0, 1.0), 0.1, (200, 200, 100), (0, 0, 0)),
        probe=_default_probe(), tip=_default_tip(), fire=Fire(),
        scan=Scan(p0=np.array([2.5, 2.5, 10.0]), dx=np.array([0.1, 0, 0.0]), dy=np.array([0, 0.1, 0.0]),
                  npx=150, npy=150, nz=40, dz=0.1),
        df=DfSpec(), seed=seed)


def _slab():
    """5 layers x (10 x 10) atoms, in-layer spacing 2.5 Å, alternate rows offset 1.25 Å, ABCAB stacking,
    interlayer 2.2 Å, top layer z = -3.0.  No RNG."""
    shifts = {"A": (0.0, 0.0), "B": (1.25, 0.8333333333333334), "C": (2.5 * 0.25, 1.6666666666666667)}
    out = []
    for layer, tag in enumerate("ABCAB"):            # layer 0 = top
        sx, sy = shifts[tag]
        z = -3.0 - 2.2 * layer
        for j in range(10):
            for i in range(10):
                x = (i * 2.5 + (1.25 if j % 2 else 0.0) + sx) % 25.0
                y = (j * 2.5 + sy) % 25.0
                out.append((x, y, z, 0.0))
    return np.array(out), np.full(len(out), T_X, dtype=np.int32)


def config2(seed: int = 3000) -> Workload:
    rng = np.random.default_rng(seed)
    mol, mtypes = _planar_molecule(rng, (12.5, 12.5), 0.15)
    slab, stypes = _slab()
    return Workload(
        name="cfg2_on_slab", xyzq=_f32(np.r_[mol, slab]), types=np.r_[mtypes, stypes].astype(np.int32),
        elem_R=ELEM_R.copy(), elem_e=ELEM_E.copy(),
        lattice=_ortho_lattice((25.0, 25.0, 12.0), (1, 1, 0)),
        grid=_ortho_grid((0.0, 0.0, 1.0), 0.1, (250, 250, 120), (1, 1, 0)),
        probe=_default_probe(Q=-0.1), tip=_default_tip(), fire=Fire(),
        scan=Scan(p0=np.array([2.5, 2.5, 10.0]), dx=np.array([0.1, 0, 0.0]), dy=np.array([0, 0.1, 0.0]),
                  npx=200, npy=200, nz=40, dz=0.1),
        df=DfSpec(), Q_sweep=[-0.1, 0.0, 0.1], seed=seed)


def config3_molecule(index: int, seed: int = 4000) -> Workload:
    rng = np.random.default_rng(seed + index)
    n = int(rng.integers(20, 51))
    sites = _honeycomb_sites((8.0, 8.0), 1.4, n)
    xy = sites + rng.normal(0.0, 0.05, sites.shape)
    z = rng.uniform(-1.0, 1.0, n)
    types = rng.choice(np.array([T_C, T_H, T_N, T_O], dtype=np.int32), size=n, p=[0.50, 0.33, 0.10, 0.07])
    q = _neutral_charges(rng, n, 0.2)
    k_xy = float(rng.uniform(0.15, 0.35))
    xyzq = _f32(np.c_[xy, z, q])
    z_top = float(xyzq[:, 2].max())
    z_top = float(np.float32(z_top))
    width = 127 * 0.1
    x0 = (16.0 - width) / 2
    return Workload(
        name=f"cfg3_mol{index:02d}", xyzq=xyzq, types=types.astype(np.int32), elem_R=ELEM_R.copy(),
        elem_e=ELEM_E.copy(),
        lattice=_ortho_lattice((16.0, 16.0, 8.0), (0, 0, 0)),
        grid=_ortho_grid((0.0, 0.0, z_top + 1.0), 0.125, (128, 128, 64), (0, 0, 0)),
        probe=_default_probe(), tip=_default_tip(k_xy), fire=Fire(),
        scan=Scan(p0=np.array([x0, x0, z_top + 8.0]), dx=np.array([0.1, 0, 0.0]), dy=np.array([0, 0.1, 0.0]),
                  npx=128, npy=128, nz=20, dz=0.1),
        df=DfSpec(), seed=seed + index)


def config3(nmol: int = 64, seed: int = 4000) -> List[Workload]:
    return [config3_molecule(i, seed) for i in range(nmol)]


def config4(seed: int = 5000) -> Workload:
    rng = np.random.default_rng(seed)
    nxl, nyl, nzl = 18, 18, 16
    a_xy = 40.0 / 18.0
    a_z = 2.025
    ii, jj, kk = np.meshgrid(np.arange(nxl), np.arange(nyl), np.arange(nzl), indexing="ij")
    pos = np.c_[(ii.ravel() + 0.5) * a_xy, (jj.ravel() + 0.5) * a_xy, -0.4 - kk.ravel() * a_z]
    keep = np.ones(len(pos), dtype=bool)
    keep[rng.choice(len(pos), size=len(pos) - 5000, replace=False)] = False
    pos = pos[keep]
    jit = rng.uniform(-0.4, 0.4, pos.shape)
    pos = pos + jit
    pos[:, 2] = np.minimum(pos[:, 2], 0.0)
    n = len(pos)
    types = rng.choice(np.array([T_C, T_H, T_N, T_O], dtype=np.int32), size=n, p=[0.50, 0.33, 0.10, 0.07])
    q = _neutral_charges(rng, n, 0.15)
    return Workload(
        name="cfg4_large", xyzq=_f32(np.c_[pos, q]), types=types.astype(np.int32), elem_R=ELEM_R.copy(),
        elem_e=ELEM_E.copy(),
        lattice=_ortho_lattice((40.0, 40.0, 10.0), (1, 1, 0)),
        grid=_ortho_grid((0.0, 0.0, 1.0), 0.05, (800, 800, 200), (1, 1, 0)),
        probe=_default_probe(), tip=_default_tip(), fire=Fire(),
        scan=Scan(p0=np.array([10.0, 10.0, 10.0]), dx=np.array([0.05, 0, 0.0]), dy=np.array([0, 0.05, 0.0]),
                  npx=400, npy=400, nz=80, dz=0.05),
        df=DfSpec(), seed=seed)


def get(cfg: int, **kw):
    """Workload for BASELINE.json `configs[cfg]` (cfg 3 returns a list of 64 molecules)."""
    return {0: config0, 1: config1, 2: config2, 3: config3, 4: config4}[int(cfg)](**kw)


def with_probe_charge(w: Workload, Q: float) -> Workload:
    return replace(w, probe=Probe(R=w.probe.R, e=w.probe.e, Q=float(Q)))


def shrink(w: Workload, grid_n=None, scan_np=None, scan_nz=None) -> Workload:
    """Same system on a sub-grid / sub-scan (same origin and spacing) — used for parity cases the oracle
    can finish in seconds.  Non-periodic bookkeeping only; callers must not shrink periodic axes."""
    g, s = w.grid, w.scan
    if grid_n is not None:
        g = replace(g, n=tuple(int(v) for v in grid_n))
    if scan_np is not None or scan_nz is not None:
        s = replace(s, npx=int(scan_np[0]) if scan_np else s.npx, npy=int(scan_np[1]) if scan_np else s.npy,
                    nz=int(scan_nz) if scan_nz else s.nz)
    return replace(w, grid=g, scan=s)


def sample_indices(n_total: int, n_sample: int, seed: int) -> np.ndarray:
    """Seeded sorted sample of flat indices (grid points or pixels) for sampled parity at full size."""
    rng = np.random.default_rng(seed)
    if n_sample >= n_total:
        return np.arange(n_total, dtype=np.int64)
    return np.sort(rng.choice(n_total, size=n_sample, replace=False).astype(np.int64))
