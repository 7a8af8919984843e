"""ctypes binding + build step for the FP64 CPU oracle (oracle/ppfm_oracle.c).

TEST INFRASTRUCTURE, NOT PRODUCT CODE: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
`--impl reference` legs may import this module.  It imports nothing from the CUDA path; the only thing it
accepts from the package is a `workloads.Workload` object (plain input data).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ppfm_oracle.c")
_LIB = os.path.join(_HERE, "libppfm_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp the oracle into oracle/libppfm_oracle.so (rebuilt when the source is newer)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-fopenmp", "-D_GNU_SOURCE", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.oracle_num_threads.restype = C.c_int
    return _lib


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def _d(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def _p(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None else None


def _cell(lat):
    return _d(np.stack([lat.a, lat.b, lat.c]))


def forcefield(w, idx: Optional[np.ndarray] = None, Q: Optional[float] = None) -> np.ndarray:
    """O1-O3.  Full grid -> (nz, ny, nx, 4) float64; with idx (flat indices) -> (len(idx), 4)."""
    xyzq = _d(w.xyzq)
    types = _i(w.types)
    R, e = _d(w.elem_R), _d(w.elem_e)
    cell, nimg = _cell(w.lattice), _i(w.lattice.nimg)
    origin, step, n = _d(w.grid.origin), _d(w.grid.step), _i(w.grid.n)
    nx, ny, nz = w.grid.n
    if idx is None:
        out = np.empty((nz, ny, nx, 4), dtype=np.float64)
        nidx, pidx = 0, None
    else:
        idx = np.ascontiguousarray(idx, dtype=np.int64)
        out = np.empty((len(idx), 4), dtype=np.float64)
        nidx, pidx = len(idx), idx
    rc = lib().oracle_forcefield(C.c_int(len(types)), _p(xyzq), _p(types), C.c_int(len(R)), _p(R), _p(e), _p(cell),
                                 _p(nimg), C.c_double(w.probe.R), C.c_double(w.probe.e),
                                 C.c_double(w.probe.Q if Q is None else Q), _p(origin), _p(step), _p(n),
                                 C.c_double(w.r_min), C.c_int64(nidx), _p(pidx), _p(out))
    if rc:
        raise ValueError(f"oracle_forcefield rc={rc}")
    return out


def ff_at_points(w, pts, Q: Optional[float] = None, nimg=None, r_min=None) -> np.ndarray:
    xyzq = _d(w.xyzq)
    types = _i(w.types)
    R, e = _d(w.elem_R), _d(w.elem_e)
    cell = _cell(w.lattice)
    nimg = _i(w.lattice.nimg if nimg is None else nimg)
    pts = _d(pts).reshape(-1, 3)
    out = np.empty((len(pts), 4), dtype=np.float64)
    rc = lib().oracle_ff_at_points(C.c_int(len(types)), _p(xyzq), _p(types), C.c_int(len(R)), _p(R), _p(e),
                                   _p(cell), _p(nimg), C.c_double(w.probe.R), C.c_double(w.probe.e),
                                   C.c_double(w.probe.Q if Q is None else Q),
                                   C.c_double(w.r_min if r_min is None else r_min), C.c_int64(len(pts)), _p(pts),
                                   _p(out))
    if rc:
        raise ValueError(f"oracle_ff_at_points rc={rc}")
    return out


def _ff_args(ff, grid):
    ff = np.ascontiguousarray(ff)
    if ff.dtype == np.float32:
        is32 = 1
    elif ff.dtype == np.float64:
        is32 = 0
    else:
        raise TypeError("ff must be float32 or float64")
    nx, ny, nz = grid.n
    if ff.shape == (nz, ny, nx):          # O13: energy-only grid -> tri-cubic interpolation of the potential
        is32 |= 2
    else:
        assert ff.shape == (nz, ny, nx, 4), (ff.shape, grid.n)
    return ff, is32, _d(grid.origin), _d(grid.step), _i(grid.n), _i(grid.periodic)


def interp(ff, grid, pts) -> np.ndarray:
    ff, is32, origin, step, n, per = _ff_args(ff, grid)
    pts = _d(pts).reshape(-1, 3)
    out = np.empty((len(pts), 3), dtype=np.float64)
    rc = lib().oracle_interp(_p(ff), C.c_int(is32), _p(origin), _p(step), _p(n), _p(per), C.c_int64(len(pts)),
                             _p(pts), _p(out))
    if rc:
        raise ValueError(f"oracle_interp rc={rc}")
    return out


def total_force(ff, grid, tip, rtip, rpp) -> np.ndarray:
    ff, is32, origin, step, n, per = _ff_args(ff, grid)
    F = np.empty(3)
    rc = lib().oracle_total_force(_p(ff), C.c_int(is32), _p(origin), _p(step), _p(n), _p(per), _p(_d(tip.k_lat)),
                                  C.c_double(tip.k_rad), _p(_d(tip.d0)), _p(_d(rtip)), _p(_d(rpp)), _p(F))
    if rc:
        raise ValueError(f"oracle_total_force rc={rc}")
    return F


def hessian(ff, grid, tip, rtip, rpp):
    ff, is32, origin, step, n, per = _ff_args(ff, grid)
    H = np.empty((3, 3))
    w = np.empty(3)
    rc = lib().oracle_hessian(_p(ff), C.c_int(is32), _p(origin), _p(step), _p(n), _p(per), _p(_d(tip.k_lat)),
                              C.c_double(tip.k_rad), _p(_d(tip.d0)), _p(_d(rtip)), _p(_d(rpp)), _p(H), _p(w))
    if rc:
        raise ValueError(f"oracle_hessian rc={rc}")
    return H, w


def stiffness(ff, grid, tip, rtips, rpps) -> np.ndarray:
    """IETS stiffness map: eigenvalues (ascending, eV/Å^2) of O10's Hessian at each of the
    (r_TIP, r_PP) pairs; rtips, rpps (..., 3) -> (..., 3)."""
    ff, is32, origin, step, n, per = _ff_args(ff, grid)
    rt = np.ascontiguousarray(np.asarray(rtips, dtype=np.float64).reshape(-1, 3))
    rp = np.ascontiguousarray(np.asarray(rpps, dtype=np.float64).reshape(-1, 3))
    assert rt.shape == rp.shape
    out = np.empty_like(rp)
    rc = lib().oracle_stiffness(_p(ff), C.c_int(is32), _p(origin), _p(step), _p(n), _p(per), _p(_d(tip.k_lat)),
                                C.c_double(tip.k_rad), _p(_d(tip.d0)), C.c_int64(rt.shape[0]), _p(rt), _p(rp), _p(out))
    if rc:
        raise ValueError(f"oracle_stiffness rc={rc}")
    return out.reshape(np.asarray(rpps).shape)


def tip_positions(scan) -> np.ndarray:
    """Tip anchors of a scan, (nz, npy*npx, 3): p0 + ix dx + iy dy - (0, 0, iz dz)."""
    iz, iy, ix = np.meshgrid(np.arange(scan.nz), np.arange(scan.npy), np.arange(scan.npx), indexing="ij")
    r = (np.asarray(scan.p0, float)[None, None, None, :] + ix[..., None] * np.asarray(scan.dx, float) +
         iy[..., None] * np.asarray(scan.dy, float))
    r[..., 2] -= iz * scan.dz
    return r.reshape(scan.nz, scan.npy * scan.npx, 3)


def tip_density(grid, sigma: float, q_s: float, p_z: float, Q_zz: float) -> np.ndarray:
    """O12: Gaussian-multipole tip charge density and its analytic gradient at the grid nodes (minimum image by
    index) -> (4, nz, ny, nx): rho, d rho/dx, d rho/dy, d rho/dz."""
    step = np.ascontiguousarray(np.asarray(grid.step, dtype=np.float64).reshape(9))
    n = _i(grid.n)
    out = np.empty((4, int(grid.n[2]), int(grid.n[1]), int(grid.n[0])))
    rc = lib().oracle_tip_density(_p(step), _p(n), C.c_double(sigma), C.c_double(q_s), C.c_double(p_z),
                                  C.c_double(Q_zz), _p(out))
    if rc:
        raise ValueError(f"oracle_tip_density rc={rc}")
    return out


def fft_forcefield(V, grid, sigma: float, q_s: float, p_z: float, Q_zz: float) -> np.ndarray:
    """O12 (Eq.7; reading S21): E_el(R) = sum_r rho(r) V(r + R) dV and F_el = sum_r grad rho(r)
    V(r + R) dV on the periodic grid, by direct O(N^2) summation.  V (nz, ny, nx) in eV/e -> (nz, ny, nx, 4) =
    (Fx, Fy, Fz, E).  Small grids only."""
    V = np.ascontiguousarray(np.asarray(V, dtype=np.float64))
    rho4 = tip_density(grid, sigma, q_s, p_z, Q_zz)
    assert V.shape == rho4.shape[1:]
    dV = abs(float(np.linalg.det(np.asarray(grid.step, dtype=np.float64))))
    n = _i(grid.n)
    out = np.empty(V.shape + (4,))
    tmp = np.empty(V.shape)
    for c, lane in ((0, 3), (1, 0), (2, 1), (3, 2)):
        rc = lib().oracle_crosscorr(_p(n), _p(np.ascontiguousarray(rho4[c])), _p(V), C.c_double(dV), _p(tmp))
        if rc:
            raise ValueError(f"oracle_crosscorr rc={rc}")
        out[..., lane] = tmp
    return out


def fft_forcefield_at(V, grid, sigma: float, q_s: float, p_z: float, Q_zz: float, ijk) -> np.ndarray:
    """O12 at selected output nodes ijk (npts, 3) = (I, J, K) -> (npts, 4) = (Fx, Fy, Fz, E); O(N) per sample."""
    V = np.ascontiguousarray(np.asarray(V, dtype=np.float64))
    rho4 = tip_density(grid, sigma, q_s, p_z, Q_zz)
    dV = abs(float(np.linalg.det(np.asarray(grid.step, dtype=np.float64))))
    ijk = np.ascontiguousarray(ijk, dtype=np.int32)
    out = np.empty((ijk.shape[0], 4))
    tmp = np.empty(ijk.shape[0])
    for c, lane in ((0, 3), (1, 0), (2, 1), (3, 2)):
        rc = lib().oracle_crosscorr_at(_p(_i(grid.n)), _p(np.ascontiguousarray(rho4[c])), _p(V), C.c_double(dV),
                                       C.c_int64(ijk.shape[0]), _p(ijk), _p(tmp))
        if rc:
            raise ValueError(f"oracle_crosscorr_at rc={rc}")
        out[:, lane] = tmp
    return out


def pauli_forcefield(rho_S, grid, sigma: float, q: float, A: float, beta: float) -> np.ndarray:
    """O14 (Eq.8; reading S23): E(R) = A sum_r [rho_PP(r) rho_S(r + R)]^beta dV and F = -grad_R E on
    the periodic grid by direct O(N^2) sums; rho_PP = q g_sigma.  rho_S (nz, ny, nx) -> (nz, ny, nx, 4)."""
    S = np.ascontiguousarray(np.maximum(np.asarray(rho_S, dtype=np.float64), 0.0) ** beta)
    step = np.ascontiguousarray(np.asarray(grid.step, dtype=np.float64).reshape(9))
    n = _i(grid.n)
    T4 = np.empty((4,) + S.shape)
    rc = lib().oracle_pauli_tip(_p(step), _p(n), C.c_double(sigma), C.c_double(q), C.c_double(beta), _p(T4))
    if rc:
        raise ValueError(f"oracle_pauli_tip rc={rc}")
    dV = abs(float(np.linalg.det(np.asarray(grid.step, dtype=np.float64))))
    out = np.empty(S.shape + (4,))
    tmp = np.empty(S.shape)
    for c, lane in ((0, 3), (1, 0), (2, 1), (3, 2)):
        rc = lib().oracle_crosscorr(_p(n), _p(np.ascontiguousarray(T4[c])), _p(S), C.c_double(dV * A), _p(tmp))
        if rc:
            raise ValueError(f"oracle_crosscorr rc={rc}")
        out[..., lane] = tmp
    return out


def relax_scan(ff, grid, tip, fire, scan, pix: Optional[np.ndarray] = None, traj: bool = True):
    """O4-O8 (+O10).  Returns dict: pos_fz (nz, npix, 4), iters (nz, npix) [-1 = not converged],
    lam_min (nz, npix), clamped (nz, npix), lam_traj (nz, npix; smallest Hessian eigenvalue along the step's FIRE
    path, reading S17; None when traj=False).  Without `pix` npix = npy*npx in row-major (iy, ix) order."""
    ff, is32, origin, step, n, per = _ff_args(ff, grid)
    if pix is None:
        npix, ppix = scan.npx * scan.npy, None
    else:
        pix = np.ascontiguousarray(pix, dtype=np.int64)
        npix, ppix = len(pix), pix
    pos = np.empty((scan.nz, npix, 4))
    iters = np.empty((scan.nz, npix), dtype=np.int32)
    lam = np.empty((scan.nz, npix))
    cl = np.empty((scan.nz, npix), dtype=np.int32)
    lt = np.empty((scan.nz, npix)) if traj else None
    f = _d([fire.dt, fire.dt_max, fire.finc, fire.fdec, fire.alpha0, fire.falpha, fire.f_conv])
    rc = lib().oracle_relax_scan(_p(ff), C.c_int(is32), _p(origin), _p(step), _p(n), _p(per), _p(_d(tip.k_lat)),
                                 C.c_double(tip.k_rad), _p(_d(tip.d0)), _p(f), C.c_int(fire.n_min),
                                 C.c_int(fire.max_iter), _p(_d(scan.p0)), _p(_d(scan.dx)), _p(_d(scan.dy)),
                                 C.c_int(scan.npx), C.c_int(scan.npy), C.c_int(scan.nz), C.c_double(scan.dz),
                                 C.c_int64(npix if pix is not None else 0), _p(ppix), _p(pos), _p(iters), _p(lam),
                                 _p(cl), _p(lt))
    if rc:
        raise ValueError(f"oracle_relax_scan rc={rc}")
    return {"pos_fz": pos, "iters": iters, "lam_min": lam, "clamped": cl, "lam_traj": lt}


def relax_scan_atoms(w, pix: Optional[np.ndarray] = None, traj: bool = True, Q: Optional[float] = None,
                     tip=None, scan=None, grid=None):
    """O3-O8 (+O10) end to end WITHOUT a stored grid: the same scan as relax_scan(forcefield(w), ...), every grid node
    the interpolation touches being evaluated on demand from the atoms (ff_at_point, the value oracle_forcefield would
    store) and memoised per pixel.  Affordable on sampled pixels of grids whose full FP64 evaluation
    takes hours.  Returns relax_scan's dict plus `nodes` (npix,) = grid nodes evaluated per pixel."""
    tip = w.tip if tip is None else tip
    scan = w.scan if scan is None else scan
    grid = w.grid if grid is None else grid
    xyzq, types = _d(w.xyzq), _i(w.types)
    R, e = _d(w.elem_R), _d(w.elem_e)
    cell, nimg = _cell(w.lattice), _i(w.lattice.nimg)
    origin, step, n, per = _d(grid.origin), _d(grid.step), _i(grid.n), _i(grid.periodic)
    if pix is None:
        npix, ppix = scan.npx * scan.npy, None
    else:
        pix = np.ascontiguousarray(pix, dtype=np.int64)
        npix, ppix = len(pix), pix
    pos = np.empty((scan.nz, npix, 4))
    iters = np.empty((scan.nz, npix), dtype=np.int32)
    lam = np.empty((scan.nz, npix))
    cl = np.empty((scan.nz, npix), dtype=np.int32)
    lt = np.empty((scan.nz, npix)) if traj else None
    nodes = np.zeros(npix, dtype=np.int64)
    fire = w.fire
    f = _d([fire.dt, fire.dt_max, fire.finc, fire.fdec, fire.alpha0, fire.falpha, fire.f_conv])
    rc = lib().oracle_relax_scan_atoms(
        C.c_int(len(types)), _p(xyzq), _p(types), C.c_int(len(R)), _p(R), _p(e), _p(cell), _p(nimg),
        C.c_double(w.probe.R), C.c_double(w.probe.e), C.c_double(w.probe.Q if Q is None else Q), C.c_double(w.r_min),
        _p(origin), _p(step), _p(n), _p(per), _p(_d(tip.k_lat)), C.c_double(tip.k_rad), _p(_d(tip.d0)), _p(f),
        C.c_int(fire.n_min), C.c_int(fire.max_iter), _p(_d(scan.p0)), _p(_d(scan.dx)), _p(_d(scan.dy)),
        C.c_int(scan.npx), C.c_int(scan.npy), C.c_int(scan.nz), C.c_double(scan.dz),
        C.c_int64(npix if pix is not None else 0), _p(ppix), _p(pos), _p(iters), _p(lam), _p(cl), _p(lt), _p(nodes))
    if rc:
        raise ValueError(f"oracle_relax_scan_atoms rc={rc}")
    return {"pos_fz": pos, "iters": iters, "lam_min": lam, "clamped": cl, "lam_traj": lt, "nodes": nodes}


def df_weights(n: int, dz: float) -> np.ndarray:
    W = np.empty(n + 1)
    rc = lib().oracle_df_weights(C.c_int(n), C.c_double(dz), _p(W))
    if rc:
        raise ValueError(f"oracle_df_weights rc={rc}")
    return W


def df(fz, dz: float, A: float, k0: float, f0: float) -> np.ndarray:
    """O9.  fz (nz, npix) -> df (nz - n, npix), n = round(A/dz)."""
    fz = _d(fz)
    nz, npix = fz.shape
    n = int(round(A / dz))
    out = np.empty((max(nz - n, 0), npix))
    rc = lib().oracle_df(_p(fz), C.c_int64(npix), C.c_int(nz), C.c_double(dz), C.c_double(A), C.c_double(k0),
                         C.c_double(f0), _p(out))
    if rc:
        raise ValueError(f"oracle_df rc={rc}")
    return out


def near_unstable(lam_min: np.ndarray, thresh: float = 1e-3, lam_traj: Optional[np.ndarray] = None) -> np.ndarray:
    """O10 flag over (nz, npix): smallest Hessian eigenvalue < thresh at the relaxed point of this z-step or the
    previous one, or (reading S17, when lam_traj is given) anywhere along the FIRE path of this or the previous step."""
    f = lam_min < thresh
    if lam_traj is not None:
        f = f | (lam_traj < thresh)
    out = f.copy()
    out[1:] |= f[:-1]
    return out


def flags(res: dict, thresh: float = 1e-3) -> np.ndarray:
    """near_unstable over a relax_scan result, plus the not-converged samples."""
    return near_unstable(res["lam_min"], thresh, res.get("lam_traj")) | (res["iters"] < 0)
