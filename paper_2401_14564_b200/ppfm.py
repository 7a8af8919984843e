"""Thin Python binding over the C-ABI library libppfm.so (include/ppfm.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI; torch is used for device memory and streams.
There is no CPU fallback: if libppfm.so is missing or no CUDA device is present the calls raise.
Function names mirror the C entry points (forcefield, relax_scan, df, ..., scan_host).
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# PPFM_LIBRARY selects another build of the same ABI (the checked build libppfm_chk.so, see include/ppfm_bench.h)
LIB_PATH = os.environ.get("PPFM_LIBRARY") or os.path.join(_HERE, "libppfm.so")
_lib = None


class PpfmError(RuntimeError):
    pass


# ---- ctypes mirrors of the structs in include/ppfm.h -------------------------------------------------------
class Lattice(C.Structure):
    _fields_ = [("a", C.c_double * 3), ("b", C.c_double * 3), ("c", C.c_double * 3), ("nimg", C.c_int32 * 3)]


class Grid(C.Structure):
    _fields_ = [("origin", C.c_double * 3), ("step", (C.c_double * 3) * 3), ("n", C.c_int32 * 3),
                ("periodic", C.c_int32 * 3)]


class Probe(C.Structure):
    _fields_ = [("R", C.c_double), ("e", C.c_double), ("Q", C.c_double)]


class Tip(C.Structure):
    _fields_ = [("k_lat", C.c_double * 2), ("k_rad", C.c_double), ("d0", C.c_double * 3)]


class Fire(C.Structure):
    _fields_ = [("dt", C.c_double), ("dt_max", C.c_double), ("finc", C.c_double), ("fdec", C.c_double),
                ("alpha0", C.c_double), ("falpha", C.c_double), ("n_min", C.c_int32), ("max_iter", C.c_int32),
                ("f_conv", C.c_double)]


class Scan(C.Structure):
    _fields_ = [("p0", C.c_double * 3), ("dx", C.c_double * 3), ("dy", C.c_double * 3), ("npx", C.c_int32),
                ("npy", C.c_int32), ("nz", C.c_int32), ("dz", C.c_double)]


class TipDensity(C.Structure):
    _fields_ = [("sigma", C.c_double), ("q_s", C.c_double), ("p_z", C.c_double), ("Q_zz", C.c_double)]


class Stats(C.Structure):
    _fields_ = [("total_iters", C.c_uint64), ("n_not_converged", C.c_uint64), ("n_clamped", C.c_uint64),
                ("max_iters", C.c_uint32), ("_pad", C.c_uint32), ("warp_iters", C.c_uint64),
                ("cell_gathers", C.c_uint64), ("warp_gathers", C.c_uint64)]


# the product ABI (include/ppfm.h); the measurement interface of include/ppfm_bench.h is bound in ppfm_bench.py
EXPORTS = ["ppfm_version", "ppfm_strerror", "ppfm_fire_default", "ppfm_Nm_to_eVA2", "ppfm_forcefield",
           "ppfm_forcefield_noalloc", "ppfm_forcefield_energy",
           "ppfm_forcefield_split", "ppfm_combine", "ppfm_forcefield_batch", "ppfm_forcefield_fft",
           "ppfm_forcefield_pauli", "ppfm_relax_scan", "ppfm_relax_scan_batch", "ppfm_relax_scan_sweep", "ppfm_relax_scan_stiffness",
           "ppfm_relax_scan_stiffness_batch", "ppfm_relax_scan_tricubic",
           "ppfm_relax_scan_tricubic_batch", "ppfm_energy_grid", "ppfm_stiffness", "ppfm_stiffness_batch", "ppfm_df",
           "ppfm_df_batch", "ppfm_df_weights", "ppfm_scan_host", "ppfm_scan_host_batch", "ppfm_scan_host_sweep",
           "ppfm_release_scratch"]


HEADER_VERSION = 200            # PPFM_VERSION of the include/ppfm.h this binding mirrors


def lib():
    """Load libppfm.so (fails loudly when it has not been built: `python -m paper_2401_14564_b200.build`)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise PpfmError(f"{LIB_PATH} not found — build it with `python -m paper_2401_14564_b200.build`; "
                            "there is no CPU fallback")
        L = C.CDLL(LIB_PATH)
        L.ppfm_version.restype = C.c_int
        if int(L.ppfm_version()) != HEADER_VERSION:      # argument lists differ between ABI versions: never guess
            raise PpfmError(f"{LIB_PATH} is ABI version {int(L.ppfm_version())}, this binding was written against "
                            f"include/ppfm.h version {HEADER_VERSION}; rebuild with `python -m paper_2401_14564_b200.build`")
        L.ppfm_strerror.restype = C.c_char_p
        L.ppfm_strerror.argtypes = [C.c_int]
        L.ppfm_Nm_to_eVA2.restype = C.c_double
        L.ppfm_Nm_to_eVA2.argtypes = [C.c_double]
        _lib = L
    return _lib


def _check(rc: int, what: str):
    if rc != 0:
        raise PpfmError(f"{what} failed: {rc} ({lib().ppfm_strerror(rc).decode()})")


def version() -> int:
    return int(lib().ppfm_version())


def release_scratch() -> None:
    _check(lib().ppfm_release_scratch(), "ppfm_release_scratch")


def Nm_to_eVA2(k: float) -> float:
    return float(lib().ppfm_Nm_to_eVA2(k))


def fire_default() -> Fire:
    f = Fire()
    lib().ppfm_fire_default(C.byref(f))
    return f


# ---- marshalling from workloads.* dataclasses (or anything with the same attributes) ------------------------
def _vec(ctype, vals):
    return ctype(*[float(v) for v in vals])


def c_lattice(l) -> Lattice:
    if isinstance(l, Lattice):
        return l
    return Lattice(_vec(C.c_double * 3, l.a), _vec(C.c_double * 3, l.b), _vec(C.c_double * 3, l.c),
                   (C.c_int32 * 3)(*[int(v) for v in l.nimg]))


def c_grid(g) -> Grid:
    if isinstance(g, Grid):
        return g
    out = Grid()
    for a in range(3):
        out.origin[a] = float(g.origin[a])
        out.n[a] = int(g.n[a])
        out.periodic[a] = int(g.periodic[a])
        for c in range(3):
            out.step[a][c] = float(g.step[a][c])
    return out


def c_probe(p, Q: Optional[float] = None) -> Probe:
    if isinstance(p, Probe) and Q is None:
        return p
    return Probe(float(p.R), float(p.e), float(p.Q if Q is None else Q))


def c_tip(t) -> Tip:
    if isinstance(t, Tip):
        return t
    return Tip(_vec(C.c_double * 2, t.k_lat), float(t.k_rad), _vec(C.c_double * 3, t.d0))


def c_fire(f) -> Fire:
    if isinstance(f, Fire):
        return f
    return Fire(float(f.dt), float(f.dt_max), float(f.finc), float(f.fdec), float(f.alpha0), float(f.falpha),
                int(f.n_min), int(f.max_iter), float(f.f_conv))


def c_scan(s) -> Scan:
    if isinstance(s, Scan):
        return s
    return Scan(_vec(C.c_double * 3, s.p0), _vec(C.c_double * 3, s.dx), _vec(C.c_double * 3, s.dy), int(s.npx),
                int(s.npy), int(s.nz), float(s.dz))


def c_array(items, conv):
    """ctypes array of converted structs, e.g. c_array(grids, c_grid); a ready ctypes array passes through."""
    if isinstance(items, C.Array):
        return items
    cs = [conv(x) for x in items]
    return (type(cs[0]) * len(cs))(*cs)


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise PpfmError("no CUDA device: the ppfm hot path runs only on the GPU (no CPU fallback)")
    return torch


def _stream():
    return C.c_void_p(_torch().cuda.current_stream().cuda_stream)


def _dptr(t, dtype=None):
    if t is None:
        return C.c_void_p(0)
    torch = _torch()
    if not t.is_cuda or not t.is_contiguous():
        raise PpfmError("expected a contiguous CUDA tensor")
    if dtype is not None and t.dtype != dtype:
        raise PpfmError(f"expected dtype {dtype}, got {t.dtype}")
    return C.c_void_p(t.data_ptr())


def _darr(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(C.POINTER(C.c_double))


# ---- (1) force field ----------------------------------------------------------------------------------------
def new_ff_status(device="cuda"):
    """Device ppfm_ff_status (8 bytes) for the `status` argument of the force-field calls; read with read_ff_status."""
    torch = _torch()
    return torch.zeros(2, dtype=torch.int32, device=device)


def read_ff_status(status) -> dict:
    raw = status.cpu().numpy().view(np.uint32)
    return {"n_bad_type": int(raw[0]), "n_clamped": int(raw[1])}


def forcefield(xyzq, types, elem_R, elem_e, lattice, probe, grid, r_min=0.1, out=None, Q=None, status=None):
    """ppfm_forcefield: xyzq (N,4) float32 CUDA, types (N,) int32 CUDA -> (nz, ny, nx, 4) float32 CUDA."""
    torch = _torch()
    nx, ny, nz = (int(v) for v in grid.n)
    if out is None:
        out = torch.empty((nz, ny, nx, 4), dtype=torch.float32, device=xyzq.device)
    R, pR = _darr(elem_R)
    e, pe = _darr(elem_e)
    rc = lib().ppfm_forcefield(C.c_int32(xyzq.shape[0]), _dptr(xyzq, torch.float32), _dptr(types, torch.int32),
                               C.c_int32(len(R)), pR, pe, C.byref(c_lattice(lattice)), C.byref(c_probe(probe, Q)),
                               C.byref(c_grid(grid)), C.c_double(r_min), _dptr(out, torch.float32), _dptr(status),
                               _stream())
    _check(rc, "ppfm_forcefield")
    return out


NOALLOC_MAX_ATOMS = 16384       # PPFM_NOALLOC_MAX_ATOMS (include/ppfm.h)
ELIMIT = -4                     # PPFM_ELIMIT


def forcefield_noalloc(xyzq, types, elem_R, elem_e, lattice, probe, grid, out, r_min=0.1, Q=None, status=None):
    """ppfm_forcefield_noalloc: ppfm_forcefield for callers that must not allocate device memory once they are
    running (a process whose GPU memory was carved up at start-up, a real-time loop that cannot wait on an allocator
    or the driver, a host whose allocator hook forbids cudaMalloc* after initialisation).  Same kernels and the same
    bits as `forcefield`, but the library's scratch is a fixed 768 KiB array inside the library, so:

    * at most NOALLOC_MAX_ATOMS (16384) atoms — more raises PpfmError with PPFM_ELIMIT and nothing runs;
    * `out` is required (a (nz, ny, nx, 4) float32 CUDA tensor): this wrapper allocates nothing on the device either;
    * every call on a device shares that one array: calls that can overlap on the GPU (different streams) race —
      keep them on one stream or order them with events;
    * the first call on a device looks the array's address up (and may load the library's device code): make it at
      start-up, outside any stream capture.
    """
    torch = _torch()
    nx, ny, nz = (int(v) for v in grid.n)
    if out is None or out.numel() != nx * ny * nz * 4 or out.dtype != torch.float32 or not out.is_contiguous():
        raise PpfmError("forcefield_noalloc needs a contiguous float32 CUDA `out` of nz*ny*nx*4 elements")
    R, pR = _darr(elem_R)
    e, pe = _darr(elem_e)
    rc = lib().ppfm_forcefield_noalloc(C.c_int32(xyzq.shape[0]), _dptr(xyzq, torch.float32),
                                       _dptr(types, torch.int32), C.c_int32(len(R)), pR, pe,
                                       C.byref(c_lattice(lattice)), C.byref(c_probe(probe, Q)), C.byref(c_grid(grid)),
                                       C.c_double(r_min), _dptr(out, torch.float32), _dptr(status), _stream())
    _check(rc, "ppfm_forcefield_noalloc")
    return out


def forcefield_energy(xyzq, types, elem_R, elem_e, lattice, probe, grid, r_min=0.1, out=None, Q=None, status=None):
    """ppfm_forcefield_energy: the energy-only grid (nz, ny, nx) float32 CUDA for relax_scan_tricubic — a quarter of
    the float4 grid's memory, no force arithmetic, FP64 totals per point."""
    torch = _torch()
    nx, ny, nz = (int(v) for v in grid.n)
    if out is None:
        out = torch.empty((nz, ny, nx), dtype=torch.float32, device=xyzq.device)
    R, pR = _darr(elem_R)
    e, pe = _darr(elem_e)
    rc = lib().ppfm_forcefield_energy(C.c_int32(xyzq.shape[0]), _dptr(xyzq, torch.float32), _dptr(types, torch.int32),
                                      C.c_int32(len(R)), pR, pe, C.byref(c_lattice(lattice)),
                                      C.byref(c_probe(probe, Q)), C.byref(c_grid(grid)), C.c_double(r_min),
                                      _dptr(out, torch.float32), _dptr(status), _stream())
    _check(rc, "ppfm_forcefield_energy")
    return out


def forcefield_split(xyzq, types, elem_R, elem_e, lattice, probe, grid, r_min=0.1, out_lj=None, out_el=None,
                     status=None):
    torch = _torch()
    nx, ny, nz = (int(v) for v in grid.n)
    if out_lj is None:
        out_lj = torch.empty((nz, ny, nx, 4), dtype=torch.float32, device=xyzq.device)
    if out_el is None:
        out_el = torch.empty((nz, ny, nx, 4), dtype=torch.float32, device=xyzq.device)
    R, pR = _darr(elem_R)
    e, pe = _darr(elem_e)
    rc = lib().ppfm_forcefield_split(C.c_int32(xyzq.shape[0]), _dptr(xyzq, torch.float32),
                                     _dptr(types, torch.int32), C.c_int32(len(R)), pR, pe,
                                     C.byref(c_lattice(lattice)), C.byref(c_probe(probe)), C.byref(c_grid(grid)),
                                     C.c_double(r_min), _dptr(out_lj, torch.float32), _dptr(out_el, torch.float32),
                                     _dptr(status), _stream())
    _check(rc, "ppfm_forcefield_split")
    return out_lj, out_el


def combine(ff_lj, ff_el, Q: float, out=None):
    torch = _torch()
    if out is None:
        out = torch.empty_like(ff_lj)
    rc = lib().ppfm_combine(_dptr(ff_lj, torch.float32), _dptr(ff_el, torch.float32), C.c_double(Q),
                            C.c_int64(ff_lj.numel() // 4), _dptr(out, torch.float32), _stream())
    _check(rc, "ppfm_combine")
    return out


def forcefield_batch(atom_offset: Sequence[int], xyzq, types, elem_R, elem_e, lattices, probes, grids, r_min=0.1,
                     out=None, status=None):
    """ppfm_forcefield_batch: concatenated atoms, one launch; returns a flat (sum points, 4) float32 tensor."""
    torch = _torch()
    nsys = len(grids)
    off = atom_offset if isinstance(atom_offset, C.Array) else (C.c_int32 * (nsys + 1))(*[int(v) for v in atom_offset])
    lat, pr, gr = c_array(lattices, c_lattice), c_array(probes, c_probe), c_array(grids, c_grid)
    if out is None:
        npts = sum(int(g.n[0]) * int(g.n[1]) * int(g.n[2]) for g in gr)
        out = torch.empty((npts, 4), dtype=torch.float32, device=xyzq.device)
    R, pR = _darr(elem_R)
    e, pe = _darr(elem_e)
    rc = lib().ppfm_forcefield_batch(C.c_int32(nsys), off, _dptr(xyzq, torch.float32), _dptr(types, torch.int32),
                                     C.c_int32(len(R)), pR, pe, lat, pr, gr, C.c_double(r_min),
                                     _dptr(out, torch.float32), _dptr(status), _stream())
    _check(rc, "ppfm_forcefield_batch")
    return out


# ---- (1b) Eq.7 electrostatics of an extended tip density (cuFFT) -------------------------------------------------
def forcefield_fft(V, grid, sigma: float, q_s: float = 0.0, p_z: float = 0.0, Q_zz: float = 0.0, out=None):
    """ppfm_forcefield_fft: V (nz, ny, nx) float32 device tensor in eV/e -> (nz, ny, nx, 4) = (Fx, Fy, Fz, E_el)."""
    torch = _torch()
    nx, ny, nz = (int(v) for v in (grid.n if not isinstance(grid, Grid) else grid.n))
    if out is None:
        out = torch.empty((nz, ny, nx, 4), dtype=torch.float32, device=V.device)
    td = TipDensity(float(sigma), float(q_s), float(p_z), float(Q_zz))
    rc = lib().ppfm_forcefield_fft(_dptr(V, torch.float32), C.byref(c_grid(grid)), C.byref(td),
                                   _dptr(out, torch.float32), _stream())
    _check(rc, "ppfm_forcefield_fft")
    return out


def forcefield_pauli(rho_S, grid, sigma: float, q_tip: float, A: float, beta: float, out=None):
    """ppfm_forcefield_pauli (Eq.8): rho_S (nz, ny, nx) float32 device tensor -> (nz, ny, nx, 4) = (Fx, Fy, Fz, E)."""
    torch = _torch()
    nx, ny, nz = (int(v) for v in grid.n)
    if out is None:
        out = torch.empty((nz, ny, nx, 4), dtype=torch.float32, device=rho_S.device)
    rc = lib().ppfm_forcefield_pauli(_dptr(rho_S, torch.float32), C.byref(c_grid(grid)), C.c_double(sigma),
                                     C.c_double(q_tip), C.c_double(A), C.c_double(beta), _dptr(out, torch.float32),
                                     _stream())
    _check(rc, "ppfm_forcefield_pauli")
    return out


# ---- (2) relaxation scan --------------------------------------------------------------------------------------
def new_stats(device="cuda"):
    torch = _torch()
    return torch.zeros(7, dtype=torch.int64, device=device)      # 56 bytes = sizeof(ppfm_stats)


def read_stats(stats) -> dict:
    raw = stats.cpu().numpy().view(np.uint64)
    return {"total_iters": int(raw[0]), "n_not_converged": int(raw[1]), "n_clamped": int(raw[2]),
            "max_iters": int(raw[3] & np.uint64(0xFFFFFFFF)), "warp_iters": int(raw[4]), "cell_gathers": int(raw[5]),
            "warp_gathers": int(raw[6])}


def relax_scan(ff, grid, tip, fire, scan, pos_fz=None, iters=None, stats=None, want_iters=True):
    """ppfm_relax_scan -> (pos_fz (nz, npy, npx, 4) float32, iters (nz, npy, npx) int16-as-uint16 or None)."""
    torch = _torch()
    shape = (int(scan.nz), int(scan.npy), int(scan.npx))
    if pos_fz is None:
        pos_fz = torch.empty(shape + (4,), dtype=torch.float32, device=ff.device)
    if iters is None and want_iters:
        iters = torch.empty(shape, dtype=torch.int16, device=ff.device)
    rc = lib().ppfm_relax_scan(_dptr(ff, torch.float32), C.byref(c_grid(grid)), C.byref(c_tip(tip)),
                               C.byref(c_fire(fire)), C.byref(c_scan(scan)), _dptr(pos_fz, torch.float32),
                               _dptr(iters), _dptr(stats), _stream())
    _check(rc, "ppfm_relax_scan")
    return pos_fz, iters


def relax_scan_batch(ff, grids, tips, fire, scans, pos_fz=None, iters=None, stats=None, want_iters=True):
    torch = _torch()
    nsys = len(grids)
    gr, tp, sc = c_array(grids, c_grid), c_array(tips, c_tip), c_array(scans, c_scan)
    nps = sum(int(s.nz) * int(s.npy) * int(s.npx) for s in sc)
    if pos_fz is None:
        pos_fz = torch.empty((nps, 4), dtype=torch.float32, device=ff.device)
    if iters is None and want_iters:
        iters = torch.empty((nps,), dtype=torch.int16, device=ff.device)
    rc = lib().ppfm_relax_scan_batch(C.c_int32(nsys), _dptr(ff, torch.float32), gr, tp, C.byref(c_fire(fire)), sc,
                                     _dptr(pos_fz, torch.float32), _dptr(iters), _dptr(stats), _stream())
    _check(rc, "ppfm_relax_scan_batch")
    return pos_fz, iters


def relax_scan_sweep(ff, grid, tips, fire, scans, pos_fz=None, iters=None, stats=None, want_iters=True):
    """ppfm_relax_scan_sweep: len(tips) scans (own springs, d0 and scan geometry each) on ONE resident grid `ff`, one
    launch, nothing replicated; outputs concatenated as in relax_scan_batch."""
    torch = _torch()
    assert len(tips) == len(scans)
    tp, sc = c_array(tips, c_tip), c_array(scans, c_scan)
    nps = sum(int(s.nz) * int(s.npy) * int(s.npx) for s in sc)
    if pos_fz is None:
        pos_fz = torch.empty((nps, 4), dtype=torch.float32, device=ff.device)
    if iters is None and want_iters:
        iters = torch.empty((nps,), dtype=torch.int16, device=ff.device)
    rc = lib().ppfm_relax_scan_sweep(C.c_int32(len(tips)), _dptr(ff, torch.float32), C.byref(c_grid(grid)), tp,
                                     C.byref(c_fire(fire)), sc, _dptr(pos_fz, torch.float32), _dptr(iters),
                                     _dptr(stats), _stream())
    _check(rc, "ppfm_relax_scan_sweep")
    return pos_fz, iters


def relax_scan_stiffness(ff, grid, tip, fire, scan, pos_fz=None, iters=None, eig=None, stats=None, want_iters=True):
    """ppfm_relax_scan_stiffness -> (pos_fz, iters, eig (nz, npy, npx, 4) float32): the scan with the stiffness map
    (Hessian eigenvalues, ascending; 4th lane 0) of every relaxed point written at the end of its z-step."""
    torch = _torch()
    shape = (int(scan.nz), int(scan.npy), int(scan.npx))
    if pos_fz is None:
        pos_fz = torch.empty(shape + (4,), dtype=torch.float32, device=ff.device)
    if iters is None and want_iters:
        iters = torch.empty(shape, dtype=torch.int16, device=ff.device)
    if eig is None:
        eig = torch.empty(shape + (4,), dtype=torch.float32, device=ff.device)
    rc = lib().ppfm_relax_scan_stiffness(_dptr(ff, torch.float32), C.byref(c_grid(grid)), C.byref(c_tip(tip)),
                                         C.byref(c_fire(fire)), C.byref(c_scan(scan)), _dptr(pos_fz, torch.float32),
                                         _dptr(iters), _dptr(eig, torch.float32), _dptr(stats), _stream())
    _check(rc, "ppfm_relax_scan_stiffness")
    return pos_fz, iters, eig


def relax_scan_stiffness_batch(ff, grids, tips, fire, scans, pos_fz=None, iters=None, eig=None, stats=None,
                               want_iters=True):
    torch = _torch()
    gr, tp, sc = c_array(grids, c_grid), c_array(tips, c_tip), c_array(scans, c_scan)
    nps = sum(int(s.nz) * int(s.npy) * int(s.npx) for s in sc)
    if pos_fz is None:
        pos_fz = torch.empty((nps, 4), dtype=torch.float32, device=ff.device)
    if iters is None and want_iters:
        iters = torch.empty((nps,), dtype=torch.int16, device=ff.device)
    if eig is None:
        eig = torch.empty((nps, 4), dtype=torch.float32, device=ff.device)
    rc = lib().ppfm_relax_scan_stiffness_batch(C.c_int32(len(grids)), _dptr(ff, torch.float32), gr, tp,
                                               C.byref(c_fire(fire)), sc, _dptr(pos_fz, torch.float32), _dptr(iters),
                                               _dptr(eig, torch.float32), _dptr(stats), _stream())
    _check(rc, "ppfm_relax_scan_stiffness_batch")
    return pos_fz, iters, eig


# ---- (2a) relaxation on an energy-only grid, tri-cubic interpolation of the potential ---------------
def energy_grid(ff, out=None):
    """ppfm_energy_grid: the .w lane of a float4 force-field grid as a contiguous float32 array of the same shape[:-1]."""
    torch = _torch()
    if out is None:
        out = torch.empty(ff.shape[:-1], dtype=torch.float32, device=ff.device)
    rc = lib().ppfm_energy_grid(_dptr(ff, torch.float32), C.c_int64(out.numel()), _dptr(out, torch.float32), _stream())
    _check(rc, "ppfm_energy_grid")
    return out


def relax_scan_tricubic(E, grid, tip, fire, scan, pos_fz=None, iters=None, stats=None, want_iters=True):
    """ppfm_relax_scan_tricubic: as relax_scan, on an energy grid E (nz, ny, nx) float32."""
    torch = _torch()
    shape = (int(scan.nz), int(scan.npy), int(scan.npx))
    if pos_fz is None:
        pos_fz = torch.empty(shape + (4,), dtype=torch.float32, device=E.device)
    if iters is None and want_iters:
        iters = torch.empty(shape, dtype=torch.int16, device=E.device)
    rc = lib().ppfm_relax_scan_tricubic(_dptr(E, torch.float32), C.byref(c_grid(grid)), C.byref(c_tip(tip)),
                                        C.byref(c_fire(fire)), C.byref(c_scan(scan)), _dptr(pos_fz, torch.float32),
                                        _dptr(iters), _dptr(stats), _stream())
    _check(rc, "ppfm_relax_scan_tricubic")
    return pos_fz, iters


def relax_scan_tricubic_batch(E, grids, tips, fire, scans, pos_fz=None, iters=None, stats=None, want_iters=True):
    torch = _torch()
    gr, tp, sc = c_array(grids, c_grid), c_array(tips, c_tip), c_array(scans, c_scan)
    nps = sum(int(s.nz) * int(s.npy) * int(s.npx) for s in sc)
    if pos_fz is None:
        pos_fz = torch.empty((nps, 4), dtype=torch.float32, device=E.device)
    if iters is None and want_iters:
        iters = torch.empty((nps,), dtype=torch.int16, device=E.device)
    rc = lib().ppfm_relax_scan_tricubic_batch(C.c_int32(len(grids)), _dptr(E, torch.float32), gr, tp,
                                              C.byref(c_fire(fire)), sc, _dptr(pos_fz, torch.float32), _dptr(iters),
                                              _dptr(stats), _stream())
    _check(rc, "ppfm_relax_scan_tricubic_batch")
    return pos_fz, iters


# ---- (2b) stiffness map (IETS module) -------------------------------------------------------------
def stiffness(ff, grid, tip, scan, pos_fz, out=None):
    """ppfm_stiffness -> (nz, npy, npx, 4) float32: Hessian eigenvalues (ascending) of the PP at pos_fz, 4th lane 0."""
    torch = _torch()
    if out is None:
        out = torch.empty((int(scan.nz), int(scan.npy), int(scan.npx), 4), dtype=torch.float32, device=ff.device)
    rc = lib().ppfm_stiffness(_dptr(ff, torch.float32), C.byref(c_grid(grid)), C.byref(c_tip(tip)),
                              C.byref(c_scan(scan)), _dptr(pos_fz, torch.float32), _dptr(out, torch.float32), _stream())
    _check(rc, "ppfm_stiffness")
    return out


def stiffness_batch(ff, grids, tips, scans, pos_fz, out=None):
    """ppfm_stiffness_batch over nsys systems laid out as in relax_scan_batch; out is (total pixel-steps, 4)."""
    torch = _torch()
    gr, tp, sc = c_array(grids, c_grid), c_array(tips, c_tip), c_array(scans, c_scan)
    if out is None:
        nps = sum(int(s.nz) * int(s.npy) * int(s.npx) for s in sc)
        out = torch.empty((nps, 4), dtype=torch.float32, device=ff.device)
    rc = lib().ppfm_stiffness_batch(C.c_int32(len(grids)), _dptr(ff, torch.float32), gr, tp, sc,
                                    _dptr(pos_fz, torch.float32), _dptr(out, torch.float32), _stream())
    _check(rc, "ppfm_stiffness_batch")
    return out


# ---- (3) df ------------------------------------------------------------------------------------------------------
def df(pos_fz, npx, npy, nz, dz, A, k0, f0, out=None, nsys=1):
    torch = _torch()
    n = int(round(A / dz))
    if out is None:
        shape = (max(nz - n, 0), npy, npx) if nsys == 1 else (nsys, max(nz - n, 0), npy, npx)
        out = torch.empty(shape, dtype=torch.float32, device=pos_fz.device)
    if nsys == 1:
        rc = lib().ppfm_df(_dptr(pos_fz, torch.float32), C.c_int32(npx), C.c_int32(npy), C.c_int32(nz),
                           C.c_double(dz), C.c_double(A), C.c_double(k0), C.c_double(f0),
                           _dptr(out, torch.float32), _stream())
    else:
        rc = lib().ppfm_df_batch(C.c_int32(nsys), _dptr(pos_fz, torch.float32), C.c_int32(npx), C.c_int32(npy),
                                 C.c_int32(nz), C.c_double(dz), C.c_double(A), C.c_double(k0), C.c_double(f0),
                                 _dptr(out, torch.float32), _stream())
    _check(rc, "ppfm_df")
    return out


def df_weights(n: int, dz: float) -> np.ndarray:
    W = np.empty(n + 1)
    _check(lib().ppfm_df_weights(C.c_int32(n), C.c_double(dz), W.ctypes.data_as(C.POINTER(C.c_double))),
           "ppfm_df_weights")
    return W


# ---- whole simulation, host buffers ------------------------------------------------------------------------------
def _hptr(x):
    """Host pointer of a torch CPU tensor or numpy array (None -> NULL)."""
    if x is None:
        return C.c_void_p(0)
    return C.c_void_p(x.data_ptr() if hasattr(x, "data_ptr") else x.ctypes.data)


def _stats_dict(st: Stats) -> dict:
    return {"total_iters": int(st.total_iters), "n_not_converged": int(st.n_not_converged),
            "n_clamped": int(st.n_clamped), "max_iters": int(st.max_iters), "warp_iters": int(st.warp_iters),
            "cell_gathers": int(st.cell_gathers), "warp_gathers": int(st.warp_gathers)}


def scan_host(w, h_xyzq, h_types, h_pos_fz=None, h_iters=None, h_df=None, Q=None) -> dict:
    """ppfm_scan_host on a workload: host (ideally pinned) torch CPU tensors or numpy arrays in and out."""
    _torch()

    R, pR = _darr(w.elem_R)
    e, pe = _darr(w.elem_e)
    st = Stats()
    rc = lib().ppfm_scan_host(C.c_int32(int(h_xyzq.shape[0])), _hptr(h_xyzq), _hptr(h_types), C.c_int32(len(R)), pR, pe,
                              C.byref(c_lattice(w.lattice)), C.byref(c_probe(w.probe, Q)), C.byref(c_grid(w.grid)),
                              C.c_double(w.r_min), C.byref(c_tip(w.tip)), C.byref(c_fire(w.fire)),
                              C.byref(c_scan(w.scan)), C.c_double(w.df.A), C.c_double(w.df.k0), C.c_double(w.df.f0),
                              _hptr(h_pos_fz), _hptr(h_iters), _hptr(h_df), C.byref(st), _stream())
    _check(rc, "ppfm_scan_host")
    return _stats_dict(st)


def scan_host_sweep(w, Qs, h_xyzq, h_types, h_pos_fz=None, h_iters=None, h_df=None) -> dict:
    """ppfm_scan_host_sweep: one split force-field pass, then combine + scan + df per tip charge in Qs; the host
    outputs hold len(Qs) consecutive result sets."""
    _torch()

    R, pR = _darr(w.elem_R)
    e, pe = _darr(w.elem_e)
    Q, pQ = _darr(list(Qs))
    st = Stats()
    rc = lib().ppfm_scan_host_sweep(C.c_int32(len(Q)), pQ, C.c_int32(int(h_xyzq.shape[0])), _hptr(h_xyzq), _hptr(h_types),
                                    C.c_int32(len(R)), pR, pe, C.byref(c_lattice(w.lattice)), C.byref(c_probe(w.probe)),
                                    C.byref(c_grid(w.grid)), C.c_double(w.r_min), C.byref(c_tip(w.tip)),
                                    C.byref(c_fire(w.fire)), C.byref(c_scan(w.scan)), C.c_double(w.df.A),
                                    C.c_double(w.df.k0), C.c_double(w.df.f0), _hptr(h_pos_fz), _hptr(h_iters), _hptr(h_df),
                                    C.byref(st), _stream())
    _check(rc, "ppfm_scan_host_sweep")
    return _stats_dict(st)


def scan_host_batch(ws, h_xyzq, h_types, h_pos_fz=None, h_iters=None, h_df=None) -> dict:
    """ppfm_scan_host_batch on a list of workloads (atoms concatenated in h_xyzq / h_types, outputs concatenated)."""
    _torch()

    w0 = ws[0]
    R, pR = _darr(w0.elem_R)
    e, pe = _darr(w0.elem_e)
    off = np.concatenate([[0], np.cumsum([w.natoms for w in ws])]).astype(np.int32)
    st = Stats()
    rc = lib().ppfm_scan_host_batch(C.c_int32(len(ws)), off.ctypes.data_as(C.c_void_p), _hptr(h_xyzq), _hptr(h_types),
                                    C.c_int32(len(R)), pR, pe, c_array([w.lattice for w in ws], c_lattice),
                                    c_array([w.probe for w in ws], c_probe), c_array([w.grid for w in ws], c_grid),
                                    C.c_double(w0.r_min), c_array([w.tip for w in ws], c_tip), C.byref(c_fire(w0.fire)),
                                    c_array([w.scan for w in ws], c_scan), C.c_double(w0.df.A), C.c_double(w0.df.k0),
                                    C.c_double(w0.df.f0), _hptr(h_pos_fz), _hptr(h_iters), _hptr(h_df), C.byref(st), _stream())
    _check(rc, "ppfm_scan_host_batch")
    return _stats_dict(st)


# ---- convenience: run a workloads.Workload end to end on device-resident inputs ------------------------------------
def upload(w, device="cuda"):
    torch = _torch()
    return (torch.from_numpy(np.ascontiguousarray(w.xyzq, dtype=np.float32)).to(device),
            torch.from_numpy(np.ascontiguousarray(w.types, dtype=np.int32)).to(device))
