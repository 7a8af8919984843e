"""CPU-only checks of the C-ABI libraries: they load without a GPU, libppfm.so exports every symbol include/ppfm.h
declares (and the launch counter / timers of include/ppfm_bench.h), libppfm_probes.so exports the probes, the ctypes
struct mirrors have the header's layout, and argument validation returns PPFM_EINVAL before any CUDA call."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2401_14564_b200 import build as ppfm_build
from paper_2401_14564_b200 import ppfm, ppfm_bench
from paper_2401_14564_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    ppfm_build.build()
    return ppfm.lib()


def header_symbols(name="ppfm.h"):
    text = open(os.path.join(ROOT, "include", name)).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(ppfm_[A-Za-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol(lib):
    names = header_symbols()
    assert len(names) >= 15
    for n in names:
        assert hasattr(lib, n), f"libppfm.so does not export {n}"
    assert set(names) == set(ppfm.EXPORTS)
    header_version = int(re.search(r"#define\s+PPFM_VERSION\s+(\d+)", open(os.path.join(ROOT, "include", "ppfm.h")).read()).group(1))
    assert lib.ppfm_version() == header_version == ppfm.HEADER_VERSION == 200
    # the measurement interface lives in its own header; the probes in their own library
    bench = header_symbols("ppfm_bench.h")
    assert set(bench) == set(ppfm_bench.EXPORTS_LIBPPFM) | set(ppfm_bench.EXPORTS_PROBES)
    assert not set(bench) & set(names)
    for n in ppfm_bench.EXPORTS_LIBPPFM:
        assert hasattr(lib, n), f"libppfm.so does not export {n}"
    probes = ppfm_bench.probes_lib()
    for n in ppfm_bench.EXPORTS_PROBES:
        assert hasattr(probes, n) and not hasattr(lib, n), n


def test_struct_layouts_match_header():
    assert C.sizeof(ppfm.Lattice) == 9 * 8 + 3 * 4 + 4
    assert C.sizeof(ppfm.Grid) == 3 * 8 + 9 * 8 + 6 * 4
    assert C.sizeof(ppfm.Probe) == 24 and C.sizeof(ppfm.Tip) == 48
    assert C.sizeof(ppfm.Fire) == 6 * 8 + 2 * 4 + 8
    assert C.sizeof(ppfm.Scan) == 9 * 8 + 3 * 4 + 4 + 8
    assert C.sizeof(ppfm.Stats) == 56


def test_defaults_and_units(lib):
    f = ppfm.fire_default()
    assert (f.dt, f.dt_max, f.finc, f.fdec, f.alpha0, f.falpha, f.n_min, f.max_iter, f.f_conv) == (
        0.5, 0.5, 1.1, 0.5, 0.1, 0.99, 5, 1000, 1e-6)
    assert ppfm.Nm_to_eVA2(0.25) == pytest.approx(0.0156037727, rel=1e-8)
    assert lib.ppfm_strerror(0) == b"ok" and lib.ppfm_strerror(-1) == b"invalid argument"


def test_invalid_arguments_are_rejected_on_the_host(lib):
    w = W.get(0)
    R = np.ascontiguousarray(w.elem_R)
    e = np.ascontiguousarray(w.elem_e)
    pd = lambda a: a.ctypes.data_as(C.POINTER(C.c_double))
    lat, pr, gr = ppfm.c_lattice(w.lattice), ppfm.c_probe(w.probe), ppfm.c_grid(w.grid)
    null = C.c_void_p(0)
    fake = C.c_void_p(0x1000)          # never dereferenced: validation fails first
    EINVAL = -1
    ff = lib.ppfm_forcefield
    assert ff(C.c_int32(10), null, fake, C.c_int32(5), pd(R), pd(e), C.byref(lat), C.byref(pr), C.byref(gr),
              C.c_double(0.1), fake, null, null) == EINVAL                       # null atoms
    assert ff(C.c_int32(-1), fake, fake, C.c_int32(5), pd(R), pd(e), C.byref(lat), C.byref(pr), C.byref(gr),
              C.c_double(0.1), fake, null, null) == EINVAL                       # negative count
    assert ff(C.c_int32(10), fake, fake, C.c_int32(0), pd(R), pd(e), C.byref(lat), C.byref(pr), C.byref(gr),
              C.c_double(0.1), fake, null, null) == EINVAL                       # no types
    assert ff(C.c_int32(10), fake, fake, C.c_int32(5), pd(R), pd(e), C.byref(lat), C.byref(pr), C.byref(gr),
              C.c_double(-1.0), fake, null, null) == EINVAL                      # negative r_min
    bad = ppfm.c_grid(w.grid)
    bad.step[2][2] = 0.0                                                   # singular step matrix
    assert ff(C.c_int32(10), fake, fake, C.c_int32(5), pd(R), pd(e), C.byref(lat), C.byref(pr), C.byref(bad),
              C.c_double(0.1), fake, null, null) == EINVAL
    bad = ppfm.c_grid(w.grid)
    bad.n[1] = 0
    assert ff(C.c_int32(10), fake, fake, C.c_int32(5), pd(R), pd(e), C.byref(lat), C.byref(pr), C.byref(bad),
              C.c_double(0.1), fake, null, null) == EINVAL
    assert ff(C.c_int32(10), C.c_void_p(0x1004), fake, C.c_int32(5), pd(R), pd(e), C.byref(lat), C.byref(pr),
              C.byref(gr), C.c_double(0.1), fake, null, null) == EINVAL          # misaligned float4 buffer

    tip, fire, sc = ppfm.c_tip(w.tip), ppfm.c_fire(w.fire), ppfm.c_scan(w.scan)
    rx = lib.ppfm_relax_scan
    assert rx(null, C.byref(gr), C.byref(tip), C.byref(fire), C.byref(sc), fake, null, null, null) == EINVAL
    badf = ppfm.c_fire(w.fire)
    badf.f_conv = 0.0
    assert rx(fake, C.byref(gr), C.byref(tip), C.byref(badf), C.byref(sc), fake, null, null, null) == EINVAL
    badt = ppfm.c_tip(w.tip)
    badt.d0[2] = 0.0                                                       # R0 = |d0| = 0
    assert rx(fake, C.byref(gr), C.byref(badt), C.byref(fire), C.byref(sc), fake, null, null, null) == EINVAL
    bads = ppfm.c_scan(w.scan)
    bads.npx = 0
    assert rx(fake, C.byref(gr), C.byref(tip), C.byref(fire), C.byref(bads), fake, null, null, null) == EINVAL

    df = lib.ppfm_df
    args = lambda nz, dz, A: (fake, C.c_int32(4), C.c_int32(4), C.c_int32(nz), C.c_double(dz), C.c_double(A),
                              C.c_double(1800.0), C.c_double(30300.0), fake, null)
    assert df(*args(40, 0.1, 0.55)) == EINVAL                              # A/dz not an integer
    assert df(*args(10, 0.1, 1.0)) == EINVAL                               # nz <= n
    assert df(*args(40, 0.0, 1.0)) == EINVAL
    assert df(*args(4000, 0.001, 1.0)) == EINVAL                           # n = 1000 > PPFM_DF_MAX_N
    # the 8(f) entry points and the host forms validate before any CUDA call too
    td = ppfm.TipDensity(0.0, 1.0, 0.0, 0.0)                               # sigma must be > 0
    assert lib.ppfm_forcefield_fft(fake, C.byref(gr), C.byref(td), fake, null) == EINVAL
    td = ppfm.TipDensity(0.5, 1.0, 0.0, 0.0)
    assert lib.ppfm_forcefield_fft(null, C.byref(gr), C.byref(td), fake, null) == EINVAL
    assert lib.ppfm_stiffness(fake, C.byref(gr), C.byref(tip), C.byref(sc), null, fake, null) == EINVAL
    assert lib.ppfm_stiffness(fake, C.byref(gr), C.byref(badt), C.byref(sc), fake, fake, null) == EINVAL
    assert lib.ppfm_relax_scan_tricubic(C.c_void_p(0x1002), C.byref(gr), C.byref(tip), C.byref(fire), C.byref(sc), fake,
                                        null, null, null) == EINVAL        # misaligned float grid
    assert lib.ppfm_energy_grid(fake, C.c_int64(-1), fake, null) == EINVAL
    rxs = lib.ppfm_relax_scan_stiffness
    assert rxs(fake, C.byref(gr), C.byref(tip), C.byref(fire), C.byref(sc), fake, null, null, null, null) == EINVAL   # no d_eig
    assert rxs(fake, C.byref(gr), C.byref(tip), C.byref(fire), C.byref(sc), fake, null, C.c_void_p(0x1004), null,
               null) == EINVAL                                             # misaligned d_eig
    assert rxs(fake, C.byref(gr), C.byref(badt), C.byref(fire), C.byref(sc), fake, null, fake, null, null) == EINVAL
    sweep = lib.ppfm_scan_host_sweep
    assert sweep(C.c_int32(0), pd(np.zeros(1)), C.c_int32(10), fake, fake, C.c_int32(5), pd(R), pd(e), C.byref(lat),
                 C.byref(pr), C.byref(gr), C.c_double(0.1), C.byref(tip), C.byref(fire), C.byref(sc), C.c_double(1.0),
                 C.c_double(1800.0), C.c_double(30300.0), fake, null, null, null, null) == EINVAL     # no charges
    off = (C.c_int32 * 3)(0, 5, 10)
    grs, tips = (ppfm.Grid * 2)(gr, gr), (ppfm.Tip * 2)(tip, tip)
    lats, prs = (ppfm.Lattice * 2)(lat, lat), (ppfm.Probe * 2)(pr, pr)
    sc2 = ppfm.c_scan(w.scan)
    sc2.nz = sc.nz + 1
    scs = (ppfm.Scan * 2)(sc, sc2)
    assert lib.ppfm_scan_host_batch(C.c_int32(2), off, fake, fake, C.c_int32(5), pd(R), pd(e), lats, prs, grs,
                                    C.c_double(0.1), tips, C.byref(fire), scs, C.c_double(1.0), C.c_double(1800.0),
                                    C.c_double(30300.0), fake, null, fake, null, null) == EINVAL      # df needs one shape
    assert lib.ppfm_combine(null, fake, C.c_double(0.1), C.c_int64(4), fake, null) == EINVAL
    assert lib.ppfm_df_weights(C.c_int32(0), C.c_double(0.1), pd(np.zeros(4))) == EINVAL


def test_host_side_df_weights_against_the_oracle(lib):
    from oracle import oracle
    for n, dz in ((10, 0.1), (20, 0.05), (1, 0.3), (64, 0.01)):
        a = ppfm.df_weights(n, dz)
        assert abs(a.sum()) < 1e-12
        assert np.allclose(a, oracle.df_weights(n, dz), rtol=1e-11, atol=1e-13)


def test_binding_fails_loudly_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    w = W.get(0)
    with pytest.raises(ppfm.PpfmError):
        ppfm.upload(w)
    with pytest.raises(ppfm.PpfmError):
        ppfm_bench.probe_fma()
    with pytest.raises(ppfm.PpfmError):
        ppfm.new_stats()
