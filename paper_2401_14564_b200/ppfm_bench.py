"""Binding of the measurement interface (include/ppfm_bench.h): launch counter and per-kernel device timers exported
by libppfm.so, and the two roofline probes of the separate libppfm_probes.so.  Used by bench.py and the tests; the
product binding (ppfm.py) does not import this module."""
from __future__ import annotations

import ctypes as C
import os

from . import ppfm

PROBES_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libppfm_probes.so")
EXPORTS_LIBPPFM = ["ppfm_launch_count", "ppfm_timing_enable", "ppfm_timing_read", "ppfm_checks_read"]
CHECK_KINDS = ["ring_acquire", "ring_release", "ff_store", "relax_gather", "relax_store", "df_load", "df_store", "visits"]
EXPORTS_PROBES = ["ppfm_probe_fma", "ppfm_probe_gather"]
KERNEL_IDS = {"ff_prep": 0, "ff": 1, "combine": 2, "relax": 3, "df": 4, "stiffness": 5, "fft_el": 6, "relax_tricubic": 7, "ff_energy": 8}
_probes = None


def probes_lib():
    global _probes
    if _probes is None:
        if not os.path.exists(PROBES_PATH):
            raise ppfm.PpfmError(f"{PROBES_PATH} not found - build it with `python -m paper_2401_14564_b200.build`")
        _probes = C.CDLL(PROBES_PATH)
    return _probes


def launch_count() -> int:
    f = ppfm.lib().ppfm_launch_count
    f.restype = C.c_int64
    return int(f())


def timing_enable(on: bool = True) -> None:
    """ppfm_timing_enable: bracket every kernel launch with CUDA events inside the library (clears the totals)."""
    ppfm._check(ppfm.lib().ppfm_timing_enable(C.c_int(int(on))), "ppfm_timing_enable")


def timing_read() -> dict:
    """ppfm_timing_read for every kernel: {name: (total ms, launches)}."""
    out = {}
    for name, kid in KERNEL_IDS.items():
        ms, n = C.c_double(0.0), C.c_int64(0)
        ppfm._check(ppfm.lib().ppfm_timing_read(C.c_int(kid), C.byref(ms), C.byref(n)), "ppfm_timing_read")
        out[name] = (ms.value, int(n.value))
    return out


def checks_read():
    """ppfm_checks_read: {kind: count} since the last call, or None when the loaded library is not the checked build."""
    c = (C.c_uint64 * 8)()
    rc = ppfm.lib().ppfm_checks_read(c)
    if rc:
        return None
    return {k: int(v) for k, v in zip(CHECK_KINDS, c)}


def probe_fma() -> float:
    """FP32 lane-instructions per second of an FFMA-only kernel."""
    v = C.c_double(0.0)
    rc = probes_lib().ppfm_probe_fma(C.byref(v), ppfm._stream())
    if rc:
        raise ppfm.PpfmError(f"ppfm_probe_fma failed: {rc}")
    return v.value


def probe_gather(n_float4: int, bypass_l1: bool) -> float:
    """GB/s of the relaxation's 8-corner float4 gather pattern without dependent math (L2-only when bypass_l1)."""
    v = C.c_double(0.0)
    rc = probes_lib().ppfm_probe_gather(C.c_int64(n_float4), C.c_int32(int(bypass_l1)), C.byref(v), ppfm._stream())
    if rc:
        raise ppfm.PpfmError(f"ppfm_probe_gather failed: {rc}")
    return v.value
