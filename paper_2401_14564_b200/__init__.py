"""Probe-Particle Model hot path for B200 (sm_100a): force-field grid, FIRE relaxation scan, Giessibl df.

`workloads` (seeded inputs) imports without the CUDA library; `ppfm` (the thin binding over the C-ABI library
libppfm.so) fails loudly if the library is missing.  There is no CPU fallback.
"""
__all__ = ["workloads", "ppfm"]
