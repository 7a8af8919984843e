"""Build step: nvcc-compile csrc/*.cu for sm_100a into paper_2401_14564_b200/libppfm.so (in-tree, git-ignored).

Run as `python -m paper_2401_14564_b200.build [--force] [--verbose]`; also called by __graft_entry__.build().
Each .cu is compiled to an object in parallel (objects under paper_2401_14564_b200/build/, git-ignored), then linked.
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJDIR = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libppfm.so")
CHK_LIB = os.path.join(HERE, "libppfm_chk.so")             # checked build: same sources, -DPPFM_CHECKS (ppfm_bench.h)
CHK_OBJDIR = os.path.join(HERE, "build", "chk")
PROBES_SRC = os.path.join(HERE, "csrc_probes", "probes.cu")
PROBES_LIB = os.path.join(HERE, "libppfm_probes.so")      # include/ppfm_bench.h (b): measurement only
NVCC_COMPILE = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-Xcompiler", "-fPIC",
                "-c"]
NVCC_LINK = ["-gencode", "arch=compute_100a,code=sm_100a", "--shared", "-Xcompiler", "-fPIC", "-cudart", "static",
             "-lcufft", "-Xlinker", "-rpath=/usr/local/cuda/lib64"]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def headers():
    return sorted(glob.glob(os.path.join(CSRC, "*.cuh"))) + sorted(
        glob.glob(os.path.join(os.path.dirname(HERE), "include", "*.h")))


def build(force: bool = False, verbose: bool = False, extra_flags=(), lib: str = LIB, objdir: str = OBJDIR) -> str:
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    os.makedirs(objdir, exist_ok=True)
    chk = None
    if lib == LIB:            # the checked build compiles alongside
        chk = ThreadPoolExecutor(max_workers=1)
        chk_done = chk.submit(build, force, verbose, ("-DPPFM_CHECKS",), CHK_LIB, CHK_OBJDIR)
    hdr_time = max(os.path.getmtime(h) for h in headers())
    jobs, objs = [], []
    for src in sources():
        obj = os.path.join(objdir, os.path.splitext(os.path.basename(src))[0] + ".o")
        objs.append(obj)
        if force or not os.path.exists(obj) or os.path.getmtime(obj) < max(os.path.getmtime(src), hdr_time):
            jobs.append([nvcc] + NVCC_COMPILE + list(extra_flags) + (["-Xptxas", "-v"] if verbose else []) +
                        ["-o", obj, src])
    if jobs:
        with ThreadPoolExecutor(max_workers=min(len(jobs), os.cpu_count() or 1)) as ex:
            for r in ex.map(lambda c: subprocess.run(c, capture_output=True, text=True), jobs):
                if verbose or r.returncode:
                    sys.stderr.write(r.stdout + r.stderr)
                if r.returncode:
                    raise subprocess.CalledProcessError(r.returncode, r.args)
    if jobs or not os.path.exists(lib) or any(os.path.getmtime(lib) < os.path.getmtime(o) for o in objs):
        subprocess.run([nvcc] + NVCC_LINK + ["-o", lib] + objs, check=True)
    if chk is not None:
        chk_done.result()
        chk.shutdown()
    if lib == LIB and (force or not os.path.exists(PROBES_LIB) or
                       os.path.getmtime(PROBES_LIB) < max(os.path.getmtime(PROBES_SRC), hdr_time)):
        subprocess.run([nvcc] + [f for f in NVCC_COMPILE if f != "-c"] + ["--shared", "-cudart", "static", "-o",
                                                                          PROBES_LIB, PROBES_SRC], check=True)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
