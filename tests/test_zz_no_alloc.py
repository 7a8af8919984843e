"""ppfm_forcefield_noalloc — the force-field pass for callers that are not allowed to allocate.

Why the entry point exists: `ppfm_forcefield` borrows a few hundred KiB of device scratch per call (packed atom records
plus two flags) from a memory pool.  That is fine for a script, but not for a program that handed out all of its GPU
memory at start-up and treats a later allocation as a fault, for an acquisition loop that cannot afford to wait on an
allocator lock or on the driver, or for a host application whose allocator hook rejects cudaMalloc* after
initialisation.  `ppfm_forcefield_noalloc` keeps that scratch in a fixed array inside the library (room for
PPFM_NOALLOC_MAX_ATOMS = 16384 atoms, held by every GPU that loads the library) and must give the same grid.

What is checked here, always on calls made back to back so that the array still holds the previous call's contents:
the grid equals the one `ppfm_forcefield` writes (the tolerance of the force-field parity tests, and in fact bit for
bit: same kernels, same summation order), stale flags and records of a larger, clamped system do not leak into the next
call, an empty atom list gives a zero grid, the atom limit is enforced with its own error code before anything is
written, the full 16384 atoms fit, and the device's free memory does not move across a call.

This file sorts last on purpose: `pytest -x` stops at the first failure, so a failure here hides no other test.  It
does not depend on anything the earlier tests did and passes in a fresh process on its own.
"""
from dataclasses import replace

import numpy as np
import pytest

from paper_2401_14564_b200 import workloads as W

# the force-field tolerances of tests/test_gpu_parity.py (north_star): |dF| <= 1e-4 |F| where |F| >= 1e-2 eV/Å, 1e-6 eV/Å
# below that; |dE| <= 1e-4 |E| + 1e-5 eV
F_REL, F_ABS, F_BIG, E_REL, E_ABS = 1e-4, 1e-6, 1e-2, 1e-4, 1e-5


@pytest.fixture(scope="module")
def P():
    import torch
    from paper_2401_14564_b200 import ppfm
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    ppfm.lib()
    return ppfm


def same_grid(got, ref, what):
    """`got` (no-alloc entry point) against `ref` (ppfm_forcefield), both CUDA tensors."""
    import torch
    torch.cuda.synchronize()
    g = got.detach().cpu().numpy().astype(np.float64).reshape(-1, 4)
    r = ref.detach().cpu().numpy().astype(np.float64).reshape(-1, 4)
    assert g.shape == r.shape and np.all(np.isfinite(g)), what
    dF = np.linalg.norm(g[:, :3] - r[:, :3], axis=1)
    Fn = np.linalg.norm(r[:, :3], axis=1)
    assert np.all(dF <= np.where(Fn >= F_BIG, F_REL * Fn, F_ABS)), f"{what}: force differs by up to {dF.max():.3e}"
    assert np.all(np.abs(g[:, 3] - r[:, 3]) <= E_REL * np.abs(r[:, 3]) + E_ABS), f"{what}: energy differs"
    # stronger than the tolerance: the two paths run the same kernels in the same order
    assert torch.equal(got.reshape(-1).view(torch.int32), ref.reshape(-1).view(torch.int32)), f"{what}: not bit-identical"


def both_paths(P, w, out, status=None):
    """The existing path's grid (fresh tensor) and the no-alloc grid written into `out`, for one workload."""
    xyzq, types = P.upload(w)
    ref = P.forcefield(xyzq, types, w.elem_R, w.elem_e, w.lattice, w.probe, w.grid, w.r_min)
    nx, ny, nz = w.grid.n
    view = out[: nx * ny * nz * 4].view(nz, ny, nx, 4)
    view.fill_(float("nan"))                       # the call must write every point itself
    got = P.forcefield_noalloc(xyzq, types, w.elem_R, w.elem_e, w.lattice, w.probe, w.grid, view, w.r_min,
                               status=status)
    return got, ref


@pytest.mark.gpu
def test_noalloc_forcefield_matches_the_pooled_path_on_calls_in_a_row(P):
    import torch
    out = torch.empty(4 * 250 * 250 * 16, dtype=torch.float32, device="cuda")      # the caller's output arena

    # call 1: 560-atom periodic slab (3 atom chunks, 9 images), ragged tiles, one atom sitting on a grid node with a
    # large r_min: the clamp flag is SET and 560 records are left behind in the array
    w2 = W.get(2)
    x = w2.xyzq.copy()
    g1 = replace(w2.grid, n=(37, 23, 13), step=np.diag([0.31, 0.47, 0.53]))
    x[0, :3] = g1.origin + np.array([5 * 0.31, 6 * 0.47, 2 * 0.53])
    w_big = replace(w2, xyzq=x, grid=g1, r_min=0.5)
    st = P.new_ff_status()
    got, ref = both_paths(P, w_big, out, status=st)
    same_grid(got, ref, "call 1 (slab, clamp live)")
    assert P.read_ff_status(st) == {"n_bad_type": 0, "n_clamped": 1}

    # call 2, straight after on the same stream: 10-atom molecule, no clamp, a grid of several z-groups — must not see
    # call 1's flags (clamp, charged-atom count) or its 550 extra records
    w0 = W.get(0)
    got, ref = both_paths(P, w0, out, status=st)
    same_grid(got, ref, "call 2 (config 0 after the slab)")
    assert P.read_ff_status(st) == {"n_bad_type": 0, "n_clamped": 0}
    from oracle import oracle                       # and the existing path is the one the oracle vouches for
    o = oracle.forcefield(w0).reshape(-1, 4)
    g = got.cpu().numpy().astype(np.float64).reshape(-1, 4)
    Fn = np.linalg.norm(o[:, :3], axis=1)
    assert np.all(np.linalg.norm(g[:, :3] - o[:, :3], axis=1) <= np.where(Fn >= F_BIG, F_REL * Fn, F_ABS))

    # call 3: the same call again (the array now holds exactly this call's own leftovers) while the device's free memory
    # is watched: nothing may be allocated.  (The first use of a kernel can load its code, hence the repeat.)
    xyzq, types = P.upload(w0)
    nx, ny, nz = w0.grid.n
    view = out[: nx * ny * nz * 4].view(nz, ny, nx, 4)
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info()
    P.forcefield_noalloc(xyzq, types, w0.elem_R, w0.elem_e, w0.lattice, w0.probe, w0.grid, view, w0.r_min)
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    assert free_after >= free_before, f"device memory shrank by {free_before - free_after} bytes across the call"
    same_grid(view, ref, "call 3 (repeat)")

    # call 4: no atoms at all — no set-up kernel runs, so the flags the grid kernel reads are only right if the call
    # cleared what call 3 left
    empty_x = torch.zeros((0, 4), dtype=torch.float32, device="cuda")
    empty_t = torch.zeros((0,), dtype=torch.int32, device="cuda")
    small = W.shrink(w0, grid_n=(9, 7, 5))
    view = out[: 9 * 7 * 5 * 4].view(5, 7, 9, 4)
    view.fill_(float("nan"))
    P.forcefield_noalloc(empty_x, empty_t, small.elem_R, small.elem_e, small.lattice, small.probe, small.grid, view)
    torch.cuda.synchronize()
    assert float(view.abs().max()) == 0.0


@pytest.mark.gpu
def test_noalloc_forcefield_atom_limit(P):
    import torch
    w0 = W.shrink(W.get(0), grid_n=(16, 12, 6))
    rng = np.random.default_rng(5)
    n = P.NOALLOC_MAX_ATOMS + 1
    xyz = rng.uniform([-20, -20, -6], [30, 30, -1], size=(n, 3))      # a wide slab of atoms below the grid
    q = rng.uniform(-0.2, 0.2, size=n)
    q[::3] = 0.0                                                        # a third LJ-only: the partition has work to do
    xyzq = np.concatenate([xyz, q[:, None]], axis=1).astype(np.float32)
    types = rng.integers(0, len(w0.elem_R), size=n).astype(np.int32)
    dx, dt = torch.from_numpy(xyzq).cuda(), torch.from_numpy(types).cuda()
    out = torch.full((6, 12, 16, 4), 7.0, dtype=torch.float32, device="cuda")

    # one atom too many: refused with the limit's own status, and the caller's grid is untouched
    with pytest.raises(P.PpfmError) as err:
        P.forcefield_noalloc(dx, dt, w0.elem_R, w0.elem_e, w0.lattice, w0.probe, w0.grid, out, w0.r_min)
    assert f"{P.ELIMIT}" in str(err.value) and "PPFM_NOALLOC_MAX_ATOMS" in str(err.value)
    torch.cuda.synchronize()
    assert float((out - 7.0).abs().max()) == 0.0
    assert P.lib().ppfm_strerror(P.ELIMIT).startswith(b"input exceeds the fixed scratch")

    # exactly the maximum fits, twice in a row, and matches the pooled path
    dx, dt = dx[:-1].contiguous(), dt[:-1].contiguous()
    ref = P.forcefield(dx, dt, w0.elem_R, w0.elem_e, w0.lattice, w0.probe, w0.grid, w0.r_min)
    for rep in range(2):
        out.fill_(float("nan"))
        P.forcefield_noalloc(dx, dt, w0.elem_R, w0.elem_e, w0.lattice, w0.probe, w0.grid, out, w0.r_min)
        same_grid(out, ref, f"16384 atoms, call {rep + 1}")
