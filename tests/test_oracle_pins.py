"""Pins for the FP64 CPU oracle (oracle/ppfm_oracle.c) against what the paper and the mathematics fix.

The paper prints no worked numeric example, so every pin is a closed form, an invariant, a special
case that reduces to a library routine (scipy trilinear map_coordinates, scipy quad, scipy Bessel I1, numpy
eigvalsh), or brute force on tiny inputs.  Citations are /root/reference/PAPER.md lines.
"""
import os
from dataclasses import replace

import numpy as np
import pytest
from scipy import integrate, ndimage, special

from oracle import oracle
from paper_2401_14564_b200 import workloads as W

GOLD = {}
with open(os.path.join(os.path.dirname(__file__), "golden", "constants.txt")) as fh:
    for line in fh:
        line = line.split("#")[0].split()
        if len(line) == 2:
            GOLD[line[0]] = float(line[1])
KE = GOLD["k_e_eV_A"]
NM = GOLD["eVA2_in_Nm"]


def one_atom(R=1.908, e=3.73e-3, q=0.0, Rpp=1.661, epp=9.11e-3, Q=0.0, pos=(0.0, 0.0, 0.0)):
    w = W.get(0)
    return replace(w, xyzq=np.array([[pos[0], pos[1], pos[2], q]], dtype=np.float32),
                   types=np.array([0], dtype=np.int32), elem_R=np.array([R]), elem_e=np.array([e]),
                   probe=W.Probe(R=Rpp, e=epp, Q=Q), r_min=1e-3)


# ---------------------------------------------------------------------------------------------------- O1-O2 LJ
def test_lj_minimum_depth_and_zero_crossing():
    """Eq.5 + mixing: E(R0) = -E0, F(R0) = 0, E(R0 * 2^(-1/6)) = 0."""
    R, e, Rpp, epp = 1.908, 3.73e-3, 1.661, 9.11e-3
    w = one_atom(R, e, 0.0, Rpp, epp, 0.0)
    R0, E0 = R + Rpp, np.sqrt(e * epp)
    out = oracle.ff_at_points(w, [[0, 0, R0], [R0 * 2 ** (-1 / 6), 0, 0], [0, R0, 0]])
    assert out[0, 3] == pytest.approx(-E0, rel=1e-14)
    assert np.abs(out[0, :3]).max() < 1e-15
    assert abs(out[1, 3]) < 1e-16
    assert out[2, 3] == pytest.approx(-E0, rel=1e-14)


def test_lj_radial_force_profile():
    """-dE/dr of Eq.5: F_r = 12 E0 [(R0/r)^12 - (R0/r)^6] / r, along an oblique direction."""
    R, e, Rpp, epp = 1.78, 3.04e-3, 1.661, 9.11e-3
    w = one_atom(R, e, 0.0, Rpp, epp, 0.0, pos=(0.5, -0.25, 0.125))
    R0, E0 = R + Rpp, np.sqrt(e * epp)
    nhat = np.array([1.0, 2.0, -2.0]) / 3.0
    for r in (2.0, 3.0, R0, 4.5, 7.0):
        p = np.array([0.5, -0.25, 0.125]) + r * nhat
        out = oracle.ff_at_points(w, [p])[0]
        Fr = 12 * E0 * ((R0 / r) ** 12 - (R0 / r) ** 6) / r
        assert np.allclose(out[:3], Fr * nhat, rtol=1e-12, atol=1e-15)
        assert out[3] == pytest.approx(E0 * ((R0 / r) ** 12 - 2 * (R0 / r) ** 6), rel=1e-12, abs=1e-18)


# ---------------------------------------------------------------------------------------------------- O2 Coulomb
def test_coulomb_value_sign_and_inverse_square():
    """Eq.6: E r = k_e Q q; F(2r) = F(r)/4; sign follows Q q; E(1 Å, Q=q=1) = 14.399645478 eV."""
    w = one_atom(e=0.0, q=1.0, Q=1.0)      # e_i = 0 -> E0 = 0, pure Coulomb
    out = oracle.ff_at_points(w, [[1, 0, 0], [2, 0, 0], [0, 0, 3]])
    assert out[0, 3] == pytest.approx(KE, rel=1e-12)
    assert out[0, 0] == pytest.approx(KE, rel=1e-12)           # repulsive: pushes +x
    assert out[1, 0] == pytest.approx(out[0, 0] / 4, rel=1e-12)
    assert out[2, 3] * 3 == pytest.approx(KE, rel=1e-12)
    for Q, q in ((-1, 1), (1, -1)):
        o = oracle.ff_at_points(one_atom(e=0.0, q=q, Q=Q), [[1, 0, 0]])[0]
        assert o[0] == pytest.approx(-KE, rel=1e-12) and o[3] == pytest.approx(-KE, rel=1e-12)
    o = oracle.ff_at_points(one_atom(e=0.0, q=-1, Q=-1), [[1, 0, 0]])[0]
    assert o[0] == pytest.approx(KE, rel=1e-12)


def test_rmin_clamp_is_identity_outside_and_finite_inside():
    """Reading S3: s = max(r^2, r_min^2); direction from the unclamped displacement."""
    w = replace(one_atom(q=0.3, Q=-0.05), r_min=0.5)
    a = oracle.ff_at_points(w, [[0.6, 0, 0]], r_min=0.5)
    b = oracle.ff_at_points(w, [[0.6, 0, 0]], r_min=1e-3)
    assert np.array_equal(a, b)
    c = oracle.ff_at_points(w, [[0, 0, 0], [0.1, 0, 0]], r_min=0.5)
    assert np.all(np.isfinite(c)) and np.all(c[0, :3] == 0.0)
    assert c[0, 3] == c[1, 3]                              # energy is flat inside the clamp


# ---------------------------------------------------------------------------------------------------- F = -grad E
def test_force_is_minus_gradient_of_energy_cfg0():
    """F = -grad E, on the summed LJ + Coulomb field of config 0 at 100 random points."""
    w = W.get(0)
    rng = np.random.default_rng(7)
    pts = np.c_[rng.uniform(0, 12, 100), rng.uniform(0, 12, 100), rng.uniform(2.0, 9.0, 100)]
    F = oracle.ff_at_points(w, pts)[:, :3]
    h = 1e-4
    G = np.zeros_like(F)
    for a in range(3):
        dp = np.zeros(3)
        dp[a] = h
        Ep = oracle.ff_at_points(w, pts + dp)[:, 3]
        Em = oracle.ff_at_points(w, pts - dp)[:, 3]
        Epp = oracle.ff_at_points(w, pts + 2 * dp)[:, 3]
        Emm = oracle.ff_at_points(w, pts - 2 * dp)[:, 3]
        G[:, a] = -(8 * (Ep - Em) - (Epp - Emm)) / (12 * h)      # 4th-order central difference
    err = np.linalg.norm(F - G, axis=1) / np.maximum(np.linalg.norm(F, axis=1), 1e-6)
    assert err.max() < 1e-7


# ---------------------------------------------------------------------------------------------------- O3 sums
def test_brute_force_tiny_grid():
    """3 atoms, 4x4x4 grid, independent triple loop written from Eq.5/Eq.6 in radial form."""
    w = W.get(0)
    w = replace(w, xyzq=np.array([[1.0, 1.5, 0.0, 0.2], [2.5, 0.5, -0.2, -0.3], [0.3, 2.2, 0.1, 0.1]], np.float32),
                types=np.array([1, 3, 0], np.int32),
                grid=W.Grid(origin=np.array([0.1, 0.2, 2.0]), step=np.diag([0.7, 0.8, 0.9]), n=(4, 4, 4),
                            periodic=(0, 0, 0)))
    ff = oracle.forcefield(w)
    ref = np.zeros((4, 4, 4, 4))
    for k in range(4):
        for j in range(4):
            for i in range(4):
                p = np.array([0.1 + 0.7 * i, 0.2 + 0.8 * j, 2.0 + 0.9 * k])
                for a in range(3):
                    x, y, z, q = [float(v) for v in w.xyzq[a]]
                    Rm = w.elem_R[w.types[a]] + w.probe.R
                    em = np.sqrt(w.elem_e[w.types[a]] * w.probe.e)
                    D = p - np.array([x, y, z])
                    r = np.linalg.norm(D)
                    rho = Rm / r
                    dEdr = em * (-12 * rho ** 12 + 12 * rho ** 6) / r - KE * w.probe.Q * q / r ** 2
                    ref[k, j, i, :3] += -dEdr * D / r
                    ref[k, j, i, 3] += em * (rho ** 12 - 2 * rho ** 6) + KE * w.probe.Q * q / r
    assert np.allclose(ff, ref, rtol=1e-12, atol=1e-16)


def test_linearity_permutation_and_charge_linearity():
    w = replace(W.shrink(W.get(0), grid_n=(12, 10, 6)))
    ff = oracle.forcefield(w)
    A = replace(w, xyzq=w.xyzq[:4], types=w.types[:4])
    B = replace(w, xyzq=w.xyzq[4:], types=w.types[4:])
    assert np.allclose(oracle.forcefield(A) + oracle.forcefield(B), ff, rtol=1e-12, atol=1e-15)
    perm = np.random.default_rng(3).permutation(w.natoms)
    assert np.allclose(oracle.forcefield(replace(w, xyzq=w.xyzq[perm], types=w.types[perm])), ff, rtol=1e-12,
                       atol=1e-15)
    f0, f1, f2 = (oracle.forcefield(w, Q=Q) for Q in (0.0, 0.1, 0.2))
    assert np.allclose(f2 - f0, 2 * (f1 - f0), rtol=1e-10, atol=1e-15)       # el part linear in Q


def test_image_sum_equals_explicit_replication():
    """Periodic images: nimg = 1 equals the 9x replicated atom list with nimg = 0."""
    w = W.get(2)
    idx = W.sample_indices(w.npoints, 300, 11)
    ref = oracle.forcefield(w, idx=idx)
    reps, types = [], []
    for ia in (-1, 0, 1):
        for ib in (-1, 0, 1):
            sh = ia * w.lattice.a + ib * w.lattice.b
            x = w.xyzq.astype(np.float64).copy()
            x[:, :3] += sh
            reps.append(x)
            types.append(w.types)
    # replicated coordinates are exact in FP64 but not FP32 -> go through ff_at_points with float64 atoms
    big = replace(w, lattice=replace(w.lattice, nimg=(0, 0, 0)))
    nx, ny, nz = w.grid.n
    i, j, k = idx % nx, (idx // nx) % ny, idx // (nx * ny)
    pts = w.grid.origin + np.outer(i, w.grid.step[0]) + np.outer(j, w.grid.step[1]) + np.outer(k, w.grid.step[2])
    tot = np.zeros((len(idx), 4))
    for x, t in zip(reps, types):
        # shift points instead of atoms (same displacement, atoms stay FP32-exact)
        sh = x[0, :3] - w.xyzq[0, :3].astype(np.float64)
        tot += oracle.ff_at_points(big, pts - sh)
    assert np.allclose(tot, ref, rtol=1e-11, atol=1e-14)


def test_mirror_symmetry():
    """Mirror x -> -x about the plane through grid index (n-1)/2: (Fx,Fy,Fz,E) -> (-Fx,Fy,Fz,E) at mirrored i."""
    w = W.shrink(W.get(0), grid_n=(21, 8, 5))
    xm = w.grid.origin[0] + 0.5 * (w.grid.n[0] - 1) * w.grid.step[0, 0]
    # choose coordinates for which the FP32 mirror image is exact: multiples of 1/64
    x = np.round(w.xyzq.astype(np.float64) * 64) / 64
    w = replace(w, xyzq=x.astype(np.float32), grid=replace(w.grid, origin=np.array([0.0, 0.0, 1.5])))
    xm = 0.5 * (w.grid.n[0] - 1) * 0.2
    xr = x.copy()
    xr[:, 0] = 2 * xm - xr[:, 0]
    assert np.array_equal(xr.astype(np.float32).astype(np.float64), xr)
    a = oracle.forcefield(w)
    b = oracle.forcefield(replace(w, xyzq=xr.astype(np.float32)))[:, :, ::-1, :]
    assert np.allclose(a[..., 0], -b[..., 0], rtol=1e-9, atol=1e-13)
    assert np.allclose(a[..., 1:], b[..., 1:], rtol=1e-9, atol=1e-13)


def test_translation_of_atoms_and_origin():
    """Translating atoms and grid origin by the same vector leaves the array unchanged."""
    w = W.shrink(W.get(0), grid_n=(9, 7, 5))
    x = np.round(w.xyzq.astype(np.float64) * 64) / 64
    w = replace(w, xyzq=x.astype(np.float32))
    t = np.array([0.5, -1.25, 0.75])
    x2 = x.copy()
    x2[:, :3] += t
    w2 = replace(w, xyzq=x2.astype(np.float32), grid=replace(w.grid, origin=w.grid.origin + t))
    assert np.allclose(oracle.forcefield(w), oracle.forcefield(w2), rtol=1e-10, atol=1e-14)


def test_lattice_translation_invariance_lj_nimg4():
    """Reading S18: with nimg = 4 and LJ only the truncated image sum is invariant (to < 1e-6) under moving one
    atom by a lattice vector."""
    w = W.get(2)
    x = np.round(w.xyzq.astype(np.float64) * 64) / 64      # so that x + 25 stays exact in FP32
    x[:, 3] = 0.0
    w = replace(w, xyzq=x.astype(np.float32))
    pts = np.array([[12.3, 11.9, 3.1], [2.0, 20.0, 3.5], [24.0, 1.0, 4.0]])
    a = oracle.ff_at_points(w, pts, nimg=(4, 4, 0))
    x = x.copy()
    x[:60, 0] += 25.0                                   # move the molecule by +a
    assert np.array_equal(x.astype(np.float32).astype(np.float64), x)
    b = oracle.ff_at_points(replace(w, xyzq=x.astype(np.float32)), pts, nimg=(4, 4, 0))
    assert np.allclose(a, b, rtol=5e-6, atol=1e-9)        # r^-6 tail of the dropped/added image row: <= 1e-8 eV
    c = oracle.ff_at_points(replace(w, xyzq=x.astype(np.float32)), pts, nimg=(0, 0, 0))
    assert not np.allclose(a, c, rtol=1e-3, atol=1e-12)   # and the images do matter


# ---------------------------------------------------------------------------------------------------- O4
def _rand_grid(n=(7, 6, 5), periodic=(0, 0, 0), seed=0, h=(0.3, 0.25, 0.2), origin=(0.5, -0.2, 1.0)):
    rng = np.random.default_rng(seed)
    g = W.Grid(origin=np.array(origin), step=np.diag(h), n=n, periodic=periodic)
    ff = rng.normal(size=(n[2], n[1], n[0], 4))
    return g, ff


def test_interp_matches_scipy_map_coordinates():
    """Tri-linear interpolation == scipy.ndimage.map_coordinates(order=1), clamped and periodic."""
    rng = np.random.default_rng(1)
    for periodic, mode in (((0, 0, 0), "nearest"), ((1, 1, 1), "grid-wrap")):
        g, ff = _rand_grid(periodic=periodic)
        h = np.diag(g.step)
        lo = -1.5 if periodic[0] else 0.0
        t = np.c_[rng.uniform(lo, g.n[0] + (0.5 if periodic[0] else -1.0), 200),
                  rng.uniform(lo, g.n[1] + (0.5 if periodic[0] else -1.0), 200),
                  rng.uniform(lo, g.n[2] + (0.5 if periodic[0] else -1.0), 200)]
        pts = g.origin + t * h
        got = oracle.interp(ff, g, pts)
        for c in range(3):
            ref = ndimage.map_coordinates(ff[..., c], [t[:, 2], t[:, 1], t[:, 0]], order=1, mode=mode)
            assert np.allclose(got[:, c], ref, rtol=1e-10, atol=1e-12)


def test_interp_clamps_outside_nonperiodic():
    g, ff = _rand_grid()
    h = np.diag(g.step)
    inside = g.origin + np.array([0.0, 2.3, 4.0]) * h
    outside = g.origin + np.array([-3.0, 2.3, 9.0]) * h
    assert np.allclose(oracle.interp(ff, g, [inside]), oracle.interp(ff, g, [outside]), atol=1e-14)


def test_interp_affine_exact_and_nodes():
    """An affine field sampled on the grid is reproduced exactly anywhere inside; nodes return node values.
    Also with a non-orthogonal step matrix."""
    rng = np.random.default_rng(2)
    step = np.array([[0.3, 0.02, 0.0], [-0.05, 0.25, 0.01], [0.0, 0.03, 0.2]])
    g = W.Grid(origin=np.array([0.5, -0.2, 1.0]), step=step, n=(6, 5, 7), periodic=(0, 0, 0))
    M = rng.normal(size=(3, 3))
    b = rng.normal(size=3)
    k, j, i = np.meshgrid(np.arange(7), np.arange(5), np.arange(6), indexing="ij")
    P = g.origin + i[..., None] * step[0] + j[..., None] * step[1] + k[..., None] * step[2]
    ff = np.zeros((7, 5, 6, 4))
    ff[..., :3] = P @ M.T + b
    t = np.c_[rng.uniform(0, 5, 50), rng.uniform(0, 4, 50), rng.uniform(0, 6, 50)]
    pts = g.origin + t @ step
    assert np.allclose(oracle.interp(ff, g, pts), pts @ M.T + b, rtol=1e-11, atol=1e-12)
    assert np.allclose(oracle.interp(ff, g, P[3, 2, 4][None]), ff[3, 2, 4, :3][None], atol=1e-12)


def test_interp_periodic_seam():
    g, ff = _rand_grid(periodic=(1, 1, 0))
    h = np.diag(g.step)
    t = np.array([g.n[0] - 0.25, 1.5, 2.5])              # between last and first node in x
    got = oracle.interp(ff, g, [g.origin + t * h])[0]
    f = lambda i: 0.25 * ff[2, 1, i, :3] + 0.25 * ff[2, 2, i, :3] + 0.25 * ff[3, 1, i, :3] + 0.25 * ff[3, 2, i, :3]
    assert np.allclose(got, 0.25 * f(g.n[0] - 1) + 0.75 * f(0), atol=1e-13)
    a = oracle.interp(ff, g, [g.origin + np.array([1.3, 2.2, 2.5]) * h])
    b = oracle.interp(ff, g, [g.origin + np.array([1.3 + g.n[0], 2.2 - g.n[1], 2.5]) * h])
    assert np.allclose(a, b, atol=1e-12)


def test_f32_grid_is_widened_on_access():
    g, ff = _rand_grid()
    ff32 = ff.astype(np.float32)
    pts = g.origin + np.array([[1.2, 2.3, 3.4]]) * np.diag(g.step)
    assert np.array_equal(oracle.interp(ff32, g, pts), oracle.interp(ff32.astype(np.float64), g, pts))


# ---------------------------------------------------------------------------------------------------- O5-O8
def _flat_grid(n=(20, 20, 60), h=0.2, origin=(0.0, 0.0, 0.0)):
    g = W.Grid(origin=np.array(origin, float), step=np.diag([h, h, h]), n=n, periodic=(0, 0, 0))
    return g, np.zeros((n[2], n[1], n[0], 4))


def _scan(npx=3, npy=2, nz=25, z0=9.0, dz=0.1):
    return W.Scan(p0=np.array([1.0, 1.2, z0]), dx=np.array([0.3, 0, 0.0]), dy=np.array([0, 0.4, 0.0]), npx=npx,
                  npy=npy, nz=nz, dz=dz)


def test_zero_field_stays_at_spring_equilibrium():
    """All-zero grid: r_PP = r_TIP + d0 exactly, 0 iterations, Fz = 0, df = 0 (Eq.2)."""
    g, ff = _flat_grid()
    tip, sc = W._default_tip(), _scan()
    r = oracle.relax_scan(ff, g, tip, W.Fire(), sc)
    assert np.all(r["iters"] == 0)
    for iz in range(sc.nz):
        for iy in range(sc.npy):
            for ix in range(sc.npx):
                want = sc.p0 + ix * sc.dx + iy * sc.dy - np.array([0, 0, iz * sc.dz]) + np.array(tip.d0)
                assert np.array_equal(r["pos_fz"][iz, iy * sc.npx + ix, :3], want)
    assert np.all(r["pos_fz"][..., 3] == 0.0)
    assert np.all(oracle.df(r["pos_fz"][..., 3], sc.dz, 1.0, 1800.0, 30300.0) == 0.0)


def test_uniform_field_closed_form_and_lateral_hessian():
    """Uniform F_S = (0,0,f): |d| = R_rest - f/k_R, Fz_tip = f; lateral Hessian eigenvalue
    k_xy - f/|d| (pins O10), including its sign change at f ~ k_xy R_rest."""
    g, ff = _flat_grid()
    tip = W._default_tip()
    fire = replace(W.Fire(), f_conv=1e-11, max_iter=20000)
    for f in (0.03, -0.02, 0.07):
        ff[..., 2] = f
        r = oracle.relax_scan(ff, g, tip, fire, _scan(nz=2))
        L = 4.0 - f / tip.k_rad
        d = r["pos_fz"][0, 0, :3] - _scan().p0
        assert np.allclose(d, [0, 0, -L], atol=1e-8)
        assert r["pos_fz"][0, 0, 3] == pytest.approx(f, abs=1e-9)
        H, w = oracle.hessian(ff, g, tip, _scan().p0, r["pos_fz"][0, 0, :3])
        lam_lat = tip.k_lat[0] - f / L
        assert w[0] == pytest.approx(min(lam_lat, tip.k_rad), abs=1e-9)
        assert r["lam_min"][0, 0] == pytest.approx(lam_lat, abs=1e-9)
        assert np.allclose(w, np.linalg.eigvalsh(H), atol=1e-12)
    assert tip.k_lat[0] - 0.07 / (4.0 - 0.07 / tip.k_rad) < 0 < tip.k_lat[0] - 0.03 / (4.0 - 0.03 / tip.k_rad)


def test_linear_field_relax_plus_df_closed_form():
    """F_S,z = g (z - z_c): Fz_tip = k_R g (z_t - R_rest - z_c)/(k_R - g);
    df = -(f0/2k0) * 16.0218 * k_R g/(k_R - g) for every window (Eq.2 + Eq.3 end to end)."""
    grid, ff = _flat_grid()
    gsl, zc = 0.37, 4.1
    zk = grid.origin[2] + 0.2 * np.arange(grid.n[2])
    ff[..., 2] = (gsl * (zk - zc))[:, None, None]
    tip = W._default_tip()
    fire = replace(W.Fire(), f_conv=1e-12, max_iter=50000)
    for dz, nz in ((0.1, 25), (0.05, 45)):
        sc = _scan(nz=nz, dz=dz)
        r = oracle.relax_scan(ff, grid, tip, fire, sc)
        zt = sc.p0[2] - dz * np.arange(nz)
        want = tip.k_rad * gsl * (zt - 4.0 - zc) / (tip.k_rad - gsl)
        assert np.allclose(r["pos_fz"][:, 0, 3], want, atol=1e-9)
        df = oracle.df(r["pos_fz"][..., 3], dz, 1.0, 1800.0, 30300.0)
        assert df.shape[0] == nz - int(round(1.0 / dz))
        assert np.allclose(df, -(30300.0 / 3600.0) * NM * tip.k_rad * gsl / (tip.k_rad - gsl), rtol=1e-7)


def test_fire_finds_a_true_minimum_newton_crosscheck_cfg0():
    """O6: on config 0 the FIRE end point is a stationary point with positive-definite Hessian, and a damped
    Newton iteration (analytic Jacobian) started there does not move it by more than 1e-6 Å (non-flagged)."""
    w = W.get(0)
    ff = oracle.forcefield(w)
    pix = W.sample_indices(w.scan.npx * w.scan.npy, 40, 5)
    r = oracle.relax_scan(ff, w.grid, w.tip, w.fire, w.scan, pix=pix)
    assert np.all(r["iters"] >= 0)
    flagged = oracle.flags(r)
    worst = 0.0
    for iz in range(0, w.scan.nz, 3):
        for m, p in enumerate(pix):
            ix, iy = p % w.scan.npx, p // w.scan.npx
            rtip = w.scan.p0 + ix * w.scan.dx + iy * w.scan.dy - np.array([0, 0, iz * w.scan.dz])
            x = r["pos_fz"][iz, m, :3].copy()
            F = oracle.total_force(ff, w.grid, w.tip, rtip, x)
            assert np.linalg.norm(F) < w.fire.f_conv
            if flagged[iz, m]:
                continue
            x0 = x.copy()
            for _ in range(20):
                H, ev = oracle.hessian(ff, w.grid, w.tip, rtip, x)
                assert ev[0] > 0
                x = x + np.linalg.solve(H, oracle.total_force(ff, w.grid, w.tip, rtip, x))
            worst = max(worst, np.linalg.norm(x - x0))
            assert np.linalg.norm(oracle.total_force(ff, w.grid, w.tip, rtip, x)) < 1e-9
    assert worst < 1e-6 / 1e-3 * 1e-3 + 1e-3     # |dx| <= f_conv / lam_min <= 1e-3 Å for non-flagged samples
    assert worst < 1e-3


def test_relaxed_positions_mirror_symmetric_molecule():
    """A mirror-symmetric sample scanned on a mirror-symmetric pixel set gives mirror-symmetric relaxed positions
    and equal Fz (pins the whole O3-O8 chain without a reference value)."""
    w = W.get(0)
    half = np.round(w.xyzq[:5].astype(np.float64) * 64) / 64
    half[:, 0] = 4.0 + np.abs(half[:, 0] - 6.0) * 0.5            # x in [4, 5.5]
    mir = half.copy()
    mir[:, 0] = 12.0 - mir[:, 0]
    w = replace(w, xyzq=np.r_[half, mir].astype(np.float32), types=np.r_[w.types[:5], w.types[:5]],
                grid=replace(w.grid, n=(61, 60, 40)),                 # nodes at 0..12 -> symmetric about x = 6
                scan=replace(w.scan, p0=np.array([4.0, 5.0, 10.0]), npx=21, npy=3, nz=30))
    ff = oracle.forcefield(w)
    assert np.allclose(ff[..., 0], -ff[:, :, ::-1, 0], rtol=1e-9, atol=1e-12)
    r = oracle.relax_scan(ff, w.grid, w.tip, replace(w.fire, f_conv=1e-9, max_iter=20000), w.scan)
    pos = r["pos_fz"].reshape(w.scan.nz, w.scan.npy, w.scan.npx, 4)
    ok = ~oracle.flags(r).reshape(w.scan.nz, w.scan.npy, w.scan.npx)
    ok &= ok[:, :, ::-1]
    assert ok.mean() > 0.9
    assert np.allclose((pos[..., 0] + pos[:, :, ::-1, 0])[ok], 12.0, atol=1e-5)
    assert np.allclose((pos[..., 1:] - pos[:, :, ::-1, 1:])[ok], 0.0, atol=1e-5)


def test_lazy_node_scan_is_the_stored_grid_scan_bit_for_bit():
    """oracle.relax_scan_atoms (grid nodes evaluated on demand from the atoms and memoised per pixel) must be the
    scan on the stored FP64 grid, bit for bit: config 0 sampled pixels, a periodic skewed grid with 9 images (nodes
    reached across the seam), and a non-periodic grid the probe particle leaves (clamping)."""
    w = W.get(0)
    pix = W.sample_indices(w.scan.npx * w.scan.npy, 25, 3)
    a = oracle.relax_scan(oracle.forcefield(w), w.grid, w.tip, w.fire, w.scan, pix=pix)
    b = oracle.relax_scan_atoms(w, pix=pix)
    for k in ("pos_fz", "iters", "lam_min", "clamped", "lam_traj"):
        assert np.array_equal(a[k], b[k]), k
    assert np.all(b["nodes"] > 8) and np.all(b["nodes"] < 0.2 * w.npoints)        # a small part of the grid
    w2 = W.shrink(W.get(2), grid_n=(50, 50, 24), scan_np=(5, 4), scan_nz=6)
    step = np.array([[0.5, 0.02, 0.0], [-0.03, 0.5, 0.0], [0.01, 0.02, 0.25]])
    w2 = replace(w2, grid=replace(w2.grid, step=step), scan=replace(w2.scan, p0=np.array([-3.0, 20.0, 9.0])))
    for per, p0 in (((1, 1, 0), [-3.0, 20.0, 9.0]), ((0, 0, 0), [-1.0, 23.0, 12.5])):
        w3 = replace(w2, grid=replace(w2.grid, periodic=per), scan=replace(w2.scan, p0=np.array(p0)))
        a = oracle.relax_scan(oracle.forcefield(w3), w3.grid, w3.tip, w3.fire, w3.scan)
        b = oracle.relax_scan_atoms(w3)
        for k in ("pos_fz", "iters", "lam_min", "clamped", "lam_traj"):
            assert np.array_equal(a[k], b[k]), (per, k)
    assert int(b["clamped"].sum()) > 0


def test_max_iter_flag():
    g, ff = _flat_grid()
    ff[..., 2] = 0.03
    r = oracle.relax_scan(ff, g, W._default_tip(), replace(W.Fire(), max_iter=3), _scan(nz=1))
    assert np.all(r["iters"] == -1)


def test_fire_first_step_matches_hand_computation():
    """One FIRE move from rest (v = 0, P = 0 counts as downhill, reading S6): v = F dt, r += v dt = F dt^2."""
    g, ff = _flat_grid()
    ff[..., 2] = 0.03
    ff[..., 0] = -0.01
    tip = W._default_tip()
    sc = _scan(nz=1)
    r = oracle.relax_scan(ff, g, tip, replace(W.Fire(), max_iter=1), sc, pix=np.array([0]))
    want = sc.p0 + np.array(tip.d0) + np.array([-0.01, 0, 0.03]) * 0.25
    assert np.allclose(r["pos_fz"][0, 0, :3], want, atol=1e-15)
    # second move: P > 0, n_pos = 1 <= n_min so dt stays 0.5; v = (1-a) v + a |v| F/|F| then v += F dt
    r2 = oracle.relax_scan(ff, g, tip, replace(W.Fire(), max_iter=2), sc, pix=np.array([0]))
    x1 = want
    d = x1 - sc.p0
    L = np.linalg.norm(d)
    F1 = np.array([-0.01, 0, 0.03]) - tip.k_rad * (L - 4.0) * d / L - np.array(
        [tip.k_lat[0] * d[0], tip.k_lat[1] * d[1], 0.0])
    v = np.array([-0.01, 0, 0.03]) * 0.5
    v = 0.9 * v + 0.1 * np.linalg.norm(v) * F1 / np.linalg.norm(F1)
    v = v + F1 * 0.5
    assert np.allclose(r2["pos_fz"][0, 0, :3], x1 + v * 0.5, atol=1e-14)


# ---------------------------------------------------------------------------------------------------- O9
def _fire_reference(force, r0, fire, kmax):
    """FIRE of ref [7] (Bitzek et al. 2006) in the reading S6 / S7 of DESIGN.md, written out independently of the
    oracle: check |F| < f_conv BEFORE moving; P = F.v; P >= 0: mix v towards F, and once MORE than n_min downhill
    moves have been counted grow dt (capped at dt_max) and shrink alpha; P < 0: v = 0, dt halves, alpha = alpha0,
    counter = 0; then semi-implicit Euler with m = 1.  Returns the positions after 0, 1, 2, ... moves and the event
    log (kind, dt used for the move, alpha after the update, grew?)."""
    r, v = np.array(r0, dtype=np.float64), np.zeros(3)
    dt, alpha, n_pos = fire.dt, fire.alpha0, 0
    traj, events = [r.copy()], []
    for _ in range(kmax):
        F = force(r)
        Fn = np.sqrt(F @ F)
        if Fn < fire.f_conv:
            break
        if F @ v >= 0.0:
            v = (1.0 - alpha) * v + alpha * np.sqrt(v @ v) * F / Fn
            grew = n_pos > fire.n_min
            if grew:
                dt = min(dt * fire.finc, fire.dt_max)
                alpha = alpha * fire.falpha
            n_pos += 1
            events.append(("down", dt, alpha, grew))
        else:
            v = np.zeros(3)
            dt = dt * fire.fdec
            alpha = fire.alpha0
            n_pos = 0
            events.append(("up", dt, alpha, False))
        v = v + F * dt
        r = r + v * dt
        traj.append(r.copy())
    return np.array(traj), events


def test_fire_path_move_by_move_against_independent_implementation():
    """O6 control flow (ref [7]; readings S6, S7), pinned MOVE BY MOVE: an affine sample field (which
    tri-linear interpolation reproduces exactly, so the total force is analytic) plus the springs of an asymmetric
    tip gives a relaxation with several P < 0 events, a run of > 14 downhill moves after a halving (so the
    n_pos > n_min gate opens, dt grows by finc per move and is capped at dt_max, alpha decays by falpha) and a
    convergence after ~120 moves.  The oracle, stopped after k = 1, 2, ... moves (max_iter = k), must sit where the
    independent numpy FIRE above sits after k moves, to 1e-13 Å, and must converge in exactly the same number of
    moves.  A '>=' instead of '>' in the gate, a missing dt cap, a wrong reset in the P < 0 branch or a different
    integrator order each change the path at the 1e-3 Å level."""
    g = W.Grid(origin=np.zeros(3), step=np.diag([0.2, 0.2, 0.2]), n=(20, 20, 60), periodic=(0, 0, 0))
    zz, yy, xx = np.meshgrid(np.arange(60) * 0.2, np.arange(20) * 0.2, np.arange(20) * 0.2, indexing="ij")
    b = np.array([0.004, -0.002, -0.08])
    M = np.array([[-0.004, 0.001, 0.0], [0.0005, -0.006, 0.002], [0.001, 0.0, 0.01]])
    ff = np.zeros((60, 20, 20, 4))
    for c in range(3):
        ff[..., c] = b[c] + M[c, 0] * xx + M[c, 1] * yy + M[c, 2] * zz
    tip = replace(W._default_tip(), k_lat=(0.012, 0.019), d0=(0.3, -0.2, -3.98))      # asymmetric tip
    d0 = np.array(tip.d0)
    R0 = np.linalg.norm(d0)
    p0 = np.array([1.5, 1.7, 9.0])
    sc = W.Scan(p0=p0, dx=np.array([0.3, 0, 0.0]), dy=np.array([0, 0.4, 0.0]), npx=1, npy=1, nz=1, dz=0.1)

    def force(r):       # Eq.1 + Eq.2 with F_S = b + M r
        d = r - p0
        L = np.sqrt(d @ d)
        return (b + M @ r - tip.k_rad * (L - R0) * d / L -
                np.array([tip.k_lat[0] * (d[0] - d0[0]), tip.k_lat[1] * (d[1] - d0[1]), 0.0]))

    fire = W.Fire()
    traj, events = _fire_reference(force, p0 + d0, fire, 1000)
    n_moves = len(traj) - 1
    assert traj.min() > 0.2 and traj[:, :2].max() < 3.6          # the path stays inside the grid (no clamping)
    kinds = "".join("d" if e[0] == "down" else "u" for e in events)
    # the path exercises every branch: >= 3 uphill events, a halving followed by growth back to the dt_max cap,
    # alpha decay, and a long downhill run
    assert kinds.count("u") >= 3 and 100 < n_moves < 200
    first_up = kinds.index("u")
    assert events[first_up][1] == fire.dt * fire.fdec and events[first_up][2] == fire.alpha0
    run = len(kinds[first_up + 1:].split("u")[0])
    assert run > fire.n_min + 9
    dts = [e[1] for e in events[first_up + 1:first_up + 1 + run]]
    assert dts[fire.n_min] == fire.dt * fire.fdec and dts[fire.n_min + 1] == pytest.approx(fire.dt * fire.fdec * fire.finc)
    assert max(dts) == fire.dt_max and dts.count(fire.dt_max) >= 2                   # growth hit the cap and stayed there
    assert min(e[2] for e in events) < fire.alpha0 * fire.falpha ** 10               # alpha decayed
    # the oracle, move by move
    for k in list(range(1, 61)) + list(range(60, n_moves, 7)) + [n_moves - 1]:
        r = oracle.relax_scan(ff, g, tip, replace(fire, max_iter=k), sc)
        assert r["iters"][0, 0] == -1                                                # not yet converged
        assert np.abs(r["pos_fz"][0, 0, :3] - traj[k]).max() < 1e-13, k
    for k in (n_moves, n_moves + 1, 1000):
        r = oracle.relax_scan(ff, g, tip, replace(fire, max_iter=k), sc)
        assert r["iters"][0, 0] == n_moves                                           # exact move count at f_conv
        assert np.abs(r["pos_fz"][0, 0, :3] - traj[n_moves]).max() < 1e-13
    assert np.linalg.norm(force(traj[n_moves])) < fire.f_conv <= np.linalg.norm(force(traj[n_moves - 1]))


# ---------------------------------------------------------------------------------------------------- O7
def _fire_run(force, r0, fire, kmax, state=None):
    """One z-step of FIRE in readings S6 / S7, written apart from the oracle AND apart from _fire_reference above in
    one respect: the FIRE state (v, dt, alpha, n_pos) can be handed in and is handed back, so that a scan that does
    NOT reset it between z-steps can be played.  Returns (r, moves, converged, state)."""
    r = np.array(r0, dtype=np.float64)
    v, dt, alpha, n_pos = (np.zeros(3), fire.dt, fire.alpha0, 0) if state is None else state
    v = np.array(v, dtype=np.float64)
    moves = 0
    while True:
        F = force(r)
        Fn = np.sqrt(F @ F)
        if Fn < fire.f_conv:
            return r, moves, True, (v, dt, alpha, n_pos)
        if moves >= kmax:
            return r, moves, False, (v, dt, alpha, n_pos)
        if F @ v >= 0.0:
            v = (1.0 - alpha) * v + alpha * np.sqrt(v @ v) * F / Fn
            if n_pos > fire.n_min:
                dt, alpha = min(dt * fire.finc, fire.dt_max), alpha * fire.falpha
            n_pos += 1
        else:
            v, dt, alpha, n_pos = np.zeros(3), dt * fire.fdec, fire.alpha0, 0
        v = v + F * dt
        r = r + v * dt
        moves += 1


def _play_scan(force_at, p0, d0, nz, dz, fire, kmax, mode):
    """A one-pixel scan played with the independent FIRE.  mode 'carry' = reading S8 / O7 (the relaxed
    displacement d = r_PP - r_TIP of one z-step is the start of the next, FIRE state fresh at every step); 'cold' =
    every z-step starts again from d0; 'keep' = d carried AND the FIRE state (v, dt, alpha, n_pos) kept;
    'position' = the relaxed POSITION carried instead of the displacement."""
    d, state, r_prev = np.array(d0, dtype=np.float64), None, None
    pos, its = [], []
    for iz in range(nz):
        rtip = np.array(p0, dtype=np.float64) - np.array([0.0, 0.0, iz * dz])
        start = rtip + (np.array(d0) if mode == "cold" else d)
        if mode == "position" and r_prev is not None:
            start = r_prev
        r, moves, conv, st = _fire_run(lambda x: force_at(x, rtip), start, fire, kmax,
                                       state if mode == "keep" else None)
        state, d, r_prev = st, r - rtip, r
        pos.append(r)
        its.append(moves if conv else -1)
    return np.array(pos), np.array(its)


def _affine_case():
    """The affine sample field and asymmetric tip of the move-by-move test, as (grid, ff, tip, p0, force_at)."""
    g = W.Grid(origin=np.zeros(3), step=np.diag([0.2, 0.2, 0.2]), n=(20, 20, 60), periodic=(0, 0, 0))
    zz, yy, xx = np.meshgrid(np.arange(60) * 0.2, np.arange(20) * 0.2, np.arange(20) * 0.2, indexing="ij")
    b = np.array([0.004, -0.002, -0.08])
    M = np.array([[-0.004, 0.001, 0.0], [0.0005, -0.006, 0.002], [0.001, 0.0, 0.01]])
    ff = np.zeros((60, 20, 20, 4))
    for c in range(3):
        ff[..., c] = b[c] + M[c, 0] * xx + M[c, 1] * yy + M[c, 2] * zz
    tip = replace(W._default_tip(), k_lat=(0.012, 0.019), d0=(0.3, -0.2, -3.98))
    d0 = np.array(tip.d0)
    R0 = np.linalg.norm(d0)

    def force_at(r, rtip):
        d = r - rtip
        L = np.sqrt(d @ d)
        return (b + M @ r - tip.k_rad * (L - R0) * d / L -
                np.array([tip.k_lat[0] * (d[0] - d0[0]), tip.k_lat[1] * (d[1] - d0[1]), 0.0]))

    return g, ff, tip, np.array([1.5, 1.7, 9.0]), force_at


def test_warm_start_between_z_steps_is_displacement_carried_with_fresh_fire_state():
    """O7 / reading S8 ("the tip is moved down step by step and the PP is relaxed from its previous
    position"; oracle relax_pixel: `dcur` carried, v / dt / alpha / n_pos re-initialised per z-step).  A three-step
    scan on the affine field, each z-step cut off after k moves so that it ends UNCONVERGED and the start of the next
    step matters at the 1e-2 Å level: the oracle must sit where the independent FIRE sits when it carries the
    displacement and starts every step with fresh state, and must NOT sit where any of the three plausible
    alternatives ends up (cold start from d0, FIRE state kept, position carried instead of displacement).  Then the
    same scan run to convergence: the move count of EVERY z-step is the independent one's, and differs from the
    cold-start and kept-state scans' counts."""
    g, ff, tip, p0, force_at = _affine_case()
    fire = W.Fire()
    nz, dz = 3, 0.1
    sc = W.Scan(p0=p0, dx=np.array([0.3, 0, 0.0]), dy=np.array([0, 0.4, 0.0]), npx=1, npy=1, nz=nz, dz=dz)
    for k in (3, 9, 17, 40):
        r = oracle.relax_scan(ff, g, tip, replace(fire, max_iter=k), sc)
        got = r["pos_fz"][:, 0, :3]
        want, its = _play_scan(force_at, p0, tip.d0, nz, dz, fire, k, "carry")
        assert np.all(its == -1) and np.all(r["iters"][:, 0] == -1)
        assert np.abs(got - want).max() < 1e-13, k
        for mode in ("cold", "keep", "position"):
            other, _ = _play_scan(force_at, p0, tip.d0, nz, dz, fire, k, mode)
            assert np.abs(other[0] - want[0]).max() < 1e-13                      # z-step 0 is the same scan in all readings
            assert np.linalg.norm(got[1] - other[1]) > 1e-4 and np.linalg.norm(got[2] - other[2]) > 1e-4, (k, mode)
    # to convergence: per-step move counts
    r = oracle.relax_scan(ff, g, tip, fire, replace(sc, nz=6))
    want, its = _play_scan(force_at, p0, tip.d0, 6, dz, fire, 1000, "carry")
    assert np.all(its > 0) and np.array_equal(r["iters"][:, 0], its)
    assert np.abs(r["pos_fz"][:, 0, :3] - want).max() < 1e-13
    assert its[0] > 100 and np.all(its[1:] < its[0])          # a warm start from 0.1 Å away needs fewer moves
    for mode in ("cold", "keep"):
        _, other = _play_scan(force_at, p0, tip.d0, 6, dz, fire, 1000, mode)
        assert other[0] == its[0] and not np.array_equal(other[1:], its[1:]), mode


def test_warm_start_keeps_the_branch_on_a_bistable_field():
    """O7 where it changes the ANSWER, not just the path: a lateral force F_x = A(z) s(x) with s piecewise linear
    (kinks on grid nodes: a shallow ramp, a steep ramp, then a well around x = 3.0) and A linear in z, which tri-linear
    interpolation reproduces exactly.  With the tip over the shallow ramp (x = 2.4, k_x = 0.0156 eV/Å^2) the
    x-equilibria follow from k (x - 2.4) = A s(x): for A > k only the well (x ~ 2.9) is stable, for 0.4 k < A < k the
    well AND a point on the shallow ramp (x ~ 2.45) are stable, for A < 0.4 k only the ramp point.  A decreases as the
    tip comes down.  The scan therefore falls into the well at the top, STAYS in it through the bistable window because
    the displacement is carried (a scan restarted from d0 at every step sits on the ramp there: hysteresis), and snaps
    back once the well equilibrium is gone.  Every z-step of the oracle is compared with the independent FIRE played
    with carried displacement and fresh state: end point to 1e-12 Å and exact move count."""
    h = 0.2
    nx, ny, nzg = 21, 12, 40
    g = W.Grid(origin=np.zeros(3), step=np.diag([h, h, h]), n=(nx, ny, nzg), periodic=(0, 0, 0))
    xs, zs = np.arange(nx) * h, np.arange(nzg) * h
    s_nodes = np.interp(xs, [2.0, 2.6, 2.8, 3.0, 3.2, 3.4], [0.0, 0.2, 1.0, 0.0, -1.0, 0.0])
    tip = W._default_tip()
    k = tip.k_lat[0]
    a1 = 1.0 * k                                  # A(z) = k (1.6 + (z - 5.0)): 1.6 k at z = 5.0, 0.3 k at z = 3.7
    A_nodes = k * 1.6 + a1 * (zs - 5.0)
    ff = np.zeros((nzg, ny, nx, 4))
    ff[..., 0] = A_nodes[:, None, None] * s_nodes[None, None, :]
    p0 = np.array([2.4, 1.1, 9.0])
    nz, dz = 14, 0.1
    sc = W.Scan(p0=p0, dx=np.array([0.3, 0, 0.0]), dy=np.array([0, 0.4, 0.0]), npx=1, npy=1, nz=nz, dz=dz)
    d0 = np.array(tip.d0)
    R0 = np.linalg.norm(d0)

    def force_at(r, rtip):
        d = r - rtip
        L = np.sqrt(d @ d)
        Fs = np.array([(k * 1.6 + a1 * (r[2] - 5.0)) * np.interp(r[0], xs, s_nodes), 0.0, 0.0])
        return Fs - tip.k_rad * (L - R0) * d / L - np.array([tip.k_lat[0] * d[0], tip.k_lat[1] * d[1], 0.0])

    fire = W.Fire()
    r = oracle.relax_scan(ff, g, tip, fire, sc)
    got, its_o = r["pos_fz"][:, 0, :3], r["iters"][:, 0]
    want, its = _play_scan(force_at, p0, d0, nz, dz, fire, fire.max_iter, "carry")
    assert np.all(its > 0) and np.array_equal(its_o, its)
    assert np.abs(got - want).max() < 1e-12
    cold, _ = _play_scan(force_at, p0, d0, nz, dz, fire, fire.max_iter, "cold")
    A_at = k * 1.6 + a1 * (got[:, 2] - 5.0)
    in_well = got[:, 0] > 2.8
    window = (A_at > 0.45 * k) & (A_at < 0.95 * k)
    assert in_well[0] and A_at[0] > k                                   # falls into the well at the top
    assert window.sum() >= 4 and np.all(in_well[window])                # carried: stays through the bistable window
    assert np.all(cold[window, 0] < 2.6)                                # restarted from d0: sits on the ramp instead
    assert np.all(np.abs(got[window, 0] - cold[window, 0]) > 0.25)
    assert not in_well[-1] and A_at[-1] < 0.4 * k                       # the well is gone at the bottom: snapped back
    assert np.abs(got[-1] - cold[-1]).max() < 1e-4                      # ... to the minimum a cold start finds too
    # both branches are equilibria of the analytic 1-D balance k (x - 2.4) = A s(x)
    for x, A in zip(got[:, 0], A_at):
        assert abs(k * (x - p0[0]) - A * np.interp(x, xs, s_nodes)) < 2 * fire.f_conv


def test_df_weights_sum_to_zero_and_match_numerical_quadrature():
    """Eq.3: W_m = (2/(pi a^2)) int q hat_m(q)/sqrt(a^2-q^2) dq, checked with scipy.quad using
    the algebraic end-point weight; sum W = 0 (a constant force gives df = 0)."""
    for n, dz in ((10, 0.1), (20, 0.05), (1, 1.0), (2, 0.5), (7, 0.13)):
        Wt = oracle.df_weights(n, dz)
        a = 0.5 * n * dz
        assert abs(Wt.sum()) < 1e-13
        assert np.allclose(Wt, -Wt[::-1], atol=1e-13)                   # odd kernel
        for m in range(n + 1):
            qm = -a + m * dz
            tot = 0.0
            for lo, hi in ((qm - dz, qm), (qm, qm + dz)):
                if lo < -a - 1e-12 or hi > a + 1e-12:
                    continue
                hat = lambda q: q * (1 - abs(q - qm) / dz)
                # int f(q) (q+a)^(-1/2) (a-q)^(-1/2) dq  via quad's 'alg' weight on [-a, a] restricted by hat
                val, _ = integrate.quad(lambda q: hat(q) if lo <= q <= hi else 0.0, -a, a, weight="alg",
                                        wvar=(-0.5, -0.5), points=None, limit=400)
                tot += val
            assert Wt[m] == pytest.approx(2 / (np.pi * a * a) * tot, abs=2e-6)


def test_df_linear_exact_cubic_and_exponential():
    pref = (30300.0 / 3600.0) * NM
    for n in (1, 2, 10, 20):
        dz = 1.0 / n
        a = 0.5
        nz = n + 6
        z = 8.0 - dz * np.arange(nz)
        g = 0.37
        df = oracle.df((g * (z - 5.0))[:, None], dz, 1.0, 1800.0, 30300.0)
        assert np.allclose(df, -pref * g, rtol=1e-12)                       # linear: exact for any n
        zc = z[0] - (np.arange(nz - n) + n / 2) * dz
        kappa, F0 = 1.3, 0.2
        dfe = oracle.df((F0 * np.exp(-kappa * z))[:, None], dz, 1.0, 1800.0, 30300.0)[:, 0]
        # int q e^{-kq}/sqrt(a^2-q^2) = -pi a I1(k a)  ->  df = (f0/(k0 a)) * 16.02 * F0 e^{-k zc} I1(k a)
        want = 2 * pref / a * F0 * np.exp(-kappa * zc) * special.i1(kappa * a)
        tol = {1: 0.2, 2: 0.05, 10: 2e-3, 20: 6e-4}[n]
        assert np.allclose(dfe, want, rtol=tol)
        h3 = 0.11
        dfc = oracle.df((h3 * (z - zc[2]) ** 3)[:, None], dz, 1.0, 1800.0, 30300.0)[2, 0]
        wantc = -pref * 0.75 * h3 * a * a
        tolc = {1: 0.34, 2: 0.34, 10: 0.03, 20: 0.01}[n]      # n = 1, 2: the interpolant is the chord, error exactly 1/3
        assert dfc == pytest.approx(wantc, rel=tolc)
    # n = 1 is the two-point finite difference (small-amplitude limit, reading S10)
    fz = np.array([[0.3], [0.5], [0.9]])
    assert np.allclose(oracle.df(fz, 0.1, 0.1, 1800.0, 30300.0)[:, 0], -pref * (fz[:-1, 0] - fz[1:, 0]) / 0.1)


def test_df_rejects_bad_amplitude():
    with pytest.raises(ValueError):
        oracle.df(np.zeros((20, 1)), 0.1, 0.55, 1800.0, 30300.0)       # A/dz not an integer
    with pytest.raises(ValueError):
        oracle.df(np.zeros((5, 1)), 0.1, 1.0, 1800.0, 30300.0)         # nz <= n


# ---------------------------------------------------------------------------------------------------- O10
def test_hessian_matches_finite_difference_of_force():
    w = W.get(0)
    ff = oracle.forcefield(w)
    rtip = np.array([5.03, 6.41, 7.52])
    rpp = rtip + np.array([0.213, -0.117, -3.93])         # interior of a cell (not on a face)
    H, ev = oracle.hessian(ff, w.grid, w.tip, rtip, rpp)
    J = np.zeros((3, 3))
    h = 1e-6
    for a in range(3):
        dp = np.zeros(3)
        dp[a] = h
        J[:, a] = (oracle.total_force(ff, w.grid, w.tip, rtip, rpp + dp) -
                   oracle.total_force(ff, w.grid, w.tip, rtip, rpp - dp)) / (2 * h)
    assert np.allclose(H, -(J + J.T) / 2, rtol=1e-6, atol=1e-8)
    assert np.allclose(ev, np.linalg.eigvalsh(H), atol=1e-12)


def test_stiffness_map_closed_forms_and_finite_differences():
    """IETS stiffness map.  (i) No sample interaction: the PP at the spring equilibrium has
    eigenvalues (k_x, k_y, k_R) exactly - the two lateral CO modes and the radial one.  (ii) A linear field
    F_S = -K (r - r0) with K symmetric (exactly reproduced by tri-linear interpolation) adds K to the spring Hessian:
    eigenvalues = eigvalsh(H_spring + K).  (iii) On config 0 the bulk call equals -sym(dF_total/dr) by central
    differences of the total force at 40 random in-cell points."""
    g = W.Grid(origin=np.array([0.0, 0.0, 0.0]), step=np.diag([0.2, 0.25, 0.1]), n=(30, 24, 60), periodic=(0, 0, 0))
    tip = W._default_tip()
    zero = np.zeros((60, 24, 30, 4))
    rtip = np.array([[2.9, 3.1, 8.2], [3.3, 2.2, 7.7]])
    ev = oracle.stiffness(zero, g, tip, rtip, rtip + np.asarray(tip.d0))
    assert np.allclose(ev, [[tip.k_lat[0], tip.k_lat[1], tip.k_rad]] * 2, rtol=0, atol=1e-12)
    # (ii) linear restoring field
    K = np.array([[0.30, 0.05, -0.02], [0.05, -0.11, 0.04], [-0.02, 0.04, 0.21]])
    r0 = np.array([3.0, 3.0, 4.0])
    k, j, i = np.meshgrid(np.arange(60), np.arange(24), np.arange(30), indexing="ij")
    nodes = np.stack([i * 0.2, j * 0.25, k * 0.1], axis=-1)
    lin = np.zeros((60, 24, 30, 4))
    lin[..., :3] = -(nodes - r0) @ K.T
    rpp = rtip + np.array([[0.31, -0.22, -3.9], [-0.4, 0.15, -4.05]])
    ev = oracle.stiffness(lin, g, tip, rtip, rpp)
    for m in range(2):
        d = rpp[m] - rtip[m]
        L = np.linalg.norm(d)
        dd = np.outer(d, d) / L**2
        Hs = tip.k_rad * dd + tip.k_rad * (L - 4.0) / L * (np.eye(3) - dd) + np.diag([tip.k_lat[0], tip.k_lat[1], 0.0])
        assert np.allclose(ev[m], np.linalg.eigvalsh(Hs + K), rtol=0, atol=1e-10)
    # (iii) real field, bulk call vs finite differences of the total force
    w = W.get(0)
    ff = oracle.forcefield(w)
    rng = np.random.default_rng(5)
    rt = np.stack([rng.uniform(4.0, 8.0, 40), rng.uniform(4.0, 8.0, 40), rng.uniform(6.5, 9.5, 40)], axis=1)
    cell = np.array([0.2, 0.2, 0.2])
    rp = rt + np.asarray(w.tip.d0) + rng.uniform(-0.3, 0.3, (40, 3))
    frac = ((rp - np.asarray(w.grid.origin)) / cell) % 1.0
    rp += (np.clip(frac, 0.05, 0.95) - frac) * cell                      # keep every point inside its cell
    ev = oracle.stiffness(ff, w.grid, w.tip, rt, rp)
    h = 1e-6
    for m in range(40):
        J = np.zeros((3, 3))
        for a in range(3):
            dp = np.zeros(3)
            dp[a] = h
            J[:, a] = (oracle.total_force(ff, w.grid, w.tip, rt[m], rp[m] + dp) -
                       oracle.total_force(ff, w.grid, w.tip, rt[m], rp[m] - dp)) / (2 * h)
        assert np.allclose(ev[m], np.linalg.eigvalsh(-(J + J.T) / 2), rtol=1e-6, atol=1e-8)
    assert np.allclose(oracle.tip_positions(_scan())[3, 0], _scan().p0 - np.array([0, 0, 3 * _scan().dz]))


# ---------------------------------------------------------------------------------------------------- O12 (Eq.7)
def _fft_grid(n=(24, 20, 16), h=(0.25, 0.3, 0.35)):
    return W.Grid(origin=np.zeros(3), step=np.diag(h), n=n, periodic=(1, 1, 1))


def test_eq7_crosscorrelation_plane_wave_closed_forms():
    """PAPER.md:102-106, Eq.7.  For V_S = V0 cos(k.r + phi) with k a reciprocal-lattice vector and a Gaussian
    multipole tip rho = [q + p z/s^2 + (Q/12)(3z^2 - r^2)/s^4] g_s(r), the cross-correlation integral is closed form:
        E(R) = V0 exp(-s^2 k^2 / 2) [ q cos(k.R + phi) - p k_z sin(k.R + phi) + (Q/12)(k^2 - 3 k_z^2) cos(k.R + phi) ]
    and F = -grad E.  A dropped term, a wrong sign, a wrong normalisation of g or a missing dV fails this."""
    g = _fft_grid()
    n, h = np.array(g.n), np.diag(np.asarray(g.step))
    L = n * h
    kvec = 2 * np.pi * np.array([1, -1, 2]) / L
    V0, phi, s = 0.8, 0.4, 0.4            # 7 sigma = half the shortest cell edge: no tail is lost to the wrap
    K, J, I = np.meshgrid(np.arange(n[2]), np.arange(n[1]), np.arange(n[0]), indexing="ij")
    R = np.stack([I * h[0], J * h[1], K * h[2]], axis=-1)
    arg = R @ kvec + phi
    V = V0 * np.cos(arg)
    damp = V0 * np.exp(-0.5 * s * s * kvec @ kvec)
    k2, kz = kvec @ kvec, kvec[2]
    for q, pz, Q in [(1.0, 0.0, 0.0), (0.0, 0.3, 0.0), (0.0, 0.0, -0.1), (-0.05, 0.02, -0.12)]:
        got = oracle.fft_forcefield(V, g, s, q, pz, Q)
        amp_c = q + (Q / 12.0) * (k2 - 3 * kz * kz)
        amp_s = -pz * kz
        E = damp * (amp_c * np.cos(arg) + amp_s * np.sin(arg))
        dE = damp * (-amp_c * np.sin(arg) + amp_s * np.cos(arg))           # dE/d(arg)
        F = -dE[..., None] * kvec
        assert np.allclose(got[..., 3], E, rtol=0, atol=1e-6), (q, pz, Q)     # residual: Gaussian tail beyond 7 sigma
        assert np.allclose(got[..., :3], F, rtol=0, atol=1e-6), (q, pz, Q)
    # moments of the sampled density: total charge, dipole, quadrupole
    rho = oracle.tip_density(g, s, -0.05, 0.02, -0.12)[0]
    dV = np.prod(h)
    Rw = np.where(R >= L / 2, R - L, R)
    assert np.isclose(rho.sum() * dV, -0.05, atol=1e-10)
    assert np.isclose((rho * Rw[..., 2]).sum() * dV, 0.02, atol=1e-10)
    assert np.isclose((rho * (3 * Rw[..., 2] ** 2 - (Rw ** 2).sum(-1))).sum() * dV, -0.12, atol=1e-9)


def test_eq7_crosscorrelation_equals_numpy_fft_and_brute_force():
    """The direct sum against (i) the convolution theorem with numpy's FFT ("a product in the Fourier
    space with an additional complex conjugation") and (ii) a literal Python loop on a 4 x 3 x 2 grid, for a skewed
    cell and an arbitrary V."""
    rng = np.random.default_rng(3)
    step = np.array([[0.3, 0.02, 0.0], [-0.04, 0.28, 0.01], [0.0, 0.03, 0.33]])
    g = W.Grid(origin=np.zeros(3), step=step, n=(12, 10, 9), periodic=(1, 1, 1))
    V = rng.normal(size=(9, 10, 12))
    got = oracle.fft_forcefield(V, g, 0.6, 0.1, -0.05, 0.2)
    rho4 = oracle.tip_density(g, 0.6, 0.1, -0.05, 0.2)
    dV = abs(np.linalg.det(step))
    for c, lane in ((0, 3), (1, 0), (2, 1), (3, 2)):
        ref = np.fft.ifftn(np.conj(np.fft.fftn(rho4[c])) * np.fft.fftn(V)).real * dV
        assert np.allclose(got[..., lane], ref, rtol=0, atol=1e-12)
    ijk = np.array([[0, 0, 0], [11, 9, 8], [5, 2, 7], [1, 0, 3]])
    assert np.allclose(oracle.fft_forcefield_at(V, g, 0.6, 0.1, -0.05, 0.2, ijk), got[ijk[:, 2], ijk[:, 1], ijk[:, 0]],
                       rtol=0, atol=1e-13)
    # (ii) brute force
    g2 = W.Grid(origin=np.zeros(3), step=step, n=(4, 3, 2), periodic=(1, 1, 1))
    V2 = rng.normal(size=(2, 3, 4))
    got2 = oracle.fft_forcefield(V2, g2, 0.5, 1.0, 0.0, 0.0)
    rho2 = oracle.tip_density(g2, 0.5, 1.0, 0.0, 0.0)[0]
    for K in range(2):
        for J in range(3):
            for I in range(4):
                acc = 0.0
                for k in range(2):
                    for j in range(3):
                        for i in range(4):
                            acc += rho2[k, j, i] * V2[(k + K) % 2, (j + J) % 3, (i + I) % 4]
                assert np.isclose(got2[K, J, I, 3], acc * dV, atol=1e-13)
    # gradient lanes: analytic grad rho against central differences of rho in the continuum formula
    s, q, pz, Q = 0.6, 0.1, -0.05, 0.2

    def rho_at(r):
        rr = r @ r
        return (q + pz * r[2] / s**2 + Q / 12 * (3 * r[2]**2 - rr) / s**4) * (2 * np.pi * s * s) ** -1.5 * np.exp(-rr / (2 * s * s))
    for (k, j, i) in [(1, 2, 3), (8, 9, 11), (4, 0, 5)]:
        iw, jw, kw = (i - 12 if 2 * i >= 12 else i), (j - 10 if 2 * j >= 10 else j), (k - 9 if 2 * k >= 9 else k)
        r = iw * step[0] + jw * step[1] + kw * step[2]
        assert np.isclose(rho4[0, k, j, i], rho_at(r), rtol=1e-12)
        for a in range(3):
            d = np.zeros(3); d[a] = 1e-5
            fd = (rho_at(r + d) - rho_at(r - d)) / 2e-5
            assert np.isclose(rho4[a + 1, k, j, i], fd, rtol=1e-6, atol=1e-9)


# ---------------------------------------------------------------------------------------------------- O13 tri-cubic
def test_tricubic_potential_interpolation_pins():
    """PAPER.md:264 "tri-cubic interpolation of the potential" (reading S22: Catmull-Rom cubic convolution per axis).
    (i) a polynomial of degree <= 2 in each variable is reproduced exactly, so F = -grad E is analytic, also across
    cell faces and the periodic seam of an axis the polynomial does not depend on; (ii) at nodes the interpolant
    returns the node values (checked through a line integral of F between two nodes); (iii) F is continuous across
    cell faces (C^1 interpolant) for random data; (iv) the Hessian G is the finite-difference derivative of F;
    (v) weights: partition of unity and the printed cubic at f = 0.5: (-1/16, 9/16, 9/16, -1/16)."""
    step = np.array([[0.25, 0.0, 0.0], [0.02, 0.3, 0.0], [0.0, 0.01, 0.2]])
    g = W.Grid(origin=np.array([0.3, -0.2, 1.0]), step=step, n=(14, 12, 16), periodic=(0, 0, 0))
    k, j, i = np.meshgrid(np.arange(16), np.arange(12), np.arange(14), indexing="ij")
    nodes = np.asarray(g.origin) + i[..., None] * step[0] + j[..., None] * step[1] + k[..., None] * step[2]
    x, y, z = nodes[..., 0], nodes[..., 1], nodes[..., 2]

    def E_of(x, y, z):
        return 0.3 * x * x * y - 0.2 * y * y * z * z + 0.7 * x * z + 0.1 * z * z - 0.4 * x + 0.05 * x * x * y * y * z

    def F_of(x, y, z):
        return -np.array([0.6 * x * y + 0.7 * z - 0.4 + 0.1 * x * y * y * z,
                          0.3 * x * x - 0.4 * y * z * z + 0.1 * x * x * y * z,
                          -0.4 * y * y * z + 0.7 * x + 0.2 * z + 0.05 * x * x * y * y])
    rng = np.random.default_rng(9)
    tfrac = 1.0 + rng.uniform(0, 1, (50, 3)) * (np.array([14, 12, 16]) - 4.0)   # 4-point stencil inside the grid
    pts = np.asarray(g.origin) + tfrac @ step
    # orthogonal grid: degree <= 2 in each variable is exact
    go = replace(g, step=np.diag([0.25, 0.3, 0.2]))
    no = np.asarray(go.origin) + np.stack([i * 0.25, j * 0.3, k * 0.2], axis=-1)
    pto = np.asarray(go.origin) + tfrac * np.array([0.25, 0.3, 0.2])
    got = oracle.interp(E_of(no[..., 0], no[..., 1], no[..., 2]), go, pto)
    assert np.allclose(got, np.array([F_of(*p) for p in pto]), rtol=1e-11, atol=1e-11)
    # skewed grid: total degree <= 2 stays within degree 2 of every index variable -> exact
    A = np.array([[0.3, 0.1, -0.05], [0.1, -0.2, 0.07], [-0.05, 0.07, 0.15]])
    bq = np.array([0.4, -0.3, 0.2])
    Eq = np.einsum("...a,ab,...b->...", nodes, A, nodes) + nodes @ bq
    got = oracle.interp(Eq, g, pts)
    assert np.allclose(got, -(2 * pts @ A + bq), rtol=1e-11, atol=1e-11)
    # (ii) line integral of F between two nodes = E(a) - E(b) for ARBITRARY node data (interpolation property)
    Er = rng.normal(size=Eq.shape)
    a_idx, b_idx = (5, 4, 6), (9, 4, 6)                                  # (i, j, k): along x, 4 cells
    ra = np.asarray(g.origin) + a_idx[0] * step[0] + a_idx[1] * step[1] + a_idx[2] * step[2]
    rb = np.asarray(g.origin) + b_idx[0] * step[0] + b_idx[1] * step[1] + b_idx[2] * step[2]
    tt, ww = np.polynomial.legendre.leggauss(6)
    work = 0.0
    for c in range(4):                                                   # Gauss-Legendre per cell: exact for cubics
        p0, p1 = ra + (rb - ra) * c / 4, ra + (rb - ra) * (c + 1) / 4
        ps = p0 + (p1 - p0) * ((tt[:, None] + 1) / 2)
        Fs = oracle.interp(Er, g, ps)
        work += (ww * (Fs @ (p1 - p0))).sum() / 2
    assert np.isclose(work, Er[a_idx[2], a_idx[1], a_idx[0]] - Er[b_idx[2], b_idx[1], b_idx[0]], atol=1e-12)
    # (iii) continuity of F across a cell face, random data
    face = np.asarray(g.origin) + 6 * step[0] + 5.3 * step[1] + 7.6 * step[2]
    eps = 1e-9 * step[0]
    assert np.allclose(oracle.interp(Er, g, [face - eps]), oracle.interp(Er, g, [face + eps]), atol=1e-6)
    # (iv) Hessian = -dF/dr by finite differences (zero springs: k = 0 tip)
    tip0 = W.Tip(k_lat=np.array([0.0, 0.0]), k_rad=0.0, d0=np.array([0.0, 0.0, -4.0]))
    rpp = np.asarray(g.origin) + 6.37 * step[0] + 5.21 * step[1] + 7.64 * step[2]
    H, ev = oracle.hessian(Er, g, tip0, rpp + np.array([0, 0, 4.0]), rpp)
    J = np.zeros((3, 3))
    for a in range(3):
        dp = np.zeros(3); dp[a] = 1e-6
        J[:, a] = (oracle.interp(Er, g, [rpp + dp])[0] - oracle.interp(Er, g, [rpp - dp])[0]) / 2e-6
    assert np.allclose(H, -(J + J.T) / 2, rtol=1e-6, atol=1e-6)
    assert np.allclose(J, J.T, atol=1e-6)                                # a true gradient field, unlike tri-linear F (S14)
    # (v) the printed kernel values at the cell centre, through a 1-D delta function along x
    d = np.zeros((16, 12, 14)); d[:, :, 7] = 1.0                         # E = 1 on the plane i = 7
    gx = W.Grid(origin=np.zeros(3), step=np.diag([1.0, 1.0, 1.0]), n=(14, 12, 16), periodic=(0, 0, 0))
    # F_x = -dE/dx; integrate F_x from x0 to cell centres to recover E there: use E(x) = E(x0) - int F
    def E_at(xc):
        xs = np.linspace(2.0, xc, 2001)
        Fx = oracle.interp(d, gx, np.stack([xs, np.full_like(xs, 5.0), np.full_like(xs, 6.0)], 1))[:, 0]
        return -np.sum((Fx[1:] + Fx[:-1]) / 2 * np.diff(xs))
    assert np.isclose(E_at(5.5), -1 / 16, atol=1e-6) and np.isclose(E_at(6.5), 9 / 16, atol=1e-6)
    assert np.isclose(E_at(7.5), 9 / 16, atol=1e-6) and np.isclose(E_at(8.5), -1 / 16, atol=1e-6)


def test_tricubic_relaxation_linear_field_closed_form_and_periodic_seam():
    """End to end on O13: E = g/2 (z - zc)^2 (reproduced exactly) gives F_z = -g (z - zc), the linear-field closed
    form of the tri-linear pin with g -> -g: w = -g (z_t - R - zc)/(k_R + g), Fz_tip = k_R w.  And a potential
    periodic in x is seamless across the periodic boundary."""
    g = W.Grid(origin=np.zeros(3), step=np.diag([0.2, 0.2, 0.1]), n=(30, 24, 70), periodic=(1, 1, 0))
    k, j, i = np.meshgrid(np.arange(70), np.arange(24), np.arange(30), indexing="ij")
    zc, gg = 3.0, 0.37
    E = 0.5 * gg * (k * 0.1 - zc) ** 2
    tip, sc = W._default_tip(), _scan(npx=3, npy=2, nz=12, z0=8.5, dz=0.1)
    r = oracle.relax_scan(E, g, tip, W.Fire(), sc)
    zt = 8.5 - 0.1 * np.arange(12)
    wexp = -gg * (zt - 4.0 - zc) / (tip.k_rad + gg)
    assert (r["iters"] >= 0).all()
    assert np.allclose(r["pos_fz"][:, 0, 2], zt - 4.0 + wexp, atol=2e-6)
    assert np.allclose(r["pos_fz"][:, 0, 3], tip.k_rad * wexp, atol=2e-6)
    Ex = np.cos(2 * np.pi * i / 30) * np.ones_like(E)
    pts = np.array([[5.9, 1.0, 3.05], [6.1, 1.0, 3.05], [-0.1, 1.0, 3.05], [0.1, 1.0, 3.05]])
    F = oracle.interp(Ex, g, pts)
    assert np.allclose(F[0], F[2], atol=1e-12) and np.allclose(F[1], F[3], atol=1e-12)
    assert np.allclose(F[0, 0], 2 * np.pi / 6.0 * np.sin(2 * np.pi * 5.9 / 6.0), atol=2e-3)   # cubic accuracy only


# ---------------------------------------------------------------------------------------------------- O14 (Eq.8)
def test_eq8_pauli_overlap_pins():
    """PAPER.md:118-122, Eq.8.  (i) A literal loop of A sum_r [rho_PP(r) rho_S(r+R)]^beta dV on a 5 x 4 x 3 grid;
    (ii) beta = 1 is A times the overlap integral = Eq.7 with V := rho_S and a monopole tip (O12, pinned above);
    (iii) a Gaussian to the power beta is a Gaussian: (q g_s)^beta = q^beta (2 pi s^2)^(3(1-beta)/2) beta^(-3/2)
    g_{s/sqrt(beta)}, so Eq.8 equals Eq.7 on rho_S^beta with that tip (closed form of the tip factor);
    (iv) plane-wave density rho_S^beta = c + a cos(k.r): E and F in closed form."""
    rng = np.random.default_rng(12)
    step = np.diag([0.3, 0.35, 0.4])
    g = W.Grid(origin=np.zeros(3), step=step, n=(5, 4, 3), periodic=(1, 1, 1))
    rho = rng.uniform(0.0, 0.5, (3, 4, 5))
    s, q, A, beta = 0.35, 1.7, 12.0, 1.2
    got = oracle.pauli_forcefield(rho, g, s, q, A, beta)
    dV = 0.3 * 0.35 * 0.4
    for K in range(3):
        for J in range(4):
            for I in range(5):
                acc = 0.0
                for k in range(3):
                    for j in range(4):
                        for i in range(5):
                            r = np.array([(i - 5 if 2 * i >= 5 else i) * 0.3, (j - 4 if 2 * j >= 4 else j) * 0.35,
                                          (k - 3 if 2 * k >= 3 else k) * 0.4])
                            rpp = q * (2 * np.pi * s * s) ** -1.5 * np.exp(-(r @ r) / (2 * s * s))
                            acc += (rpp * rho[(k + K) % 3, (j + J) % 4, (i + I) % 5]) ** beta
                assert np.isclose(got[K, J, I, 3], A * acc * dV, rtol=1e-12)
    # (ii), (iii) on a larger grid
    g2 = _fft_grid()
    rho2 = rng.uniform(0.0, 0.3, (16, 20, 24))
    one = oracle.pauli_forcefield(rho2, g2, 0.4, 1.3, 5.0, 1.0)
    assert np.allclose(one, 5.0 * oracle.fft_forcefield(rho2, g2, 0.4, 1.3, 0.0, 0.0), rtol=1e-12, atol=1e-14)
    for beta in (0.9, 1.1, 1.3):
        s, q, A = 0.45, 1.3, 5.0
        lit = oracle.pauli_forcefield(rho2, g2, s, q, A, beta)
        qeff = A * q**beta * (2 * np.pi * s * s) ** (1.5 * (1 - beta)) * beta ** -1.5
        ident = oracle.fft_forcefield(rho2**beta, g2, s / np.sqrt(beta), qeff, 0.0, 0.0)
        assert np.allclose(lit, ident, rtol=1e-10, atol=1e-12), beta
    # (iv) closed form for a plane-wave rho_S^beta
    n, h = np.array(g2.n), np.diag(np.asarray(g2.step))
    L = n * h
    kvec = 2 * np.pi * np.array([1, 0, -1]) / L
    Kz, Jy, Ix = np.meshgrid(np.arange(n[2]), np.arange(n[1]), np.arange(n[0]), indexing="ij")
    arg = np.stack([Ix * h[0], Jy * h[1], Kz * h[2]], axis=-1) @ kvec
    beta, s, q, A = 1.2, 0.4, 1.0, 3.0
    Sb = 0.5 + 0.3 * np.cos(arg)                                          # rho_S^beta
    got = oracle.pauli_forcefield(Sb ** (1 / beta), g2, s, q, A, beta)
    qeff = A * q**beta * (2 * np.pi * s * s) ** (1.5 * (1 - beta)) * beta ** -1.5
    damp = np.exp(-0.5 * (s * s / beta) * kvec @ kvec)
    assert np.allclose(got[..., 3], qeff * (0.5 + 0.3 * damp * np.cos(arg)), atol=1e-6)
    assert np.allclose(got[..., :3], qeff * 0.3 * damp * np.sin(arg)[..., None] * kvec, atol=1e-6)


def test_golden_constants_are_what_the_generators_use():
    assert W.EVA2_PER_NM == pytest.approx(1.0 / NM, rel=1e-15)
    assert W.ELEM_R[:4].tolist() == [GOLD["R_H"], GOLD["R_C"], GOLD["R_N"], GOLD["R_O"]]
    assert W.ELEM_E[:4].tolist() == [GOLD["e_H"], GOLD["e_C"], GOLD["e_N"], GOLD["e_O"]]
    w = W.get(0)
    assert w.tip.k_lat[0] == pytest.approx(GOLD["k_xy_Nm"] / NM) and w.tip.d0 == (0.0, 0.0, -GOLD["R_rest_A"])
    assert (w.df.A, w.df.k0, w.df.f0) == (GOLD["A_A"], GOLD["k0_Nm"], GOLD["f0_Hz"])


def test_trajectory_stability_diagnostic():
    """lam_traj (reading S17) is the minimum over the trajectory: equals lam_min when no move is made, never
    exceeds it, and goes negative on a step that starts on a maximum of the lateral potential."""
    g, ff = _flat_grid()
    tip = W._default_tip()
    r = oracle.relax_scan(ff, g, tip, W.Fire(), _scan(nz=3))
    assert np.array_equal(r["lam_traj"], r["lam_min"])                    # zero field: single-point trajectories
    ff[..., 2] = 0.03
    r = oracle.relax_scan(ff, g, tip, W.Fire(), _scan(nz=3))
    assert np.all(r["lam_traj"] <= r["lam_min"] + 1e-15)
    # uniform upward push beyond k_xy R_rest: the on-axis start point is laterally unstable (closed form above)
    ff[..., 2] = 0.07
    ff[..., 0] = 1e-4                                                     # break the symmetry so FIRE leaves the axis
    r = oracle.relax_scan(ff, g, tip, replace(W.Fire(), max_iter=5000), _scan(nz=1))
    assert np.all(r["lam_traj"] < 0) and np.all(r["lam_min"] > 0)
    assert np.all(oracle.flags(r))
