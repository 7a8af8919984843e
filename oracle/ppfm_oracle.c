/*
 * ppfm_oracle.c — plain FP64 CPU oracle for the Probe-Particle hot path.
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT CODE.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * `--impl reference` legs may build, load or call this file.  It shares no code, header, table or helper with
 * the CUDA path under paper_2401_14564_b200/csrc/ and includes nothing from include/.
 *
 * Written from the paper (citations are /root/reference/PAPER.md lines) and the readings S1-S20 listed in
 * DESIGN.md.  Deliberately slow and literal: no blocking, no fusion, no reordering beyond what the definition
 * states.  The only parallelism is `#pragma omp parallel for` over independent outputs (grid points, pixels;
 * PAPER.md:266, 280 "perfectly parallelizable", "pixels virtually independent"); sums run in the stated order.
 *
 *   O1  mixing rules
 *   O2  LJ + Coulomb pair terms          PAPER.md:82 (Eq.5), 93 (Eq.6), 76 (F = -grad E)
 *   O3  grid projection, image sum
 *   O4  tri-linear interpolation
 *   O5  tip springs, total force         PAPER.md:45 (Eq.1), 51-54 (Eq.2)
 *   O6  FIRE                             PAPER.md:262 (ref [7]; constants = reading S6)
 *   O7  z-scan, warm start               PAPER.md:262 (reading S8)
 *   O8  Fz read-out
 *   O9  Giessibl df                      PAPER.md:64-66 (Eq.3; quadrature = reading S9)
 *   O10 stability flag (Hessian)         north_star exemption; reading S14
 *   O3+O7 with nodes evaluated lazily     SURVEY.md 8(d) (end-to-end check on sampled pixels of large grids)
 *   O11 stiffness map (IETS)
 *   O13 tri-cubic interpolation of E     PAPER.md:264 ("tri-cubic interpolation of the potential"); reading S22
 *   O14 FDBM Pauli repulsion, Eq.8       PAPER.md:118-122; reading S23
 *   O12 grid electrostatics, Eq.7        PAPER.md:102-111 (cross-correlation), 270 (convolution theorem); reading S21
 *
 * Pins: tests/test_oracle_pins.py (closed forms, invariants, brute force).  "Relaxed positions on the real
 * configs" have no value printed in the paper: PARITY UNPINNED BY THE PAPER for that one item; it is pinned
 * only by an independent Newton minimiser cross-check and by mirror symmetry.
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define KE_EV_A 14.399645478 /* Coulomb constant k_e in eV*Å/e^2 (CODATA 2018), reading S4 */
#define EVA2_TO_NM 16.02176634 /* 1 eV/Å^2 in N/m, reading S4 */

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------------------------------------------------
 * O1 + O2: one atom's contribution at displacement D = p - (r_i + shift).
 *   s = max(|D|^2, r_min^2)                                  (reading S3; identity outside the clamp)
 *   u = (R0^2/s)^3,  E_LJ = E0 (u^2 - 2u)                    (Eq.5 with R0 = R_i + R_PP, E0 = sqrt(e_i e_PP))
 *   F_LJ = -dE/dr * D/r = 12 E0 (u^2 - u)/s * D
 *   E_C = k_e Q q_i / sqrt(s),  F_C = E_C / s * D            (Eq.6)
 * ---------------------------------------------------------------------------------------------------------- */
static void pair_terms(const double D[3], double R0, double E0, double keQq, double rmin2, double out[4]) {
    double s = D[0] * D[0] + D[1] * D[1] + D[2] * D[2];
    if (s < rmin2) s = rmin2;
    double u = (R0 * R0 / s);
    u = u * u * u;
    double e_lj = E0 * (u * u - 2.0 * u);
    double f_lj = 12.0 * E0 * (u * u - u) / s;
    double e_c = keQq / sqrt(s);
    double f_c = e_c / s;
    double f = f_lj + f_c;
    out[0] = f * D[0];
    out[1] = f * D[1];
    out[2] = f * D[2];
    out[3] = e_lj + e_c;
}

/* O3: sample force field at one point p: images outer, atoms inner, plain double accumulation. */
static void ff_at_point(const double p[3], int natoms, const double *xyzq, const int *type, const double *R,
                        const double *e, const double *cell, const int *nimg, double R_pp, double e_pp,
                        double Q_pp, double r_min, double out[4]) {
    const double *a = cell, *b = cell + 3, *c = cell + 6;
    double acc[4] = {0, 0, 0, 0};
    for (int ia = -nimg[0]; ia <= nimg[0]; ia++)
        for (int ib = -nimg[1]; ib <= nimg[1]; ib++)
            for (int ic = -nimg[2]; ic <= nimg[2]; ic++) {
                double sh[3];
                for (int d = 0; d < 3; d++) sh[d] = ia * a[d] + ib * b[d] + ic * c[d];
                for (int i = 0; i < natoms; i++) {
                    int t = type[i];
                    double R0 = R[t] + R_pp;           /* O1 */
                    double E0 = sqrt(e[t] * e_pp);     /* O1 */
                    double D[3], o[4];
                    for (int d = 0; d < 3; d++) D[d] = p[d] - (xyzq[4 * i + d] + sh[d]);
                    pair_terms(D, R0, E0, KE_EV_A * Q_pp * xyzq[4 * i + 3], r_min * r_min, o);
                    for (int d = 0; d < 4; d++) acc[d] += o[d];
                }
            }
    for (int d = 0; d < 4; d++) out[d] = acc[d];
}

/* Force field at arbitrary points (used by pins: finite-difference gradient etc.). */
int oracle_ff_at_points(int natoms, const double *xyzq, const int *type, int ntypes, const double *R,
                        const double *e, const double *cell, const int *nimg, double R_pp, double e_pp,
                        double Q_pp, double r_min, int64_t npts, const double *pts, double *out) {
    for (int i = 0; i < natoms; i++)
        if (type[i] < 0 || type[i] >= ntypes) return -1;
#pragma omp parallel for schedule(static)
    for (int64_t m = 0; m < npts; m++)
        ff_at_point(pts + 3 * m, natoms, xyzq, type, R, e, cell, nimg, R_pp, e_pp, Q_pp, r_min, out + 4 * m);
    return 0;
}

/* O3: the grid.  point(i,j,k) = origin + i*step[0] + j*step[1] + k*step[2]; out[(k*ny + j)*nx + i][4].
 * If idx != NULL only the `nidx` flat indices listed are evaluated and written densely to out[m][4]. */
int oracle_forcefield(int natoms, const double *xyzq, const int *type, int ntypes, const double *R,
                      const double *e, const double *cell, const int *nimg, double R_pp, double e_pp,
                      double Q_pp, const double *origin, const double *step, const int *n, double r_min,
                      int64_t nidx, const int64_t *idx, double *out) {
    for (int i = 0; i < natoms; i++)
        if (type[i] < 0 || type[i] >= ntypes) return -1;
    int64_t nx = n[0], ny = n[1], nz = n[2];
    int64_t total = idx ? nidx : nx * ny * nz;
#pragma omp parallel for schedule(static)
    for (int64_t m = 0; m < total; m++) {
        int64_t flat = idx ? idx[m] : m;
        int64_t i = flat % nx, j = (flat / nx) % ny, k = flat / (nx * ny);
        double p[3];
        for (int d = 0; d < 3; d++) p[d] = origin[d] + i * step[d] + j * step[3 + d] + k * step[6 + d];
        ff_at_point(p, natoms, xyzq, type, R, e, cell, nimg, R_pp, e_pp, Q_pp, r_min, out + 4 * m);
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------------------------
 * Grid view used by O4..O10.
 * ---------------------------------------------------------------------------------------------------------- */
struct lazy_nodes;   /* defined below: grid nodes evaluated on demand from the atoms (O3) and memoised */

typedef struct {
    const void *ff;  /* [nz][ny][nx][4] forces + energy; or, tricubic = 1, [nz][ny][nx] energies only */
    struct lazy_nodes *lazy; /* != NULL: ff is not stored; node (i,j,k) = ff_at_point(origin + i s0 + j s1 + k s2) */
    int is_f32;      /* 1: float data, widened to double on access (GPU-produced grids) */
    int tricubic;    /* O13: the sample force is -grad of the tri-cubic interpolant of an energy grid */
    double origin[3];
    double Minv[9];  /* t = Minv * (r - origin), fractional grid coordinates */
    int n[3];
    int periodic[3];
} grid_view;

static const double *lazy_node(struct lazy_nodes *L, const grid_view *g, int i, int j, int k);

static double ff_get(const grid_view *g, int i, int j, int k, int comp) {
    if (g->lazy) return lazy_node(g->lazy, g, i, j, k)[comp];
    size_t o = (((size_t)k * g->n[1] + j) * g->n[0] + i) * (g->tricubic ? 1 : 4) + (g->tricubic ? 0 : comp);
    return g->is_f32 ? (double)((const float *)g->ff)[o] : ((const double *)g->ff)[o];
}

static int invert3(const double *S /* rows = step vectors */, double *Minv) {
    /* r - origin = S^T t  ->  t = (S^T)^-1 (r - origin).  Build A = S^T and invert by cofactors. */
    double A[9];
    for (int r = 0; r < 3; r++)
        for (int c = 0; c < 3; c++) A[3 * r + c] = S[3 * c + r];
    double det = A[0] * (A[4] * A[8] - A[5] * A[7]) - A[1] * (A[3] * A[8] - A[5] * A[6]) +
                 A[2] * (A[3] * A[7] - A[4] * A[6]);
    if (det == 0.0 || !isfinite(det)) return -1;
    double id = 1.0 / det;
    Minv[0] = (A[4] * A[8] - A[5] * A[7]) * id;
    Minv[1] = (A[2] * A[7] - A[1] * A[8]) * id;
    Minv[2] = (A[1] * A[5] - A[2] * A[4]) * id;
    Minv[3] = (A[5] * A[6] - A[3] * A[8]) * id;
    Minv[4] = (A[0] * A[8] - A[2] * A[6]) * id;
    Minv[5] = (A[2] * A[3] - A[0] * A[5]) * id;
    Minv[6] = (A[3] * A[7] - A[4] * A[6]) * id;
    Minv[7] = (A[1] * A[6] - A[0] * A[7]) * id;
    Minv[8] = (A[0] * A[4] - A[1] * A[3]) * id;
    return 0;
}

static int make_view(grid_view *g, const void *ff, int is_f32, const double *origin, const double *step,
                     const int *n, const int *periodic) {
    g->ff = ff;
    g->lazy = NULL;
    g->is_f32 = is_f32 & 1;       /* the callers' flag word: bit 0 = float data, bit 1 = tri-cubic energy grid (O13) */
    g->tricubic = (is_f32 >> 1) & 1;
    for (int d = 0; d < 3; d++) {
        g->origin[d] = origin[d];
        g->n[d] = n[d];
        g->periodic[d] = periodic[d];
        if (n[d] < 2) return -1;
    }
    return invert3(step, g->Minv);
}

/* O4: cell index pair (i0,i1) and fraction f along one axis.
 *   periodic:      i0 = floor(t) mod n, i1 = (i0+1) mod n, f = t - floor(t)
 *   non-periodic:  t clamped to [0, n-1]; i0 = min(floor(t), n-2); i1 = i0+1; f = t - i0     (reading S12)
 * returns 1 if the coordinate was clamped. */
static int axis_cell(double t, int n, int periodic, int *i0, int *i1, double *f) {
    if (periodic) {
        double fl = floor(t);
        long m = (long)fl % n;
        if (m < 0) m += n;
        *i0 = (int)m;
        *i1 = (int)((m + 1) % n);
        *f = t - fl;
        return 0;
    }
    int clamped = 0;
    if (t < 0.0) { t = 0.0; clamped = 1; }
    if (t > (double)(n - 1)) { t = (double)(n - 1); clamped = 1; }
    int i = (int)floor(t);
    if (i > n - 2) i = n - 2;
    *i0 = i;
    *i1 = i + 1;
    *f = t - (double)i;
    return clamped;
}

/* O13 (reading S22): F_S = -grad of the tri-cubic interpolant of the energy grid.  Per axis the
 * interpolating cubic convolution kernel (Catmull-Rom / Keys a = -1/2) on the four nodes i0-1 .. i0+2 around the
 * cell [i0, i0+1) that O4's axis_cell picks:
 *     w0 = (-f^3 + 2f^2 - f)/2,  w1 = (3f^3 - 5f^2 + 2)/2,  w2 = (-3f^3 + 4f^2 + f)/2,  w3 = (f^3 - f^2)/2,
 * tensor product over the three axes; stencil indices wrap on periodic axes and are clamped to [0, n-1] on the
 * others (edge replication).  E is C^1, reproduces polynomials up to degree 2 in each variable and passes through
 * the node values.  Returns F = -(dE/dt) Minv and, if G != NULL, G[c][b] = dF_c/dt_b (second derivatives). */
static void cubic_weights(double f, double w[4], double d1[4], double d2[4]) {
    w[0] = 0.5 * (-f * f * f + 2.0 * f * f - f);
    w[1] = 0.5 * (3.0 * f * f * f - 5.0 * f * f + 2.0);
    w[2] = 0.5 * (-3.0 * f * f * f + 4.0 * f * f + f);
    w[3] = 0.5 * (f * f * f - f * f);
    d1[0] = 0.5 * (-3.0 * f * f + 4.0 * f - 1.0);
    d1[1] = 0.5 * (9.0 * f * f - 10.0 * f);
    d1[2] = 0.5 * (-9.0 * f * f + 8.0 * f + 1.0);
    d1[3] = 0.5 * (3.0 * f * f - 2.0 * f);
    d2[0] = -3.0 * f + 2.0;
    d2[1] = 9.0 * f - 5.0;
    d2[2] = -9.0 * f + 4.0;
    d2[3] = 3.0 * f - 1.0;
}

static int stencil_index(int i0, int off, int n, int periodic) {
    int i = i0 + off;
    if (periodic) { i %= n; if (i < 0) i += n; return i; }
    if (i < 0) i = 0;
    if (i > n - 1) i = n - 1;
    return i;
}

static int interp_tricubic(const grid_view *g, const double r[3], double F[3], double G[9]) {
    double t[3], f[3], w[3][4], d1[3][4], d2[3][4];
    int i0[3], i1[3], idx[3][4], clamped = 0;
    for (int a = 0; a < 3; a++)
        t[a] = g->Minv[3 * a] * (r[0] - g->origin[0]) + g->Minv[3 * a + 1] * (r[1] - g->origin[1]) +
               g->Minv[3 * a + 2] * (r[2] - g->origin[2]);
    for (int a = 0; a < 3; a++) {
        clamped |= axis_cell(t[a], g->n[a], g->periodic[a], &i0[a], &i1[a], &f[a]);
        cubic_weights(f[a], w[a], d1[a], d2[a]);
        for (int m = 0; m < 4; m++) idx[a][m] = stencil_index(i0[a], m - 1, g->n[a], g->periodic[a]);
    }
    double E1[3] = {0, 0, 0}, E2[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0}; /* dE/dt_a, d2E/dt_a dt_b */
    for (int kz = 0; kz < 4; kz++)
        for (int ky = 0; ky < 4; ky++)
            for (int kx = 0; kx < 4; kx++) {
                const double e = ff_get(g, idx[0][kx], idx[1][ky], idx[2][kz], 0);
                const double W[3] = {w[0][kx], w[1][ky], w[2][kz]};
                const double D[3] = {d1[0][kx], d1[1][ky], d1[2][kz]};
                const double S[3] = {d2[0][kx], d2[1][ky], d2[2][kz]};
                E1[0] += D[0] * W[1] * W[2] * e;
                E1[1] += W[0] * D[1] * W[2] * e;
                E1[2] += W[0] * W[1] * D[2] * e;
                E2[0] += S[0] * W[1] * W[2] * e;
                E2[4] += W[0] * S[1] * W[2] * e;
                E2[8] += W[0] * W[1] * S[2] * e;
                E2[1] += D[0] * D[1] * W[2] * e;
                E2[2] += D[0] * W[1] * D[2] * e;
                E2[5] += W[0] * D[1] * D[2] * e;
            }
    E2[3] = E2[1]; E2[6] = E2[2]; E2[7] = E2[5];
    for (int c = 0; c < 3; c++) {
        F[c] = -(E1[0] * g->Minv[0 + c] + E1[1] * g->Minv[3 + c] + E1[2] * g->Minv[6 + c]);
        if (G)
            for (int b = 0; b < 3; b++)
                G[3 * c + b] = -(E2[0 + b] * g->Minv[0 + c] + E2[3 + b] * g->Minv[3 + c] + E2[6 + b] * g->Minv[6 + c]);
    }
    return clamped;
}

/* O4: F_S(r) = sum over 8 corners of w * FF.xyz.  If G != NULL also returns G[c][a] = dF_c/dt_a, the analytic
 * derivative of the interpolant with respect to the fractional coordinates inside the current cell (for O10). */
static int interp(const grid_view *g, const double r[3], double F[3], double G[9]) {
    if (g->tricubic) return interp_tricubic(g, r, F, G);
    double t[3], f[3];
    int i0[3], i1[3], clamped = 0;
    for (int a = 0; a < 3; a++)
        t[a] = g->Minv[3 * a] * (r[0] - g->origin[0]) + g->Minv[3 * a + 1] * (r[1] - g->origin[1]) +
               g->Minv[3 * a + 2] * (r[2] - g->origin[2]);
    for (int a = 0; a < 3; a++) clamped |= axis_cell(t[a], g->n[a], g->periodic[a], &i0[a], &i1[a], &f[a]);
    for (int c = 0; c < 3; c++) F[c] = 0.0;
    if (G) for (int m = 0; m < 9; m++) G[m] = 0.0;
    for (int cz = 0; cz < 2; cz++)
        for (int cy = 0; cy < 2; cy++)
            for (int cx = 0; cx < 2; cx++) {
                double wx = cx ? f[0] : 1.0 - f[0], wy = cy ? f[1] : 1.0 - f[1], wz = cz ? f[2] : 1.0 - f[2];
                double sx = cx ? 1.0 : -1.0, sy = cy ? 1.0 : -1.0, sz = cz ? 1.0 : -1.0;
                int i = cx ? i1[0] : i0[0], j = cy ? i1[1] : i0[1], k = cz ? i1[2] : i0[2];
                for (int c = 0; c < 3; c++) {
                    double v = ff_get(g, i, j, k, c);
                    F[c] += wx * wy * wz * v;
                    if (G) {
                        G[3 * c + 0] += sx * wy * wz * v;
                        G[3 * c + 1] += wx * sy * wz * v;
                        G[3 * c + 2] += wx * wy * sz * v;
                    }
                }
            }
    return clamped;
}

int oracle_interp(const void *ff, int is_f32, const double *origin, const double *step, const int *n,
                  const int *periodic, int64_t npts, const double *pts, double *out /* [npts][3] */) {
    grid_view g;
    if (make_view(&g, ff, is_f32, origin, step, n, periodic)) return -1;
    for (int64_t m = 0; m < npts; m++) interp(&g, pts + 3 * m, out + 3 * m, NULL);
    return 0;
}

/* ------------------------------------------------------------------------------------------------------------
 * O5: tip force (Eq.2) and total force (Eq.1).
 *   d = r_PP - r_TIP;  F_R = -k_R (|d| - R0) d/|d|, R0 = |d0|;  F_L = -(k_x (d_x - d0_x), k_y (d_y - d0_y), 0)
 * ---------------------------------------------------------------------------------------------------------- */
typedef struct {
    double k_lat[2], k_rad, d0[3], R_rest;
} tip_t;

static void radial_force(const tip_t *tp, const double d[3], double FR[3]) {
    double L = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
    for (int c = 0; c < 3; c++) FR[c] = (L > 0.0) ? -tp->k_rad * (L - tp->R_rest) * d[c] / L : 0.0;
}

static int total_force(const grid_view *g, const tip_t *tp, const double rtip[3], const double rpp[3],
                       double F[3]) {
    double d[3], FS[3], FR[3];
    for (int c = 0; c < 3; c++) d[c] = rpp[c] - rtip[c];
    int clamped = interp(g, rpp, FS, NULL);
    radial_force(tp, d, FR);
    F[0] = FS[0] + FR[0] - tp->k_lat[0] * (d[0] - tp->d0[0]);
    F[1] = FS[1] + FR[1] - tp->k_lat[1] * (d[1] - tp->d0[1]);
    F[2] = FS[2] + FR[2];
    return clamped;
}

int oracle_total_force(const void *ff, int is_f32, const double *origin, const double *step, const int *n,
                       const int *periodic, const double *k_lat, double k_rad, const double *d0,
                       const double *rtip, const double *rpp, double *F) {
    grid_view g;
    if (make_view(&g, ff, is_f32, origin, step, n, periodic)) return -1;
    tip_t tp = {{k_lat[0], k_lat[1]}, k_rad, {d0[0], d0[1], d0[2]},
                sqrt(d0[0] * d0[0] + d0[1] * d0[1] + d0[2] * d0[2])};
    total_force(&g, &tp, rtip, rpp, F);
    return 0;
}

/* ------------------------------------------------------------------------------------------------------------
 * O10: Hessian of the PP's total potential at r_PP:  H = H_spring - (J + J^T)/2,
 *   J = dF_S/dr = G * Minv (chain rule through t = Minv (r - origin)),
 *   H_spring = k_R dd^T/|d|^2 + k_R (|d|-R0)/|d| (I - dd^T/|d|^2) + diag(k_x, k_y, 0).
 * Eigenvalues by cyclic Jacobi rotations (symmetric 3x3).
 * ---------------------------------------------------------------------------------------------------------- */
static void hessian(const grid_view *g, const tip_t *tp, const double rtip[3], const double rpp[3], double H[9]) {
    double F[3], G[9], J[9], d[3];
    interp(g, rpp, F, G);
    for (int r = 0; r < 3; r++)
        for (int c = 0; c < 3; c++) {
            double s = 0.0;
            for (int a = 0; a < 3; a++) s += G[3 * r + a] * g->Minv[3 * a + c];
            J[3 * r + c] = s;
        }
    for (int c = 0; c < 3; c++) d[c] = rpp[c] - rtip[c];
    double L = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
    for (int r = 0; r < 3; r++)
        for (int c = 0; c < 3; c++) {
            double dd = d[r] * d[c] / (L * L);
            double I = (r == c) ? 1.0 : 0.0;
            H[3 * r + c] = tp->k_rad * dd + tp->k_rad * (L - tp->R_rest) / L * (I - dd) -
                           0.5 * (J[3 * r + c] + J[3 * c + r]);
        }
    H[0] += tp->k_lat[0];
    H[4] += tp->k_lat[1];
}

static void sym3_eig(const double Hin[9], double w[3]) {
    double A[9];
    memcpy(A, Hin, sizeof(A));
    for (int sweep = 0; sweep < 60; sweep++) {
        double off = A[1] * A[1] + A[2] * A[2] + A[5] * A[5];
        if (off < 1e-300) break;
        for (int p = 0; p < 2; p++)
            for (int q = p + 1; q < 3; q++) {
                double apq = A[3 * p + q];
                if (apq == 0.0) continue;
                double theta = (A[3 * q + q] - A[3 * p + p]) / (2.0 * apq);
                double t = (theta >= 0 ? 1.0 : -1.0) / (fabs(theta) + sqrt(theta * theta + 1.0));
                double c = 1.0 / sqrt(t * t + 1.0), s = t * c;
                for (int k = 0; k < 3; k++) { /* A <- A * R */
                    double akp = A[3 * k + p], akq = A[3 * k + q];
                    A[3 * k + p] = c * akp - s * akq;
                    A[3 * k + q] = s * akp + c * akq;
                }
                for (int k = 0; k < 3; k++) { /* A <- R^T * A */
                    double apk = A[3 * p + k], aqk = A[3 * q + k];
                    A[3 * p + k] = c * apk - s * aqk;
                    A[3 * q + k] = s * apk + c * aqk;
                }
            }
    }
    w[0] = A[0]; w[1] = A[4]; w[2] = A[8];
    for (int i = 0; i < 2; i++)
        for (int j = 0; j < 2 - i; j++)
            if (w[j] > w[j + 1]) { double t = w[j]; w[j] = w[j + 1]; w[j + 1] = t; }
}

int oracle_hessian(const void *ff, int is_f32, const double *origin, const double *step, const int *n,
                   const int *periodic, const double *k_lat, double k_rad, const double *d0,
                   const double *rtip, const double *rpp, double *H /* 9 */, double *eig /* 3 ascending */) {
    grid_view g;
    if (make_view(&g, ff, is_f32, origin, step, n, periodic)) return -1;
    tip_t tp = {{k_lat[0], k_lat[1]}, k_rad, {d0[0], d0[1], d0[2]},
                sqrt(d0[0] * d0[0] + d0[1] * d0[1] + d0[2] * d0[2])};
    hessian(&g, &tp, rtip, rpp, H);
    sym3_eig(H, eig);
    return 0;
}

/* ------------------------------------------------------------------------------------------------------------
 * Stiffness map (IETS module: "calculates the change of the stiffness (resp. vibration
 * frequency) of lateral vibration modes of the CO molecule attached to the AFM tip due to its interaction with the
 * sample"): O10's Hessian and its three eigenvalues (ascending) at npts given (r_TIP, r_PP) pairs.
 * ---------------------------------------------------------------------------------------------------------- */
int oracle_stiffness(const void *ff, int is_f32, const double *origin, const double *step, const int *n,
                     const int *periodic, const double *k_lat, double k_rad, const double *d0, int64_t npts,
                     const double *rtip /* [npts][3] */, const double *rpp /* [npts][3] */,
                     double *eig /* [npts][3] */) {
    grid_view g;
    if (make_view(&g, ff, is_f32, origin, step, n, periodic)) return -1;
    tip_t tp = {{k_lat[0], k_lat[1]}, k_rad, {d0[0], d0[1], d0[2]},
                sqrt(d0[0] * d0[0] + d0[1] * d0[1] + d0[2] * d0[2])};
#pragma omp parallel for schedule(static)
    for (int64_t m = 0; m < npts; m++) {
        double H[9];
        hessian(&g, &tp, rtip + 3 * m, rpp + 3 * m, H);
        sym3_eig(H, eig + 3 * m);
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------------------------
 * O12: electrostatics of an extended tip charge density on the grid (Eq.7):
 *     E_el(R) = integral rho_PP(r) V_S(r + R) dr,        F_el(R) = -grad_R E_el = integral grad rho_PP(r) V_S(r + R) dr
 * (integration by parts on the periodic cell).  Reading S21: the integral is the cyclic sum over the nodes of the
 * periodic grid times the cell volume element dV = |det(step)|; rho_PP is a Gaussian multipole (PAPER.md:108:
 * monopole, and "the quadrupolar charge distribution better reproduces contrast observed with a CO-tip")
 *     g(r) = (2 pi sigma^2)^(-3/2) exp(-r^2 / 2 sigma^2)
 *     rho  = [ q_s + p_z z / sigma^2 + (Q_zz / 12) (3 z^2 - r^2) / sigma^4 ] g(r)
 * (total charge q_s, dipole moment p_z, quadrupole moment Q_zz = integral rho (3z^2 - r^2) dr), evaluated with its
 * analytic gradient at node (i,j,k) -> r = i' s0 + j' s1 + k' s2, i' = i - n0 if i >= n0/2 (minimum image by index).
 * This function is the definition written out: O(N^2) direct sums, for small grids only.
 * ---------------------------------------------------------------------------------------------------------- */
int oracle_tip_density(const double *step /* [3][3] */, const int *n, double sigma, double q_s, double p_z,
                       double Q_zz, double *rho4 /* [4][nz][ny][nx]: rho, d/dx, d/dy, d/dz */) {
    if (!(sigma > 0.0) || n[0] < 1 || n[1] < 1 || n[2] < 1) return -1;
    const int64_t N = (int64_t)n[0] * n[1] * n[2];
    const double s2 = sigma * sigma, s4 = s2 * s2;
    const double norm = pow(2.0 * M_PI * s2, -1.5);
    for (int k = 0; k < n[2]; k++)
        for (int j = 0; j < n[1]; j++)
            for (int i = 0; i < n[0]; i++) {
                const int iw = (2 * i >= n[0]) ? i - n[0] : i;
                const int jw = (2 * j >= n[1]) ? j - n[1] : j;
                const int kw = (2 * k >= n[2]) ? k - n[2] : k;
                double r[3];
                for (int c = 0; c < 3; c++) r[c] = iw * step[0 + c] + jw * step[3 + c] + kw * step[6 + c];
                const double rr = r[0] * r[0] + r[1] * r[1] + r[2] * r[2];
                const double g = norm * exp(-rr / (2.0 * s2));
                const double P = q_s + p_z * r[2] / s2 + (Q_zz / 12.0) * (3.0 * r[2] * r[2] - rr) / s4;
                const double dP[3] = {(Q_zz / 12.0) * (-2.0 * r[0]) / s4, (Q_zz / 12.0) * (-2.0 * r[1]) / s4,
                                      p_z / s2 + (Q_zz / 12.0) * (4.0 * r[2]) / s4};
                const int64_t m = ((int64_t)k * n[1] + j) * n[0] + i;
                rho4[m] = P * g;
                for (int c = 0; c < 3; c++) rho4[(c + 1) * N + m] = dP[c] * g - P * g * r[c] / s2;
            }
    return 0;
}

/* out[R] = dV * sum_r rho[r] * V[(r + R) mod n]   (cyclic cross-correlation, Eq.7 on the grid) */
int oracle_crosscorr(const int *n, const double *rho, const double *V, double dV, double *out) {
    const int nx = n[0], ny = n[1], nz = n[2];
#pragma omp parallel for collapse(2) schedule(static)
    for (int K = 0; K < nz; K++)
        for (int J = 0; J < ny; J++)
            for (int I = 0; I < nx; I++) {
                double acc = 0.0;
                for (int k = 0; k < nz; k++) {
                    const int kk = (k + K) % nz;
                    for (int j = 0; j < ny; j++) {
                        const int jj = (j + J) % ny;
                        const double *pr = rho + ((int64_t)k * ny + j) * nx;
                        const double *pv = V + ((int64_t)kk * ny + jj) * nx;
                        for (int i = 0; i < nx; i++) acc += pr[i] * pv[(i + I) % nx];
                    }
                }
                out[((int64_t)K * ny + J) * nx + I] = acc * dV;
            }
    return 0;
}

/* The same sum at npts selected output nodes (I, J, K) only: full-size grids are checked on samples. */
int oracle_crosscorr_at(const int *n, const double *rho, const double *V, double dV, int64_t npts,
                        const int *ijk /* [npts][3] */, double *out /* [npts] */) {
    const int nx = n[0], ny = n[1], nz = n[2];
#pragma omp parallel for schedule(dynamic)
    for (int64_t m = 0; m < npts; m++) {
        const int I = ijk[3 * m], J = ijk[3 * m + 1], K = ijk[3 * m + 2];
        double acc = 0.0;
        for (int k = 0; k < nz; k++) {
            const int kk = (k + K) % nz;
            for (int j = 0; j < ny; j++) {
                const int jj = (j + J) % ny;
                const double *pr = rho + ((int64_t)k * ny + j) * nx;
                const double *pv = V + ((int64_t)kk * ny + jj) * nx;
                for (int i = 0; i < nx; i++) acc += pr[i] * pv[(i + I) % nx];
            }
        }
        out[m] = acc * dV;
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------------------------
 * O14: Pauli repulsion of the full density-based model (Eq.8):
 *     E_Pauli(R) = A integral [ rho_PP(r) rho_S(r + R) ]^beta dr,      F = -grad_R E_Pauli.
 * Reading S23: on the periodic grid as in S21; rho_PP = q g_sigma(r) (a Gaussian electron density of q electrons,
 * positive, so the power is defined); rho_S is clipped at 0 before the power.  This routine only tabulates the tip
 * factor literally, T0 = (q g)^beta and its analytic gradient T_a = beta (q g)^(beta-1) q dg/dr_a; the sums are
 * oracle_crosscorr(T, rho_S^beta) (the integrand factorises: [ab]^beta = a^beta b^beta for a, b >= 0).
 * ---------------------------------------------------------------------------------------------------------- */
int oracle_pauli_tip(const double *step /* [3][3] */, const int *n, double sigma, double q, double beta,
                     double *T4 /* [4][nz][ny][nx]: T0, dT0/dx, dT0/dy, dT0/dz */) {
    if (!(sigma > 0.0) || !(q > 0.0) || !(beta > 0.0)) return -1;
    const int64_t N = (int64_t)n[0] * n[1] * n[2];
    const double s2 = sigma * sigma;
    const double norm = pow(2.0 * M_PI * s2, -1.5);
    for (int k = 0; k < n[2]; k++)
        for (int j = 0; j < n[1]; j++)
            for (int i = 0; i < n[0]; i++) {
                const int iw = (2 * i >= n[0]) ? i - n[0] : i;
                const int jw = (2 * j >= n[1]) ? j - n[1] : j;
                const int kw = (2 * k >= n[2]) ? k - n[2] : k;
                double r[3];
                for (int c = 0; c < 3; c++) r[c] = iw * step[0 + c] + jw * step[3 + c] + kw * step[6 + c];
                const double rr = r[0] * r[0] + r[1] * r[1] + r[2] * r[2];
                const double rho = q * norm * exp(-rr / (2.0 * s2));          /* rho_PP(r) */
                const int64_t m = ((int64_t)k * n[1] + j) * n[0] + i;
                T4[m] = pow(rho, beta);
                for (int c = 0; c < 3; c++) {
                    const double drho = -rho * r[c] / s2;                     /* d rho_PP / d r_c */
                    T4[(c + 1) * N + m] = (rho > 0.0) ? beta * pow(rho, beta - 1.0) * drho : 0.0;
                }
            }
    return 0;
}

/* ------------------------------------------------------------------------------------------------------------
 * O6 FIRE + O7 scan + O8 read-out + O10 flag.
 *
 * fire[7] = {dt0, dt_max, finc, fdec, alpha0, falpha, f_conv}.
 * Pixel (ix,iy), step iz: r_TIP = p0 + ix*dx + iy*dy - (0,0,iz*dz).
 * iz = 0: r_PP = r_TIP + d0.  iz > 0: r_PP shifted with the tip (d carried over), FIRE state reset.
 * Outputs (dense over the selected pixels, [nz][npix]):
 *   pos_fz[.][4] = (r_PP, Fz_tip = -F_R,z);  iters = moves made, -1 if max_iter moves did not converge;
 *   lam_min = smallest Hessian eigenvalue at the relaxed point;  clamped = 1 if the final r_PP was clamped (S12).
 *   lam_traj (optional) = smallest Hessian eigenvalue over EVERY point of the step's FIRE path (warm-start point,
 *   each intermediate point, end point).  Reading S17: when it drops below 1e-3 eV/Å^2 the PP crosses a ridge of the
 *   potential on its way (snap-through, or an inertial overshoot out of a shallow basin); which basin FIRE then
 *   lands in depends on rounding-level differences of the grid, so such samples count as near-unstable just like
 *   samples whose END point has lambda < 1e-3.  (Observed: config 1, pixel 19076, z-step 35: the oracle on its own
 *   FP64 grid and on an FP32 grid that agrees with it to 1e-5 lands in two different stable minima, 0.88 Å apart,
 *   end-point lambda 8.0e-3 and 2.8e-3; path minimum -8.9e-3 and -4.0e-3.)
 * If pix != NULL only the `npix` flat pixel indices (iy*npx + ix) listed are computed.
 * ---------------------------------------------------------------------------------------------------------- */
static double norm3(const double v[3]) { return sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]); }

typedef struct {
    double dt0, dt_max, finc, fdec, alpha0, falpha, f_conv;
    int n_min, max_iter;
} fire_t;

typedef struct {
    double p0[3], dx[3], dy[3], dz;
    int npx, npy, nz;
} scan_t;

/* One pixel (ix, iy), all z-steps (O6 + O7 + O8 + O10); output column m of `total` columns. */
static void relax_pixel(const grid_view *g, const tip_t *tp, const fire_t *fp, const scan_t *sc, int ix, int iy,
                        int64_t m, int64_t total, double *pos_fz, int *iters, double *lam_min, int *clamped_out,
                        double *lam_traj) {
    double dcur[3] = {tp->d0[0], tp->d0[1], tp->d0[2]}; /* O7: d carried from step to step */
    for (int iz = 0; iz < sc->nz; iz++) {
        double rtip[3], r[3], v[3] = {0, 0, 0}, F[3];
        for (int c = 0; c < 3; c++) rtip[c] = sc->p0[c] + ix * sc->dx[c] + iy * sc->dy[c];
        rtip[2] -= iz * sc->dz;
        for (int c = 0; c < 3; c++) r[c] = rtip[c] + dcur[c];
        double dt = fp->dt0, alpha = fp->alpha0;
        int n_pos = 0, moves = 0, converged = 0, cl = 0;
        double ltraj = INFINITY;
        for (;;) { /* O6 */
            cl = total_force(g, tp, rtip, r, F);
            if (lam_traj) { /* diagnostic only (O10 / S17): does not touch the FIRE state */
                double Ht[9], wt[3];
                hessian(g, tp, rtip, r, Ht);
                sym3_eig(Ht, wt);
                if (wt[0] < ltraj) ltraj = wt[0];
            }
            double Fn = norm3(F);
            if (Fn < fp->f_conv) { converged = 1; break; } /* S7: check before moving */
            if (moves >= fp->max_iter) break;
            double P = F[0] * v[0] + F[1] * v[1] + F[2] * v[2];
            if (P >= 0.0) { /* S6: P = 0 counts as downhill */
                double vn = norm3(v);
                for (int c = 0; c < 3; c++) v[c] = (1.0 - alpha) * v[c] + alpha * vn * F[c] / Fn;
                if (n_pos > fp->n_min) {
                    dt = fmin(dt * fp->finc, fp->dt_max);
                    alpha *= fp->falpha;
                }
                n_pos += 1;
            } else {
                v[0] = v[1] = v[2] = 0.0;
                dt *= fp->fdec;
                alpha = fp->alpha0;
                n_pos = 0;
            }
            for (int c = 0; c < 3; c++) v[c] += F[c] * dt; /* semi-implicit Euler, m = 1 */
            for (int c = 0; c < 3; c++) r[c] += v[c] * dt;
            moves++;
        }
        for (int c = 0; c < 3; c++) dcur[c] = r[c] - rtip[c];
        double FR[3];
        radial_force(tp, dcur, FR); /* O8: Fz_tip = -F_R,z */
        size_t o = (size_t)iz * total + m;
        pos_fz[4 * o + 0] = r[0];
        pos_fz[4 * o + 1] = r[1];
        pos_fz[4 * o + 2] = r[2];
        pos_fz[4 * o + 3] = -FR[2];
        if (iters) iters[o] = converged ? moves : -1;
        if (clamped_out) clamped_out[o] = cl;
        if (lam_traj) lam_traj[o] = ltraj;
        if (lam_min) {
            double H[9], w[3];
            hessian(g, tp, rtip, r, H);
            sym3_eig(H, w);
            lam_min[o] = w[0];
        }
    }
}

static void pack_scan(fire_t *fp, scan_t *sc, const double *fire, int n_min, int max_iter, const double *p0,
                      const double *dx, const double *dy, int npx, int npy, int nz, double dz) {
    fp->dt0 = fire[0]; fp->dt_max = fire[1]; fp->finc = fire[2]; fp->fdec = fire[3]; fp->alpha0 = fire[4];
    fp->falpha = fire[5]; fp->f_conv = fire[6];
    fp->n_min = n_min; fp->max_iter = max_iter;
    for (int c = 0; c < 3; c++) { sc->p0[c] = p0[c]; sc->dx[c] = dx[c]; sc->dy[c] = dy[c]; }
    sc->dz = dz; sc->npx = npx; sc->npy = npy; sc->nz = nz;
}

int oracle_relax_scan(const void *ff, int is_f32, const double *origin, const double *step, const int *n,
                      const int *periodic, const double *k_lat, double k_rad, const double *d0,
                      const double *fire, int n_min, int max_iter, const double *p0, const double *dx,
                      const double *dy, int npx, int npy, int nz, double dz, int64_t npix, const int64_t *pix,
                      double *pos_fz, int *iters, double *lam_min, int *clamped_out, double *lam_traj) {
    grid_view g;
    if (make_view(&g, ff, is_f32, origin, step, n, periodic)) return -1;
    tip_t tp = {{k_lat[0], k_lat[1]}, k_rad, {d0[0], d0[1], d0[2]},
                sqrt(d0[0] * d0[0] + d0[1] * d0[1] + d0[2] * d0[2])};
    fire_t fp;
    scan_t sc;
    pack_scan(&fp, &sc, fire, n_min, max_iter, p0, dx, dy, npx, npy, nz, dz);
    int64_t total = pix ? npix : (int64_t)npx * npy;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t m = 0; m < total; m++) {
        int64_t flat = pix ? pix[m] : m;
        relax_pixel(&g, &tp, &fp, &sc, (int)(flat % npx), (int)(flat / npx), m, total, pos_fz, iters, lam_min,
                    clamped_out, lam_traj);
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------------------------
 * The same scan with the grid NOT stored: every node the interpolation touches is evaluated on demand from the
 * atoms with ff_at_point (O3, exactly the value oracle_forcefield would have stored there) and memoised per pixel.
 * This is what makes an end-to-end check (the oracle on its own FP64 grid) affordable on grids whose full
 * evaluation would take hours ("lazily evaluated, memoised FP64 nodes"); no arithmetic differs
 * from oracle_forcefield + oracle_relax_scan.  nodes_out[m] (optional) = nodes evaluated for pixel m.
 * ---------------------------------------------------------------------------------------------------------- */
struct lazy_nodes {
    int natoms;
    const double *xyzq;
    const int *type;
    const double *R, *e, *cell;
    const int *nimg;
    double R_pp, e_pp, Q_pp, r_min;
    const double *origin, *step;
    /* open-addressing table: key = flat node index + 1 (0 = empty), value = 4 doubles */
    int64_t cap, used;
    int64_t *keys;
    double *vals;
};

static const double *lazy_node(struct lazy_nodes *L, const grid_view *g, int i, int j, int k) {
    const int64_t key = (((int64_t)k * g->n[1] + j) * g->n[0] + i) + 1;
    if (2 * (L->used + 1) > L->cap) { /* grow and re-insert */
        int64_t ncap = L->cap ? 2 * L->cap : 1024;
        int64_t *nk = (int64_t *)calloc((size_t)ncap, sizeof(int64_t));
        double *nv = (double *)malloc((size_t)ncap * 4 * sizeof(double));
        for (int64_t s = 0; s < L->cap; s++)
            if (L->keys[s]) {
                int64_t h = (int64_t)(((uint64_t)L->keys[s] * 0x9E3779B97F4A7C15ull) >> 11) & (ncap - 1);
                while (nk[h]) h = (h + 1) & (ncap - 1);
                nk[h] = L->keys[s];
                memcpy(nv + 4 * h, L->vals + 4 * s, 4 * sizeof(double));
            }
        free(L->keys);
        free(L->vals);
        L->keys = nk; L->vals = nv; L->cap = ncap;
    }
    int64_t h = (int64_t)(((uint64_t)key * 0x9E3779B97F4A7C15ull) >> 11) & (L->cap - 1);
    while (L->keys[h] && L->keys[h] != key) h = (h + 1) & (L->cap - 1);
    if (!L->keys[h]) {
        double p[3];
        for (int d = 0; d < 3; d++) p[d] = L->origin[d] + i * L->step[d] + j * L->step[3 + d] + k * L->step[6 + d];
        ff_at_point(p, L->natoms, L->xyzq, L->type, L->R, L->e, L->cell, L->nimg, L->R_pp, L->e_pp, L->Q_pp,
                    L->r_min, L->vals + 4 * h);
        L->keys[h] = key;
        L->used++;
    }
    return L->vals + 4 * h;
}

int oracle_relax_scan_atoms(int natoms, const double *xyzq, const int *type, int ntypes, const double *R,
                            const double *e, const double *cell, const int *nimg, double R_pp, double e_pp,
                            double Q_pp, double r_min, const double *origin, const double *step, const int *n,
                            const int *periodic, const double *k_lat, double k_rad, const double *d0,
                            const double *fire, int n_min, int max_iter, const double *p0, const double *dx,
                            const double *dy, int npx, int npy, int nz, double dz, int64_t npix, const int64_t *pix,
                            double *pos_fz, int *iters, double *lam_min, int *clamped_out, double *lam_traj,
                            int64_t *nodes_out) {
    for (int i = 0; i < natoms; i++)
        if (type[i] < 0 || type[i] >= ntypes) return -1;
    grid_view g0;
    if (make_view(&g0, NULL, 0, origin, step, n, periodic)) return -1;
    tip_t tp = {{k_lat[0], k_lat[1]}, k_rad, {d0[0], d0[1], d0[2]},
                sqrt(d0[0] * d0[0] + d0[1] * d0[1] + d0[2] * d0[2])};
    fire_t fp;
    scan_t sc;
    pack_scan(&fp, &sc, fire, n_min, max_iter, p0, dx, dy, npx, npy, nz, dz);
    int64_t total = pix ? npix : (int64_t)npx * npy;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t m = 0; m < total; m++) {
        int64_t flat = pix ? pix[m] : m;
        struct lazy_nodes L = {natoms, xyzq, type, R, e, cell, nimg, R_pp, e_pp, Q_pp, r_min, origin, step,
                               0, 0, NULL, NULL};
        grid_view g = g0;
        g.lazy = &L;
        relax_pixel(&g, &tp, &fp, &sc, (int)(flat % npx), (int)(flat / npx), m, total, pos_fz, iters, lam_min,
                    clamped_out, lam_traj);
        if (nodes_out) nodes_out[m] = L.used;
        free(L.keys);
        free(L.vals);
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------------------------
 * O9: Giessibl frequency shift, Eq.3, by exact product integration of the piecewise-linear interpolant of Fz.
 *   a = A/2, n = A/dz (integer >= 1), nodes q_m = -a + m dz (m = 0..n);
 *   y(q) = sqrt(a^2 - q^2), G(q) = (a^2/2) asin(q/a) - (q/2) y(q)      [ int q^2/y dq = G,  int q/y dq = -y ]
 *   per interval j: I1 = y_j - y_{j+1} (= int q/y), I2 = G_{j+1} - G_j (= int q^2/y)
 *     W_j += (q_{j+1} I1 - I2)/dz,  W_{j+1} += (I2 - q_j I1)/dz;  W *= 2/(pi a^2)
 *   df_k = -(f0/(2 k0)) * 16.02176634 * sum_m W_m Fz(z_c + q_m);  sample index of z_c + q_m is k + n - m.
 * ---------------------------------------------------------------------------------------------------------- */
int oracle_df_weights(int n, double dz, double *W /* n+1 */) {
    if (n < 1 || !(dz > 0.0)) return -1;
    double a = 0.5 * n * dz;
    for (int m = 0; m <= n; m++) W[m] = 0.0;
    for (int j = 0; j < n; j++) {
        double q0 = -a + j * dz, q1 = -a + (j + 1) * dz;
        if (j == n - 1) q1 = a; /* exact end point */
        double y0 = sqrt(fmax(a * a - q0 * q0, 0.0)), y1 = sqrt(fmax(a * a - q1 * q1, 0.0));
        double G0 = 0.5 * a * a * asin(fmax(-1.0, fmin(1.0, q0 / a))) - 0.5 * q0 * y0;
        double G1 = 0.5 * a * a * asin(fmax(-1.0, fmin(1.0, q1 / a))) - 0.5 * q1 * y1;
        double I1 = y0 - y1, I2 = G1 - G0;
        W[j] += (q1 * I1 - I2) / dz;
        W[j + 1] += (I2 - q0 * I1) / dz;
    }
    for (int m = 0; m <= n; m++) W[m] *= 2.0 / (M_PI * a * a);
    return 0;
}

int oracle_df(const double *fz /* [nz][npix] */, int64_t npix, int nz, double dz, double A, double k0 /* N/m */,
              double f0 /* Hz */, double *df /* [nz-n][npix] */) {
    double nn = A / dz;
    int n = (int)llround(nn);
    if (n < 1 || fabs(nn - n) > 1e-6 || nz <= n) return -1;
    double *W = (double *)malloc((size_t)(n + 1) * sizeof(double));
    if (!W) return -2;
    oracle_df_weights(n, dz, W);
    double pref = -(f0 / (2.0 * k0)) * EVA2_TO_NM;
#pragma omp parallel for schedule(static)
    for (int64_t p = 0; p < npix; p++)
        for (int k = 0; k < nz - n; k++) {
            double s = 0.0;
            for (int m = 0; m <= n; m++) s += W[m] * fz[(size_t)(k + n - m) * npix + p];
            df[(size_t)k * npix + p] = pref * s;
        }
    free(W);
    return 0;
}
