/*
 * ppfm.h — C ABI of libppfm: the Probe-Particle Model hot path on one NVIDIA B200 (sm_100a).
 *
 * Paper: arxiv 2401.14564 ("PAPER.md" below = /root/reference/PAPER.md, cited by line).  The library implements
 * the simplest level of theory (Lennard-Jones + point charges) of the two-step scheme of
 * (1) project all sample atoms onto a uniform grid force field, (2) relax the probe particle
 * (PP) with FIRE under tri-linear interpolation of that grid plus the tip springs, for every scan pixel while
 * the tip steps down in z, and (3) convert Fz(z) to the frequency shift df.  Beyond that path:
 * (1b) Eq.7 electrostatics of an extended tip charge density and (1c) the Eq.8 Pauli overlap, both by the
 * convolution theorem; (2a) the scan with tri-cubic interpolation of an energy-only grid
 * (PAPER.md:264); (2b) the stiffness map of the relaxed PP (IETS module).
 *
 * Conventions
 *   Units: Å, eV, elementary charge e; spring constants in eV/Å^2 (ppfm_Nm_to_eVA2 converts from N/m);
 *          k0 in N/m and f0 in Hz (ppfm_df).  k_e = 14.399645478 eV·Å/e^2;  1 eV/Å^2 = 16.02176634 N/m.
 *   Pointers: a `d_` prefix = DEVICE memory on the current CUDA device, `h_` prefix = HOST memory.  Structs
 *          passed by pointer are HOST memory and are read before the call returns.
 *   Ownership: every buffer is allocated and freed by the caller.  The library keeps no pointer to caller memory
 *          after return; per-call scratch is stream-ordered (allocated and freed on `cuda_stream` inside the call)
 *          from a library-private pool that caches freed blocks until ppfm_release_scratch(); the cuFFT plans and
 *          tip spectra of (1b)/(1c) are cached until then too (the one persistent device allocation the library makes).
 *          Device entry points only enqueue work on `cuda_stream` (a cudaStream_t cast to
 *          void*, NULL = default stream); they never synchronise it and never change the current device.
 *          Host entry points (ppfm_scan_host, _batch, _sweep) synchronise the stream before returning.
 *   Threads and streams: every entry point may be called from several host threads and on several streams at once.
 *          Calls on one stream execute in order; calls on different streams may overlap on the device and share
 *          nothing but read-only caches (the cuFFT plans and tip spectra of (1b)/(1c) are guarded by a mutex on the
 *          host and by events on the device; each call brings its own cuFFT work area).
 *   Errors: 0 on success, a negative ppfm_status otherwise; no exceptions, no exit(), no output.  Per-pixel
 *          conditions (not converged, PP clamped at a non-periodic grid face) are data (d_iters, d_stats).
 *   Determinism: outputs are bit-reproducible run to run (fixed summation order, no atomics on results).
 *   Layouts: force-field grid  float[nz][ny][nx][4] = (Fx, Fy, Fz, E), x fastest;
 *            scan output       float[nzs][npy][npx][4] = (PPx, PPy, PPz, Fz_tip);
 *            df                float[nzs - n][npy][npx], n = A/dz.
 */
#ifndef PPFM_H
#define PPFM_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* ABI version of THIS header.  ppfm_version() returns the value the loaded library was built with; a client should
 * compare the two once at start-up (the Python binding and tests/c_abi/scan_c.c do) and refuse to run on a mismatch:
 * an argument list that differs between header and library is not detectable any other way from C.
 * 200 (0.2.0): the force-field calls take a ppfm_ff_status* before cuda_stream (incompatible with 100); the probe /
 *              timing / launch-count exports moved to ppfm_bench.h; ppfm_forcefield_noalloc and PPFM_ELIMIT added. */
#define PPFM_VERSION 200 /* 0.2.0 */
#define PPFM_MAX_TYPES 64
#define PPFM_DF_MAX_N 255 /* largest n = A/dz of ppfm_df */

typedef enum {
    PPFM_OK = 0,
    PPFM_EINVAL = -1, /* null pointer, n <= 0, singular step matrix, A/dz not an integer, nz <= n, bad type index */
    PPFM_ECUDA = -2,  /* CUDA runtime / launch error; text via ppfm_strerror(PPFM_ECUDA) (thread-local)          */
    PPFM_ENOMEM = -3, /* scratch allocation failed                                                              */
    PPFM_ELIMIT = -4  /* input larger than the fixed scratch of an entry point that allocates nothing
                         (ppfm_forcefield_noalloc: natoms > PPFM_NOALLOC_MAX_ATOMS)                             */
} ppfm_status;

/* Supercell vectors (Å) and periodic images: the sum runs over shifts na*a + nb*b + nc*c with
 * n? in [-nimg[?], +nimg[?]]; nimg = 0 on a non-periodic axis. */
typedef struct {
    double a[3], b[3], c[3];
    int32_t nimg[3];
} ppfm_lattice;

/* Uniform grid: point(i,j,k) = origin + i*step[0] + j*step[1] + k*step[2], i < n[0] etc..
 * periodic[ax] != 0: interpolation wraps that axis (n[ax]*step[ax] must be the cell vector); 0: clamps. */
typedef struct {
    double origin[3];
    double step[3][3];
    int32_t n[3];
    int32_t periodic[3];
} ppfm_grid;

/* Probe particle: LJ radius R_PP (Å), well depth e_PP (eV), point charge q_PP (e). */
typedef struct {
    double R, e, Q;
} ppfm_probe;

/* Tip springs of Eq.2: k_lat = (k_x, k_y), k_rad = k_R, d0 = equilibrium displacement of the PP
 * from the anchor (e.g. (0,0,-4): PP hangs 4 Å below the anchor); R0 of Eq.2 is |d0|. */
typedef struct {
    double k_lat[2];
    double k_rad;
    double d0[3];
} ppfm_tip;

/* FIRE parameters (ref [7]); ppfm_fire_default() gives dt = dt_max = 0.5, finc 1.1, fdec 0.5,
 * alpha0 0.1, falpha 0.99, n_min 5, max_iter 1000, f_conv 1e-6 eV/Å. */
typedef struct {
    double dt, dt_max, finc, fdec, alpha0, falpha;
    int32_t n_min, max_iter;
    double f_conv;
} ppfm_fire;

/* Scan: tip anchor(ix,iy,iz) = p0 + ix*dx + iy*dy - (0,0,iz*dz), iz = 0 is the far end. */
typedef struct {
    double p0[3], dx[3], dy[3];
    int32_t npx, npy, nz;
    double dz;
} ppfm_scan;

/* Counters accumulated (+=, max) by ppfm_relax_scan into a DEVICE struct the caller zeroes. */
typedef struct {
    uint64_t total_iters;     /* FIRE moves summed over all pixel-steps                   */
    uint64_t n_not_converged; /* pixel-steps that used max_iter moves without converging  */
    uint64_t n_clamped;       /* pixel-steps whose final PP position was clamped to a non-periodic grid face */
    uint32_t max_iters;       /* largest move count of any pixel-step                     */
    uint32_t _pad;
    uint64_t warp_iters;      /* trips of the warp-converged FIRE loop, summed over warps (x32 lanes = issued lane-
                                 iterations; minus total_iters = divergence cost)             */
    uint64_t cell_gathers;    /* lane-iterations in which the PP had left the grid cell the lane holds in registers */
    uint64_t warp_gathers;    /* warp loop trips that executed the 8-corner float4 gather (all 32 lanes gather when
                                 any lane left its cell)                                        */
} ppfm_stats;

int ppfm_version(void);
/* Message for a status code; for PPFM_ECUDA the text of the last CUDA error seen on this thread. */
const char *ppfm_strerror(int code);
void ppfm_fire_default(ppfm_fire *out);
double ppfm_Nm_to_eVA2(double k_Nm);

/* ---- (1) force-field grid: Eq.5 + Eq.6 summed over atoms and images ------------------
 * d_xyzq   DEVICE float[natoms][4] = (x, y, z, q_i), 16-byte aligned
 * d_type   DEVICE int32[natoms], index into h_R / h_e.  It is device memory, so it is validated on the device: an atom
 *          whose index is outside [0, ntypes) contributes nothing and is counted in d_status->n_bad_type
 * h_R,h_e  HOST double[ntypes]: element radius R_i (Å) and well depth e_i (eV); mixing R_i + R_PP, sqrt(e_i e_PP)
 * r_min    pair distances are clamped below at r_min (Å) to keep the sum finite on top of an atom; >= 0
 * d_ff     DEVICE float[n2][n1][n0][4], 16-byte aligned, written completely
 * d_status DEVICE ppfm_ff_status or NULL: per-call conditions that are data, not errors (written, not accumulated;
 *          batch form: summed over the systems)
 */
typedef struct {
    uint32_t n_bad_type;   /* atoms skipped because their type index was outside [0, ntypes)                       */
    uint32_t n_clamped;    /* systems in which some atom image lies within r_min of the grid's bounding box, i.e.
                              for which the r_min clamp was compiled into the pair loop                             */
} ppfm_ff_status;
int ppfm_forcefield(int32_t natoms, const float *d_xyzq, const int32_t *d_type, int32_t ntypes, const double *h_R,
                    const double *h_e, const ppfm_lattice *lattice, const ppfm_probe *probe, const ppfm_grid *grid,
                    double r_min, float *d_ff, ppfm_ff_status *d_status, void *cuda_stream);

/* Same pass, two grids (LJ and electrostatic fields are kept separately so the tip charge can
 * change without recomputation): d_ff_lj = Lennard-Jones only, d_ff_el = Coulomb field of a UNIT probe charge
 * (probe->Q is ignored).  Combine with ppfm_combine. */
int ppfm_forcefield_split(int32_t natoms, const float *d_xyzq, const int32_t *d_type, int32_t ntypes,
                          const double *h_R, const double *h_e, const ppfm_lattice *lattice,
                          const ppfm_probe *probe, const ppfm_grid *grid, double r_min, float *d_ff_lj,
                          float *d_ff_el, ppfm_ff_status *d_status, void *cuda_stream);

/* d_out = d_ff_lj + Q * d_ff_el over n_points float4 entries (d_out may alias d_ff_lj). */
int ppfm_combine(const float *d_ff_lj, const float *d_ff_el, double Q, int64_t n_points, float *d_out,
                 void *cuda_stream);

/* Batch of independent systems in ONE launch (ML-style batches).  Atoms are concatenated:
 * system m owns atoms h_atom_offset[m] .. h_atom_offset[m+1]-1; grids are concatenated in d_ff in order
 * (system m starts at float4 offset sum_{l<m} n0*n1*n2).  Arrays of structs are HOST arrays of length nsys. */
int ppfm_forcefield_batch(int32_t nsys, const int32_t *h_atom_offset, const float *d_xyzq, const int32_t *d_type,
                          int32_t ntypes, const double *h_R, const double *h_e, const ppfm_lattice *lattices,
                          const ppfm_probe *probes, const ppfm_grid *grids, double r_min, float *d_ff,
                          ppfm_ff_status *d_status, void *cuda_stream);

/* ---- (1') the same force-field pass for callers that must not allocate ---------------------------------------
 * Who this is for.  ppfm_forcefield takes its per-call scratch (the packed atom records and two per-system flags
 * that its set-up kernel writes and its grid kernel reads) from a stream-ordered memory pool.  Some callers cannot
 * tolerate that: code that runs under a fixed memory budget where every byte of the device has been handed out
 * beforehand (an inference / simulation server that pre-allocates its arena and treats any later allocation as a
 * fault), a real-time acquisition loop next to the microscope that must not hit an allocator lock or a driver call
 * of unbounded latency, and hosts embedding the library behind an allocator hook that forbids cudaMalloc* outside
 * start-up.  For them this entry point computes exactly what ppfm_forcefield computes (same kernels, same
 * summation order, bit-identical grid) but keeps the scratch in a fixed array inside the library image.
 *
 *   Limit:     natoms <= PPFM_NOALLOC_MAX_ATOMS (16384; the paper's largest systems are a few thousand atoms).
 *              More atoms: PPFM_ELIMIT, nothing is launched and nothing is written.  The grid size is not limited
 *              (the grid is the caller's buffer).
 *   Cost:      PPFM_NOALLOC_SCRATCH_BYTES (768 KiB + 256 B) of device memory on EVERY GPU on which the library is
 *              loaded, from the moment its code is loaded there until the process exits, whether or not this
 *              entry point is ever called.
 *   No allocation: the call makes no cudaMalloc / cudaMallocAsync / cudaFree / pool call, no host malloc, and calls
 *              no library routine that allocates; the optional per-kernel timers of ppfm_bench.h do not see its
 *              launches (they would create events).  It enqueues one 8-byte memset, the status memset if d_status
 *              is given, and the two kernels on `cuda_stream`, and returns without synchronising.
 *   First call on a device: looks up the device address of the scratch array (cudaGetSymbolAddress, once per
 *              device, with that device current — the caller must have made the device current, as for every other
 *              entry point) and remembers it.  That look-up may load the library's device code; make this first
 *              call during start-up, before any stream capture is begun.
 *   Sharing:   there is ONE array per device and every call on that device uses it.  The array keeps what the
 *              previous call left; the call re-zeroes the flags it depends on and overwrites the records it reads,
 *              so calls that follow one another on one stream are independent.  Two calls whose kernels can
 *              overlap on the GPU (different streams, or different host threads on different streams) RACE on the
 *              array and produce garbage: order them yourself (one stream, or events).  ppfm_forcefield has no
 *              such restriction.
 *   Arguments, layouts and the other error codes are those of ppfm_forcefield. */
#define PPFM_NOALLOC_MAX_ATOMS 16384
#define PPFM_NOALLOC_SCRATCH_BYTES (256 + 48 * PPFM_NOALLOC_MAX_ATOMS)
int ppfm_forcefield_noalloc(int32_t natoms, const float *d_xyzq, const int32_t *d_type, int32_t ntypes,
                            const double *h_R, const double *h_e, const ppfm_lattice *lattice,
                            const ppfm_probe *probe, const ppfm_grid *grid, double r_min, float *d_ff,
                            ppfm_ff_status *d_status, void *cuda_stream);

/* ---- (1e) energy-only grid for the tri-cubic scan ("tri-cubic interpolation of the potential ...
 * avoid storage of forces (i.e. improve memory efficiency)") ---------------------------------------------------
 * The same sum as ppfm_forcefield, but only E = E_LJ + E_C is accumulated and stored: d_E is DEVICE
 * float[n2][n1][n0] (4-byte aligned, 4 bytes per point instead of 16, written completely) in the layout
 * ppfm_relax_scan_tricubic reads.  The pair loop carries no force arithmetic (8 packed instructions + 2 MUFU per
 * pair of points against 15 + 2).  Every 256-atom partial sum is folded into an FP64 total per point, so the
 * node-to-node noise the tri-cubic derivative stencil would amplify stays at the FP32 rounding of one chunk's terms
 * (measured: <= 3e-7 eV where |E| < 1e-2 eV on configs 0-2; parity |dE| <= 1e-4 |E| + 5e-7 eV there).  All other
 * arguments, d_status and the error codes are ppfm_forcefield's; probe->Q is the tip charge. */
int ppfm_forcefield_energy(int32_t natoms, const float *d_xyzq, const int32_t *d_type, int32_t ntypes,
                           const double *h_R, const double *h_e, const ppfm_lattice *lattice,
                           const ppfm_probe *probe, const ppfm_grid *grid, double r_min, float *d_E,
                           ppfm_ff_status *d_status, void *cuda_stream);

/* ---- (2) relaxation scan: Eq.1 + Eq.2 + FIRE on the tri-linearly interpolated grid --
 * d_ff      DEVICE grid as written by ppfm_forcefield (read-only)
 * d_pos_fz  DEVICE float[nz][npy][npx][4] = relaxed PP position and Fz_tip = -F_R,z
 * d_iters   DEVICE uint16[nz][npy][npx] or NULL: FIRE moves made; 0xFFFF = max_iter reached without converging
 * d_stats   DEVICE ppfm_stats or NULL (accumulated)
 * Per pixel: iz = 0 starts at r_TIP + d0 with v = 0; each further z-step carries the displacement d over and
 * resets the FIRE state.  Convergence: |F_total|_2 < f_conv, tested before every move.
 */
int ppfm_relax_scan(const float *d_ff, const ppfm_grid *grid, const ppfm_tip *tip, const ppfm_fire *fire,
                    const ppfm_scan *scan, float *d_pos_fz, uint16_t *d_iters, ppfm_stats *d_stats,
                    void *cuda_stream);

/* Batch form: nsys scans in one launch; grids concatenated as in ppfm_forcefield_batch, outputs concatenated in
 * order (system m starts at pixel-step offset sum_{l<m} nz*npy*npx).  One fire setting for all. */
int ppfm_relax_scan_batch(int32_t nsys, const float *d_ff, const ppfm_grid *grids, const ppfm_tip *tips,
                          const ppfm_fire *fire, const ppfm_scan *scans, float *d_pos_fz, uint16_t *d_iters,
                          ppfm_stats *d_stats, void *cuda_stream);

/* Sweep form (the stored grids exist "so that" tip parameters "can change without recomputation"):
 * nscan scans on ONE resident grid in one launch.  `grid` is a single HOST struct and d_ff that one grid; tips[m]
 * and scans[m] (HOST arrays of length nscan) give scan m its own springs (k_x, k_y, k_R), equilibrium displacement
 * d0 (length and tilt) and scan geometry.  Outputs are concatenated in order as in the batch form.  Nothing is
 * replicated: a k_xy / k_R / d0 sweep costs the memory of one grid.  (A tip-CHARGE sweep changes the grid itself:
 * ppfm_forcefield_split + ppfm_combine per Q, then the batch form.)  Results equal those of ppfm_relax_scan_batch
 * on nscan copies of the grid bit for bit. */
int ppfm_relax_scan_sweep(int32_t nscan, const float *d_ff, const ppfm_grid *grid, const ppfm_tip *tips,
                          const ppfm_fire *fire, const ppfm_scan *scans, float *d_pos_fz, uint16_t *d_iters,
                          ppfm_stats *d_stats, void *cuda_stream);

/* ---- (1b) electrostatics of an extended tip charge density, Eq.7 -----
 *     E_el(R) = integral rho_PP(r) V_S(r + R) dr,   F_el(R) = -grad_R E_el = integral grad rho_PP(r) V_S(r + R) dr
 * by the convolution theorem (cuFFT, FP64) on the grid, which is taken as periodic in all three axes: the integral
 * is the cyclic sum over the nodes times dV = |det(step)|.  rho_PP is a Gaussian multipole centred on the PP,
 *     rho(r) = [ q_s + p_z z / sigma^2 + (Q_zz / 12) (3 z^2 - r^2) / sigma^4 ] (2 pi sigma^2)^(-3/2) exp(-r^2 / 2 sigma^2)
 * (charge q_s in e, dipole p_z in e Å, quadrupole Q_zz = integral rho (3z^2 - r^2) in e Å^2; the paper quotes -0.025 to
 * -0.15 e Å^2 for CO tips), sampled with its analytic gradient at the nodes (minimum image by index).  Keep
 * sigma >= ~1.5 grid steps and <= ~1/7 of the shortest cell edge.
 * d_V   DEVICE float[nz][ny][nx]: sample potential V_S in eV per unit charge (e.g. the .w lane of the unit-charge
 *       grid of ppfm_forcefield_split, or a Hartree potential)
 * d_ff  DEVICE float[nz][ny][nx][4] = (Fx, Fy, Fz, E_el); add to an LJ grid with ppfm_combine(lj, d_ff, 1.0, ...)
 * The library caches the cuFFT plans per grid size (without work areas: every call binds its own from the scratch
 * pool) and the four tip spectra of the two most recently used (grid, tip density) pairs (4 x nz*ny*(nx/2+1) complex
 * doubles each, device memory) until ppfm_release_scratch(): a run of calls on one grid with one tip costs one
 * forward and four inverse transforms each ("amortized if a batch of simulations is run using the
 * same grid").
 */
typedef struct {
    double sigma;   /* Gaussian width (Å)        */
    double q_s;     /* monopole (e)              */
    double p_z;     /* dipole along z (e Å)      */
    double Q_zz;    /* quadrupole (e Å^2)        */
} ppfm_tip_density;
int ppfm_forcefield_fft(const float *d_V, const ppfm_grid *grid, const ppfm_tip_density *tip, float *d_ff,
                        void *cuda_stream);

/* ---- (1c) Pauli repulsion of the full density-based model, Eq.8 ---------------------------------
 *     E_Pauli(R) = A integral [ rho_PP(r) rho_S(r + R) ]^beta dr,   F = -grad_R E_Pauli,
 * on the periodic grid as in (1b), with rho_PP = q_tip g_sigma(r) (a Gaussian electron density of q_tip > 0 electrons).
 * d_rho_S  DEVICE float[nz][ny][nx]: sample electron density (e/Å^3); negative values are clipped to 0.
 * d_ff     DEVICE float[nz][ny][nx][4] = (Fx, Fy, Fz, E_Pauli); A in eV Å^(3(2 beta - 1)) e^(-2 beta), beta > 0.
 */
int ppfm_forcefield_pauli(const float *d_rho_S, const ppfm_grid *grid, double sigma, double q_tip, double A, double beta,
                          float *d_ff, void *cuda_stream);

/* ---- (2a) relaxation scan on an energy-only grid, tri-cubic interpolation -------
 * "we are experimenting with tri-cubic interpolation of the potential which may allow us to use larger grid spacing
 * and avoid storage of forces".  Same scan, FIRE and outputs as ppfm_relax_scan; the sample force is
 * F_S = -grad of the tri-cubic interpolant of E: per axis the interpolating cubic convolution kernel (Catmull-Rom,
 * a = -1/2) on the nodes i0-1 .. i0+2 around the cell, tensor product; stencil indices wrap on periodic axes and are
 * clamped to [0, n-1] on the others; the coordinate is clamped as in ppfm_relax_scan.
 * d_E  DEVICE float[nz][ny][nx]: potential energy of the PP (eV), e.g. from ppfm_energy_grid (the .w lane of a
 *      force-field grid; 4 bytes per point instead of 16).  Batch form: grids concatenated.
 */
int ppfm_relax_scan_tricubic(const float *d_E, const ppfm_grid *grid, const ppfm_tip *tip, const ppfm_fire *fire,
                             const ppfm_scan *scan, float *d_pos_fz, uint16_t *d_iters, ppfm_stats *d_stats,
                             void *cuda_stream);
int ppfm_relax_scan_tricubic_batch(int32_t nsys, const float *d_E, const ppfm_grid *grids, const ppfm_tip *tips,
                                   const ppfm_fire *fire, const ppfm_scan *scans, float *d_pos_fz,
                                   uint16_t *d_iters, ppfm_stats *d_stats, void *cuda_stream);
/* d_E[i] = d_ff[i][3] for n_points grid points (both DEVICE). */
int ppfm_energy_grid(const float *d_ff, int64_t n_points, float *d_E, void *cuda_stream);

/* ---- (2b) stiffness map of the relaxed probe particle (IETS module) ------
 * "This module calculates the change of the stiffness (resp. vibration frequency) of lateral vibration modes of the
 * CO molecule attached to the AFM tip due to its interaction with the sample."  For every (pixel, z-step) sample the
 * Hessian of the PP's total potential at the given position,
 *     H = H_spring - (J + J^T)/2,   J = dF_S/dr  (analytic Jacobian of the tri-linear interpolant in the cell),
 *     H_spring = k_R dd^T/|d|^2 + k_R (|d| - R0)/|d| (I - dd^T/|d|^2) + diag(k_x, k_y, 0),   d = r_PP - r_TIP,
 * and its three eigenvalues.
 * d_ff      DEVICE grid as written by ppfm_forcefield (read-only)
 * d_pos_fz  DEVICE float[nz][npy][npx][4] as written by ppfm_relax_scan (x, y, z read; .w ignored)
 * d_eig     DEVICE float[nz][npy][npx][4] = (lambda_1 <= lambda_2 <= lambda_3, 0) in eV/Å^2.  Without sample
 *           interaction the two small ones are k_x, k_y (the lateral CO modes) and the large one is k_R.
 * Outside a non-periodic grid the position is clamped (as in the relaxation) before the cell is taken.
 */
int ppfm_stiffness(const float *d_ff, const ppfm_grid *grid, const ppfm_tip *tip, const ppfm_scan *scan,
                   const float *d_pos_fz, float *d_eig, void *cuda_stream);
int ppfm_stiffness_batch(int32_t nsys, const float *d_ff, const ppfm_grid *grids, const ppfm_tip *tips,
                         const ppfm_scan *scans, const float *d_pos_fz, float *d_eig, void *cuda_stream);
/* The relaxation scan with the stiffness map folded in: at the end of every z-step the lane that relaxed the pixel
 * forms J from the grid cell it still holds in registers (no second gather, no second launch) and writes the three
 * eigenvalues of H at the relaxed point to d_eig (same layout as above; FP32 throughout, the eigenvalues by
 * deflation on the isolated root so that the two nearly degenerate lateral modes keep full FP32 accuracy).  All other
 * arguments and outputs as ppfm_relax_scan[_batch]; d_eig must not be NULL.  ppfm_stiffness remains the entry point
 * for positions that do not come straight from a scan.  (The Jacobian of a tri-linear interpolant jumps across cell
 * faces: for a point exactly on a face the folded map uses the cell the relaxation held, ppfm_stiffness the cell
 * floor() picks from the stored FP32 position; the two can then differ by that jump.) */
int ppfm_relax_scan_stiffness(const float *d_ff, const ppfm_grid *grid, const ppfm_tip *tip, const ppfm_fire *fire,
                              const ppfm_scan *scan, float *d_pos_fz, uint16_t *d_iters, float *d_eig,
                              ppfm_stats *d_stats, void *cuda_stream);
int ppfm_relax_scan_stiffness_batch(int32_t nsys, const float *d_ff, const ppfm_grid *grids, const ppfm_tip *tips,
                                    const ppfm_fire *fire, const ppfm_scan *scans, float *d_pos_fz, uint16_t *d_iters,
                                    float *d_eig, ppfm_stats *d_stats, void *cuda_stream);

/* ---- (3) frequency shift, Giessibl's formula Eq.3 -------------------------------------------
 * Fz is read from the .w lane of d_pos_fz [nz][npy][npx][4].  A = peak-to-peak amplitude (Å); n = A/dz must be an
 * integer (within 1e-6) with 1 <= n <= PPFM_DF_MAX_N (the weights travel as a kernel parameter) and nz > n; the
 * host entry points check the same before any work is enqueued.  Eq.3 is integrated exactly for the piecewise-linear interpolant of the
 * n+1 samples of each window; output plane k belongs to tip height z0 - (k + n/2) dz.
 * d_df  DEVICE float[nz - n][npy][npx] (Hz).  ppfm_df_weights writes the n+1 quadrature weights to HOST memory.
 * The batch count `nsys` treats d_pos_fz / d_df as nsys consecutive stacks of identical shape.
 */
int ppfm_df(const float *d_pos_fz, int32_t npx, int32_t npy, int32_t nz, double dz, double A, double k0_Nm,
            double f0_Hz, float *d_df, void *cuda_stream);
int ppfm_df_batch(int32_t nsys, const float *d_pos_fz, int32_t npx, int32_t npy, int32_t nz, double dz, double A,
                  double k0_Nm, double f0_Hz, float *d_df, void *cuda_stream);
int ppfm_df_weights(int32_t n, double dz, double *h_W);

/* ---- whole simulation in one call, HOST buffers in and out ("run the whole simulation in one step")
 * Copies the inputs to the device, runs (1) -> (2) -> (3) on `cuda_stream`, copies the results back and
 * synchronises the stream.  h_pos_fz / h_df / h_iters may each be NULL (not copied back); h_stats may be NULL.
 * When the output buffers are pinned (page-locked, UVA-mapped) host memory the kernels store straight into them:
 * the PCIe writes overlap the computation and no device-to-host copy follows the scan.  Pageable buffers work too
 * (staged copies after the kernels).  The batch form runs nsys systems in one launch per step (arguments as in the
 * *_batch entry points, outputs concatenated in order; with h_df all scans must have one shape).
 */
int ppfm_scan_host(int32_t natoms, const float *h_xyzq, const int32_t *h_type, int32_t ntypes, const double *h_R,
                   const double *h_e, const ppfm_lattice *lattice, const ppfm_probe *probe, const ppfm_grid *grid,
                   double r_min, const ppfm_tip *tip, const ppfm_fire *fire, const ppfm_scan *scan, double A,
                   double k0_Nm, double f0_Hz, float *h_pos_fz, uint16_t *h_iters, float *h_df,
                   ppfm_stats *h_stats, void *cuda_stream);
int ppfm_scan_host_batch(int32_t nsys, const int32_t *h_atom_offset, const float *h_xyzq, const int32_t *h_type,
                         int32_t ntypes, const double *h_R, const double *h_e, const ppfm_lattice *lattices,
                         const ppfm_probe *probes, const ppfm_grid *grids, double r_min, const ppfm_tip *tips,
                         const ppfm_fire *fire, const ppfm_scan *scans, double A, double k0_Nm, double f0_Hz,
                         float *h_pos_fz, uint16_t *h_iters, float *h_df, ppfm_stats *h_stats, void *cuda_stream);

/* Tip-charge sweep (the LJ and electrostatic grids are separate so that the tip charge can change
 * without recomputation; reading S19): F_LJ and the unit-charge F_el are sampled once, then for each of the nQ
 * charges h_Q[i] the grids are combined and the scan + df run (the nQ scans as one batch launch while the nQ combined
 * grids fit 8 GiB of scratch, one after the other beyond that; the results do not depend on which).  Outputs hold nQ
 * consecutive result sets:
 * h_pos_fz float[nQ][nz][npy][npx][4], h_iters uint16[nQ][nz][npy][npx], h_df float[nQ][nz-n][npy][npx]; h_stats
 * accumulates over the sweep.  probe->Q is ignored. */
int ppfm_scan_host_sweep(int32_t nQ, const double *h_Q, int32_t natoms, const float *h_xyzq, const int32_t *h_type,
                         int32_t ntypes, const double *h_R, const double *h_e, const ppfm_lattice *lattice,
                         const ppfm_probe *probe, const ppfm_grid *grid, double r_min, const ppfm_tip *tip,
                         const ppfm_fire *fire, const ppfm_scan *scan, double A, double k0_Nm, double f0_Hz,
                         float *h_pos_fz, uint16_t *h_iters, float *h_df, ppfm_stats *h_stats, void *cuda_stream);

/* Scratch memory.  Per-call scratch (packed atom records, job tables; for ppfm_scan_host also the grid and the
 * scan buffers) comes from a library-private stream-ordered pool of the current device, so steady-state calls make
 * no driver allocation.  Freed blocks stay cached in that pool; ppfm_release_scratch() returns them to the driver
 * (call it when the stream work has completed). */
int ppfm_release_scratch(void);

#ifdef __cplusplus
}
#endif
#endif /* PPFM_H */
