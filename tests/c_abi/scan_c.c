/* scan_c.c — the whole hot path driven from plain C99 through include/ppfm.h (no Python, no C++, no torch): a small
 * hard-coded molecule, device buffers from the CUDA runtime's C API, ppfm_forcefield -> ppfm_relax_scan -> ppfm_df, then
 * the same scan through ppfm_scan_host with host buffers.  Writes every output to the file named on the command line
 * (tests/test_c_abi_program.py compares it with the Python binding's results for the same input) and prints a summary.
 *
 *   gcc -std=c99 -Wall -Wextra -pedantic -Iinclude -I/usr/local/cuda/include tests/c_abi/scan_c.c \
 *       -Lpaper_2401_14564_b200 -lppfm -L/usr/local/cuda/lib64 -lcudart -lm -o scan_c
 */
#include <cuda_runtime_api.h>
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "ppfm.h"

#define CK(x)                                                                   \
    do {                                                                        \
        int rc_ = (x);                                                          \
        if (rc_ != 0) {                                                         \
            fprintf(stderr, "%s -> %d (%s)\n", #x, rc_, ppfm_strerror(rc_));    \
            return 1;                                                           \
        }                                                                       \
    } while (0)
#define CU(x)                                                                   \
    do {                                                                        \
        cudaError_t e_ = (x);                                                   \
        if (e_ != cudaSuccess) {                                                \
            fprintf(stderr, "%s -> %s\n", #x, cudaGetErrorString(e_));          \
            return 1;                                                           \
        }                                                                       \
    } while (0)

enum { NATOMS = 6, NX = 40, NY = 36, NZ = 44, NPX = 17, NPY = 13, NZS = 24, NDF = 10 };

int main(int argc, char **argv) {
    if (argc < 2) { fprintf(stderr, "usage: scan_c OUTPUT_FILE\n"); return 2; }
    if (ppfm_version() != PPFM_VERSION) {       /* built against another header than the library: argument lists may differ */
        fprintf(stderr, "libppfm is version %d, this program was built against ppfm.h version %d\n", ppfm_version(),
                PPFM_VERSION);
        return 3;
    }
    /* a ring of six atoms (types 1 = C, 0 = H alternating), charges summing to zero */
    float xyzq[NATOMS][4];
    int32_t type[NATOMS];
    const double R[2] = {1.487, 1.908}, e[2] = {6.81e-4, 3.73e-3};
    for (int i = 0; i < NATOMS; i++) {
        const double a = 2.0 * 3.14159265358979323846 * i / NATOMS;
        xyzq[i][0] = (float)(4.0 + 1.4 * cos(a));
        xyzq[i][1] = (float)(3.6 + 1.4 * sin(a));
        xyzq[i][2] = (float)(0.05 * (i % 3 - 1));
        xyzq[i][3] = (i % 2) ? 0.12f : -0.12f;
        type[i] = i % 2;
    }
    ppfm_lattice lat;
    memset(&lat, 0, sizeof(lat));
    lat.a[0] = 8.0; lat.b[1] = 7.2; lat.c[2] = 9.0;              /* non-periodic: nimg = 0 */
    ppfm_grid grid;
    memset(&grid, 0, sizeof(grid));
    grid.origin[2] = 1.2;
    grid.step[0][0] = grid.step[1][1] = grid.step[2][2] = 0.2;
    grid.n[0] = NX; grid.n[1] = NY; grid.n[2] = NZ;
    ppfm_probe probe = {1.661, 9.11e-3, -0.05};
    ppfm_tip tip;
    tip.k_lat[0] = tip.k_lat[1] = ppfm_Nm_to_eVA2(0.25);
    tip.k_rad = ppfm_Nm_to_eVA2(30.0);
    tip.d0[0] = tip.d0[1] = 0.0; tip.d0[2] = -4.0;
    ppfm_fire fire;
    ppfm_fire_default(&fire);
    ppfm_scan scan;
    memset(&scan, 0, sizeof(scan));
    scan.p0[0] = 2.43; scan.p0[1] = 2.37; scan.p0[2] = 9.5;
    scan.dx[0] = 0.2; scan.dy[1] = 0.2;
    scan.npx = NPX; scan.npy = NPY; scan.nz = NZS; scan.dz = 0.1;
    const double A = NDF * 0.1, k0 = 1800.0, f0 = 30300.0;

    const size_t npts = (size_t)NX * NY * NZ, nps = (size_t)NPX * NPY * NZS, ndf = (size_t)NPX * NPY * (NZS - NDF);
    float *d_xyzq, *d_ff, *d_pos, *d_df;
    int32_t *d_type;
    uint16_t *d_it;
    ppfm_stats *d_stats;
    CU(cudaMalloc((void **)&d_xyzq, sizeof(xyzq)));
    CU(cudaMalloc((void **)&d_type, sizeof(type)));
    CU(cudaMalloc((void **)&d_ff, npts * 16));
    CU(cudaMalloc((void **)&d_pos, nps * 16));
    CU(cudaMalloc((void **)&d_it, nps * 2));
    CU(cudaMalloc((void **)&d_df, ndf * 4));
    CU(cudaMalloc((void **)&d_stats, sizeof(ppfm_stats)));
    CU(cudaMemcpy(d_xyzq, xyzq, sizeof(xyzq), cudaMemcpyHostToDevice));
    CU(cudaMemcpy(d_type, type, sizeof(type), cudaMemcpyHostToDevice));
    CU(cudaMemset(d_stats, 0, sizeof(ppfm_stats)));

    CK(ppfm_forcefield(NATOMS, d_xyzq, d_type, 2, R, e, &lat, &probe, &grid, 0.1, d_ff, NULL, NULL));
    CK(ppfm_relax_scan(d_ff, &grid, &tip, &fire, &scan, d_pos, d_it, d_stats, NULL));
    CK(ppfm_df(d_pos, NPX, NPY, NZS, scan.dz, A, k0, f0, d_df, NULL));
    CU(cudaDeviceSynchronize());

    float *ff = (float *)malloc(npts * 16), *pos = (float *)malloc(nps * 16), *df = (float *)malloc(ndf * 4);
    float *pos_h = (float *)malloc(nps * 16), *df_h = (float *)malloc(ndf * 4);
    uint16_t *it = (uint16_t *)malloc(nps * 2), *it_h = (uint16_t *)malloc(nps * 2);
    ppfm_stats st, st_h;
    if (!ff || !pos || !df || !pos_h || !df_h || !it || !it_h) return 3;
    CU(cudaMemcpy(ff, d_ff, npts * 16, cudaMemcpyDeviceToHost));
    CU(cudaMemcpy(pos, d_pos, nps * 16, cudaMemcpyDeviceToHost));
    CU(cudaMemcpy(it, d_it, nps * 2, cudaMemcpyDeviceToHost));
    CU(cudaMemcpy(df, d_df, ndf * 4, cudaMemcpyDeviceToHost));
    CU(cudaMemcpy(&st, d_stats, sizeof(st), cudaMemcpyDeviceToHost));

    /* the same scan in one call with (pageable) host buffers */
    CK(ppfm_scan_host(NATOMS, &xyzq[0][0], type, 2, R, e, &lat, &probe, &grid, 0.1, &tip, &fire, &scan, A, k0, f0, pos_h,
                      it_h, df_h, &st_h, NULL));
    int same = memcmp(pos, pos_h, nps * 16) == 0 && memcmp(it, it_h, nps * 2) == 0 && memcmp(df, df_h, ndf * 4) == 0 &&
               st.total_iters == st_h.total_iters;

    FILE *f = fopen(argv[1], "wb");
    if (!f) return 4;
    fwrite(xyzq, 1, sizeof(xyzq), f);
    fwrite(ff, 16, npts, f);
    fwrite(pos, 16, nps, f);
    fwrite(it, 2, nps, f);
    fwrite(df, 4, ndf, f);
    fclose(f);
    double dmin = 1e30, dmax = -1e30;
    for (size_t i = 0; i < ndf; i++) { if (df[i] < dmin) dmin = df[i]; if (df[i] > dmax) dmax = df[i]; }
    printf("ppfm %d: %zu grid points, %zu pixel-steps, %llu FIRE moves, %llu not converged, df in [%.3f, %.3f] Hz, "
           "host path %s\n", ppfm_version(), npts, nps, (unsigned long long)st.total_iters,
           (unsigned long long)st.n_not_converged, dmin, dmax, same ? "identical" : "DIFFERENT");
    CK(ppfm_release_scratch());
    cudaFree(d_xyzq); cudaFree(d_type); cudaFree(d_ff); cudaFree(d_pos); cudaFree(d_it); cudaFree(d_df); cudaFree(d_stats);
    free(ff); free(pos); free(df); free(pos_h); free(df_h); free(it); free(it_h);
    return same ? 0 : 5;
}
