// common.cuh — shared host-side plumbing of libppfm (error capture, launch counting, small math helpers).
// CUDA path only; the CPU oracle under oracle/ shares nothing with this tree.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstring>

#include "../../include/ppfm.h"
#include "../../include/ppfm_bench.h"

namespace ppfm {

// Coulomb constant k_e in eV*Angstrom/e^2 (Eq.6) and eV/Angstrom^2 -> N/m (exact SI e).
constexpr double kCoulomb = 14.399645478;
constexpr double kEVA2toNm = 16.02176634;

void set_cuda_error(cudaError_t e, const char *where);
extern std::atomic<long long> g_launches;
inline void count_launch(int n = 1) { g_launches.fetch_add(n, std::memory_order_relaxed); }

// Stream-ordered scratch from the library's private memory pool of the current device (api.cu): freed blocks stay
// in the pool across calls (no driver allocation on the steady-state path) until ppfm_release_scratch().
cudaError_t scratch_alloc(void **ptr, size_t bytes, cudaStream_t st);
void release_fft_plans();   // fftel.cu: cached cuFFT plans
// Internal forms used by ppfm_scan_host[_batch] (api.cu) when the caller's output buffers are mapped host memory:
// the relaxation also writes a plain Fz stack (device) for the df kernel, which then reads that instead of the
// float4 stack.
int relax_scan_fz(int nsys, const float *d_ff, const ppfm_grid *grids, const ppfm_tip *tips, const ppfm_fire *fire,
                  const ppfm_scan *scans, float *d_pos_fz, uint16_t *d_iters, ppfm_stats *d_stats, float *d_fz,
                  void *cuda_stream);
int df_from_fz(int nsys, const float *d_fz, int npx, int npy, int nz, double dz, double A, double k0, double f0,
               float *d_df, void *cuda_stream);

// Optional per-kernel device timing (ppfm_timing_enable / ppfm_timing_read): CUDA events recorded on the launching
// stream immediately around one kernel launch.  Costs nothing when timing is off.
extern std::atomic<int> g_timing_on;
void timing_begin(int kernel_id, cudaStream_t st, cudaEvent_t *e0);
void timing_end(int kernel_id, cudaStream_t st, cudaEvent_t e0);
struct KernelTimer {
    int id;
    cudaStream_t st;
    cudaEvent_t e0 = nullptr;
    bool on;
    KernelTimer(int kernel_id, cudaStream_t stream) : id(kernel_id), st(stream) {
        on = g_timing_on.load(std::memory_order_relaxed) != 0;
        if (on) timing_begin(id, st, &e0);
    }
    ~KernelTimer() {
        if (on) timing_end(id, st, e0);
    }
};

// Checked build (libppfm_chk.so, -DPPFM_CHECKS; compute-sanitizer is closed on the GPU pool this was developed on): every
// global store / gather index is tested against its buffer's extent and the force-field kernel's shared-memory ring
// is compared with the global atom records when a chunk is acquired (a stage read before its copy landed) and again
// when it is released (a stage overwritten while still in use).  Failures are counted per kind, never trapped;
// ppfm_checks_read (include/ppfm_bench.h) returns the counts.  The product build compiles none of this.
enum { PPFM_CHK_RING_ACQUIRE = 0, PPFM_CHK_RING_RELEASE = 1, PPFM_CHK_FF_STORE = 2, PPFM_CHK_RELAX_GATHER = 3,
       PPFM_CHK_RELAX_STORE = 4, PPFM_CHK_DF_LOAD = 5, PPFM_CHK_DF_STORE = 6, PPFM_CHK_VISITS = 7, PPFM_CHK_KINDS = 8 };
#ifdef PPFM_CHECKS
#define PPFM_CHK_STORAGE                                                                          \
    static __device__ unsigned long long g_chk[PPFM_CHK_KINDS];                                   \
    void PPFM_CHK_READER(unsigned long long *out) {                                               \
        unsigned long long h[PPFM_CHK_KINDS] = {}, z[PPFM_CHK_KINDS] = {};                        \
        cudaDeviceSynchronize();                                                                  \
        cudaMemcpyFromSymbol(h, g_chk, sizeof(h));                                                \
        cudaMemcpyToSymbol(g_chk, z, sizeof(z));                                                  \
        for (int k = 0; k < PPFM_CHK_KINDS; k++) out[k] += h[k];                                  \
    }
#define PPFM_CHK(kind, cond)                                                  \
    do {                                                                      \
        atomicAdd(&g_chk[PPFM_CHK_VISITS], 1ull);                             \
        if (!(cond)) atomicAdd(&g_chk[kind], 1ull);                           \
    } while (0)
#else
#define PPFM_CHK_STORAGE
#define PPFM_CHK(kind, cond) \
    do {                     \
    } while (0)
#endif
void ff_checks_read(unsigned long long *out);
void relax_checks_read(unsigned long long *out);
void df_checks_read(unsigned long long *out);

#define PPFM_CUDA(call)                                  \
    do {                                                 \
        cudaError_t _e = (call);                         \
        if (_e != cudaSuccess) {                         \
            ::ppfm::set_cuda_error(_e, #call);           \
            return (_e == cudaErrorMemoryAllocation) ? PPFM_ENOMEM : PPFM_ECUDA; \
        }                                                \
    } while (0)

#define PPFM_LAUNCH_CHECK()                              \
    do {                                                 \
        cudaError_t _e = cudaGetLastError();             \
        if (_e != cudaSuccess) {                         \
            ::ppfm::set_cuda_error(_e, "kernel launch"); \
            return PPFM_ECUDA;                           \
        }                                                \
        ::ppfm::count_launch();                          \
    } while (0)

// t = Minv (r - origin): inverse of the matrix whose COLUMNS are the grid step vectors.  false if singular.
inline bool invert_steps(const double step[3][3], double Minv[9]) {
    double A[9];
    for (int r = 0; r < 3; r++)
        for (int c = 0; c < 3; c++) A[3 * r + c] = step[c][r];
    const double det = A[0] * (A[4] * A[8] - A[5] * A[7]) - A[1] * (A[3] * A[8] - A[5] * A[6]) +
                       A[2] * (A[3] * A[7] - A[4] * A[6]);
    if (!(std::fabs(det) > 0.0) || !std::isfinite(det)) return false;
    const double id = 1.0 / det;
    Minv[0] = (A[4] * A[8] - A[5] * A[7]) * id;
    Minv[1] = (A[2] * A[7] - A[1] * A[8]) * id;
    Minv[2] = (A[1] * A[5] - A[2] * A[4]) * id;
    Minv[3] = (A[5] * A[6] - A[3] * A[8]) * id;
    Minv[4] = (A[0] * A[8] - A[2] * A[6]) * id;
    Minv[5] = (A[2] * A[3] - A[0] * A[5]) * id;
    Minv[6] = (A[3] * A[7] - A[4] * A[6]) * id;
    Minv[7] = (A[1] * A[6] - A[0] * A[7]) * id;
    Minv[8] = (A[0] * A[4] - A[1] * A[3]) * id;
    for (int i = 0; i < 9; i++)
        if (!std::isfinite(Minv[i])) return false;
    return true;
}

inline bool grid_ok(const ppfm_grid *g) {
    if (!g) return false;
    for (int a = 0; a < 3; a++) {
        if (g->n[a] < 1) return false;
        if (!std::isfinite(g->origin[a])) return false;
    }
    if ((long long)g->n[0] * g->n[1] > 0x7fffffffLL) return false;
    double Minv[9];
    return invert_steps(g->step, Minv);
}

inline long long grid_points(const ppfm_grid *g) { return (long long)g->n[0] * g->n[1] * g->n[2]; }

}  // namespace ppfm
