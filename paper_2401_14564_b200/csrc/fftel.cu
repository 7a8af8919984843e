// fftel.cu — grid electrostatics of an extended tip charge density (Eq.7):
//     E_el(R) = integral rho_PP(r) V_S(r + R) dr,      F_el(R) = -grad_R E_el = integral grad rho_PP(r) V_S(r + R) dr,
// evaluated with the convolution theorem ("a product in the Fourier space, with an additional complex
// conjugation in the cross-correlation case") on the periodic grid.  Reading S21: the integral is the
// cyclic sum over grid nodes times dV = |det(step)|; rho_PP is a Gaussian multipole (monopole q_s, dipole p_z,
// quadrupole Q_zz) sampled with its analytic gradient at the nodes, minimum image by index.
//
// Path: fill_v_kernel (V -> FP64) -> cuFFT D2Z -> spectral_kernel (conj(rho^_c) V^ dV / N, c = 0..3) -> cuFFT Z2D,
// batch 4 -> pack_kernel (float4 Fx, Fy, Fz, E).  The four tip spectra rho^_c depend only on (grid, sigma, q_s, p_z,
// Q_zz): they are computed once (fill_tip_kernel + one batch-4 D2Z) and kept on the device in a small cache next to
// the plans, so that a run of calls on one grid ("amortized if a batch of simulations is run using the same grid",
// PAPER.md:298) costs 1 forward + 4 inverse transforms each instead of 5 + 4.  The FFT itself is the library
// primitive (cuFFT, FP64: V_S spans several orders of magnitude between the atoms and the scan region, and B200 runs
// FP64 at half the FP32 rate, so there is no reason to pay FP32's 1e-6 of max|V| everywhere).
//
// Streams and threads: plans are shared per (device, grid size) but own no work area (cufftSetAutoAllocation off);
// every call binds its own work area from the stream-ordered scratch pool, and the bind + enqueue sequence on the
// shared handles runs under one mutex, so calls on different streams or from different host threads neither share
// scratch nor race on a handle.  A cached tip spectrum carries the event of the stream that produced it; other
// streams wait on that event before reading it.
#include "common.cuh"

#include <cufft.h>

#include <mutex>
#include <vector>

namespace ppfm {

struct FftJob {
    int nx, ny, nz;
    long long N, Nc;           // real points, complex points nz*ny*(nx/2+1)
    double step[3][3];
    double sigma, q_s, p_z, Q_zz;
    double scale;              // dV / N
    double vpow;               // Eq.8 (vpow > 0): the input grid is clipped at 0 and raised to this power; 0 = Eq.7: as is
};

__global__ void __launch_bounds__(256)
fft_fill_v_kernel(long long N, double vpow, const float *__restrict__ V, double *__restrict__ real1) {
    const long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= N) return;
    const double v = (double)V[m];
    real1[m] = (vpow == 0.0) ? v : pow(fmax(v, 0.0), vpow);
}

// rho_PP and its analytic gradient at the nodes (minimum image by index): four real fields
__global__ void __launch_bounds__(256)
fft_fill_tip_kernel(const __grid_constant__ FftJob job, double *__restrict__ real4) {
    const long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= job.N) return;
    const int i = (int)(m % job.nx);
    const long long t = m / job.nx;
    const int j = (int)(t % job.ny), k = (int)(t / job.ny);
    const int iw = (2 * i >= job.nx) ? i - job.nx : i;
    const int jw = (2 * j >= job.ny) ? j - job.ny : j;
    const int kw = (2 * k >= job.nz) ? k - job.nz : k;
    double r[3];
#pragma unroll
    for (int c = 0; c < 3; c++) r[c] = iw * job.step[0][c] + jw * job.step[1][c] + kw * job.step[2][c];
    const double s2 = job.sigma * job.sigma, is2 = 1.0 / s2, is4 = is2 * is2;
    const double rr = r[0] * r[0] + r[1] * r[1] + r[2] * r[2];
    const double norm = rsqrt(2.0 * 3.14159265358979323846 * s2);
    const double g = norm * norm * norm * exp(-0.5 * rr * is2);
    const double q12 = job.Q_zz * (1.0 / 12.0);
    const double P = job.q_s + job.p_z * r[2] * is2 + q12 * (3.0 * r[2] * r[2] - rr) * is4;
    const double dPx = -2.0 * q12 * r[0] * is4, dPy = -2.0 * q12 * r[1] * is4;
    const double dPz = job.p_z * is2 + 4.0 * q12 * r[2] * is4;
    const double Pg = P * g;
    real4[m] = Pg;
    real4[job.N + m] = dPx * g - Pg * r[0] * is2;
    real4[2 * job.N + m] = dPy * g - Pg * r[1] * is2;
    real4[3 * job.N + m] = dPz * g - Pg * r[2] * is2;
}

// X_c = conj(T_c) * V^ * scale for the four cached tip spectra T_c
__global__ void __launch_bounds__(256)
fft_spectral_kernel(long long Nc, double scale, const double2 *__restrict__ Vh, const double2 *__restrict__ T4,
                    double2 *__restrict__ X4) {
    const long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= Nc) return;
    const double2 v = Vh[m];
#pragma unroll
    for (int c = 0; c < 4; c++) {
        const double2 x = T4[c * Nc + m];
        X4[c * Nc + m] = make_double2((x.x * v.x + x.y * v.y) * scale, (x.x * v.y - x.y * v.x) * scale);
    }
}

__global__ void __launch_bounds__(256)
fft_pack_kernel(long long N, const double *__restrict__ real4, float4 *__restrict__ ff) {
    const long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= N) return;
    ff[m] = make_float4((float)real4[N + m], (float)real4[2 * N + m], (float)real4[3 * N + m], (float)real4[m]);
}

// ---- cuFFT plans, cached per (device, nx, ny, nz), and tip spectra; destroyed by ppfm_release_scratch() -----------
struct PlanEntry {
    int dev, nx, ny, nz;
    cufftHandle fwd1, fwd4, inv4;
    size_t work_bytes;          // max over the three plans; bound per call
};
struct TipEntry {
    int dev, nx, ny, nz;
    double step[3][3], sigma, q_s, p_z, Q_zz;
    double2 *spec;              // 4 * Nc spectra (cudaMalloc; freed on eviction / release)
    cudaEvent_t ready;
    unsigned long long stamp;
};
constexpr int TIP_CACHE_ENTRIES = 2;
static std::mutex g_fft_mu;     // guards both caches and every bind + enqueue on the shared handles
static std::vector<PlanEntry> g_plans;
static std::vector<TipEntry> g_tips;
static unsigned long long g_tip_clock = 0;

static cufftResult make_plan(cufftHandle *h, int nx, int ny, int nz, cufftType type, int batch, size_t *work) {
    int dims[3] = {nz, ny, nx};
    const long long N = (long long)nx * ny * nz, Nc = (long long)nz * ny * (nx / 2 + 1);
    cufftResult r = cufftCreate(h);
    if (r != CUFFT_SUCCESS) return r;
    r = cufftSetAutoAllocation(*h, 0);
    const int idist = (type == CUFFT_D2Z) ? (int)N : (int)Nc, odist = (type == CUFFT_D2Z) ? (int)Nc : (int)N;
    if (r == CUFFT_SUCCESS) r = cufftMakePlanMany(*h, 3, dims, nullptr, 1, idist, nullptr, 1, odist, type, batch, work);
    if (r != CUFFT_SUCCESS) cufftDestroy(*h);
    return r;
}

// caller holds g_fft_mu
static cufftResult get_plans(int nx, int ny, int nz, PlanEntry *out) {
    int dev = 0;
    cudaGetDevice(&dev);
    for (const PlanEntry &p : g_plans)
        if (p.dev == dev && p.nx == nx && p.ny == ny && p.nz == nz) { *out = p; return CUFFT_SUCCESS; }
    if ((long long)nx * ny * nz > 0x7fffffffLL) return CUFFT_INVALID_SIZE;
    PlanEntry e = {dev, nx, ny, nz, 0, 0, 0, 0};
    size_t w1 = 0, w4 = 0, wi = 0;
    cufftResult r = make_plan(&e.fwd1, nx, ny, nz, CUFFT_D2Z, 1, &w1);
    if (r != CUFFT_SUCCESS) return r;
    r = make_plan(&e.fwd4, nx, ny, nz, CUFFT_D2Z, 4, &w4);
    if (r != CUFFT_SUCCESS) { cufftDestroy(e.fwd1); return r; }
    r = make_plan(&e.inv4, nx, ny, nz, CUFFT_Z2D, 4, &wi);
    if (r != CUFFT_SUCCESS) { cufftDestroy(e.fwd1); cufftDestroy(e.fwd4); return r; }
    e.work_bytes = w1 > w4 ? w1 : w4;
    if (wi > e.work_bytes) e.work_bytes = wi;
    g_plans.push_back(e);
    *out = e;
    return CUFFT_SUCCESS;
}

static bool tip_matches(const TipEntry &t, int dev, const FftJob &job) {
    if (t.dev != dev || t.nx != job.nx || t.ny != job.ny || t.nz != job.nz) return false;
    if (t.sigma != job.sigma || t.q_s != job.q_s || t.p_z != job.p_z || t.Q_zz != job.Q_zz) return false;
    return memcmp(t.step, job.step, sizeof(t.step)) == 0;
}

static void free_tip(TipEntry &t) {
    cudaFree(t.spec);           // synchronises the device: no stream still reads the spectra
    cudaEventDestroy(t.ready);
}

void release_fft_plans() {
    std::lock_guard<std::mutex> lk(g_fft_mu);
    for (TipEntry &t : g_tips) free_tip(t);
    g_tips.clear();
    for (const PlanEntry &p : g_plans) { cufftDestroy(p.fwd1); cufftDestroy(p.fwd4); cufftDestroy(p.inv4); }
    g_plans.clear();
}

}  // namespace ppfm

using namespace ppfm;

static int forcefield_fft_impl(const float *d_V, const ppfm_grid *grid, const ppfm_tip_density *tip, double vpow,
                               float *d_ff, void *cuda_stream) {
    if (!d_V || !grid || !tip || !d_ff) return PPFM_EINVAL;
    if (((uintptr_t)d_V & 3) || ((uintptr_t)d_ff & 15)) return PPFM_EINVAL;
    if (!grid_ok(grid)) return PPFM_EINVAL;
    if (!(tip->sigma > 0.0) || !std::isfinite(tip->sigma) || !std::isfinite(tip->q_s) || !std::isfinite(tip->p_z) ||
        !std::isfinite(tip->Q_zz))
        return PPFM_EINVAL;
    FftJob job;
    job.nx = grid->n[0]; job.ny = grid->n[1]; job.nz = grid->n[2];
    job.N = grid_points(grid);
    job.Nc = (long long)job.nz * job.ny * (job.nx / 2 + 1);
    if (job.N > 0x7fffffffLL) return PPFM_EINVAL;
    for (int a = 0; a < 3; a++)
        for (int c = 0; c < 3; c++) job.step[a][c] = grid->step[a][c];
    const double (*s)[3] = grid->step;
    const double det = s[0][0] * (s[1][1] * s[2][2] - s[1][2] * s[2][1]) - s[0][1] * (s[1][0] * s[2][2] - s[1][2] * s[2][0]) +
                       s[0][2] * (s[1][0] * s[2][1] - s[1][1] * s[2][0]);
    job.sigma = tip->sigma; job.q_s = tip->q_s; job.p_z = tip->p_z; job.Q_zz = tip->Q_zz;
    job.scale = std::fabs(det) / (double)job.N;
    job.vpow = vpow;

    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0;
    cudaGetDevice(&dev);
    const unsigned gN = (unsigned)((job.N + 255) / 256), gC = (unsigned)((job.Nc + 255) / 256);
    std::lock_guard<std::mutex> lk(g_fft_mu);      // held across bind + enqueue (all asynchronous) on the shared handles
    PlanEntry pl;
    cufftResult fr = get_plans(job.nx, job.ny, job.nz, &pl);
    if (fr != CUFFT_SUCCESS) { set_cuda_error(cudaErrorUnknown, "cufftMakePlanMany"); return fr == CUFFT_ALLOC_FAILED ? PPFM_ENOMEM : PPFM_ECUDA; }
    double *d_real = nullptr;       // 4 N doubles: V in the first N before the forward transform, the four fields after
    double2 *d_cplx = nullptr;      // V^ (Nc) | X_c (4 Nc)
    void *d_work = nullptr;
    cudaError_t e = scratch_alloc((void **)&d_real, (size_t)4 * job.N * sizeof(double), st);
    if (e == cudaSuccess) e = scratch_alloc((void **)&d_cplx, (size_t)5 * job.Nc * sizeof(double2), st);
    if (e == cudaSuccess) e = scratch_alloc(&d_work, pl.work_bytes, st);
    if (e != cudaSuccess) {
        set_cuda_error(e, "scratch_alloc");
        if (d_real) cudaFreeAsync(d_real, st);
        if (d_cplx) cudaFreeAsync(d_cplx, st);
        return PPFM_ENOMEM;
    }
    int rc = PPFM_OK;
    int own_launches = 0;
    auto bind = [&](cufftHandle h) {
        return cufftSetStream(h, st) == CUFFT_SUCCESS && cufftSetWorkArea(h, d_work) == CUFFT_SUCCESS;
    };
    {
        KernelTimer kt(PPFM_K_FFT_EL, st);
        // ---- tip spectra: cached, or computed now into a new cache entry
        TipEntry *te = nullptr;
        for (TipEntry &t : g_tips)
            if (tip_matches(t, dev, job)) te = &t;
        if (!te) {
            if ((int)g_tips.size() >= TIP_CACHE_ENTRIES) {           // evict the least recently used entry
                size_t old = 0;
                for (size_t i = 1; i < g_tips.size(); i++)
                    if (g_tips[i].stamp < g_tips[old].stamp) old = i;
                free_tip(g_tips[old]);
                g_tips.erase(g_tips.begin() + old);
            }
            TipEntry t;
            memset(&t, 0, sizeof(t));
            t.dev = dev; t.nx = job.nx; t.ny = job.ny; t.nz = job.nz;
            memcpy(t.step, job.step, sizeof(t.step));
            t.sigma = job.sigma; t.q_s = job.q_s; t.p_z = job.p_z; t.Q_zz = job.Q_zz;
            e = cudaMalloc((void **)&t.spec, (size_t)4 * job.Nc * sizeof(double2));
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&t.ready, cudaEventDisableTiming);
            if (e != cudaSuccess) {
                if (t.spec) cudaFree(t.spec);
                set_cuda_error(e, "tip spectrum cache");
                rc = (e == cudaErrorMemoryAllocation) ? PPFM_ENOMEM : PPFM_ECUDA;
            } else {
                fft_fill_tip_kernel<<<gN, 256, 0, st>>>(job, d_real);
                own_launches++;
                if (!bind(pl.fwd4) || cufftExecD2Z(pl.fwd4, d_real, (cufftDoubleComplex *)t.spec) != CUFFT_SUCCESS) {
                    rc = PPFM_ECUDA;
                    cudaStreamSynchronize(st);
                    cudaFree(t.spec);
                    cudaEventDestroy(t.ready);
                } else {
                    cudaEventRecord(t.ready, st);
                    g_tips.push_back(t);
                    te = &g_tips.back();
                }
            }
        } else {
            cudaStreamWaitEvent(st, te->ready, 0);                  // produced on another stream, perhaps
        }
        if (rc == PPFM_OK) {
            te->stamp = ++g_tip_clock;
            fft_fill_v_kernel<<<gN, 256, 0, st>>>(job.N, job.vpow, d_V, d_real);
            if (!bind(pl.fwd1) || cufftExecD2Z(pl.fwd1, d_real, (cufftDoubleComplex *)d_cplx) != CUFFT_SUCCESS)
                rc = PPFM_ECUDA;
        }
        if (rc == PPFM_OK) {
            fft_spectral_kernel<<<gC, 256, 0, st>>>(job.Nc, job.scale, d_cplx, te->spec, d_cplx + job.Nc);
            if (!bind(pl.inv4) || cufftExecZ2D(pl.inv4, (cufftDoubleComplex *)(d_cplx + job.Nc), d_real) != CUFFT_SUCCESS)
                rc = PPFM_ECUDA;
        }
        if (rc == PPFM_OK) {
            fft_pack_kernel<<<gN, 256, 0, st>>>(job.N, d_real, reinterpret_cast<float4 *>(d_ff));
            own_launches += 3;
        }
    }
    e = cudaGetLastError();
    if (rc == PPFM_ECUDA && e == cudaSuccess) set_cuda_error(cudaErrorUnknown, "cuFFT exec");
    else if (rc == PPFM_OK && e != cudaSuccess) { set_cuda_error(e, "fft kernels"); rc = PPFM_ECUDA; }
    if (rc == PPFM_OK) count_launch(own_launches);
    cudaFreeAsync(d_work, st);
    cudaFreeAsync(d_cplx, st);
    cudaFreeAsync(d_real, st);
    return rc;
}

extern "C" int ppfm_forcefield_fft(const float *d_V, const ppfm_grid *grid, const ppfm_tip_density *tip, float *d_ff,
                                   void *cuda_stream) {
    return forcefield_fft_impl(d_V, grid, tip, 0.0, d_ff, cuda_stream);
}

// Eq.8: E_Pauli(R) = A integral [rho_PP(r) rho_S(r + R)]^beta dr with rho_PP = q g_sigma.  A Gaussian
// to the power beta is a Gaussian, (q g_s)^beta = q^beta (2 pi s^2)^(3(1-beta)/2) beta^(-3/2) g_{s/sqrt(beta)}, so this
// is the Eq.7 pipeline on rho_S^beta with a monopole tip of that width and weight.
extern "C" int ppfm_forcefield_pauli(const float *d_rho_S, const ppfm_grid *grid, double sigma, double q_tip, double A,
                                     double beta, float *d_ff, void *cuda_stream) {
    if (!(sigma > 0.0) || !(q_tip > 0.0) || !(beta > 0.0) || !std::isfinite(sigma) || !std::isfinite(q_tip) ||
        !std::isfinite(beta) || !std::isfinite(A))
        return PPFM_EINVAL;
    ppfm_tip_density td;
    td.sigma = sigma / std::sqrt(beta);
    td.q_s = A * std::pow(q_tip, beta) * std::pow(2.0 * M_PI * sigma * sigma, 1.5 * (1.0 - beta)) * std::pow(beta, -1.5);
    td.p_z = 0.0;
    td.Q_zz = 0.0;
    return forcefield_fft_impl(d_rho_S, grid, &td, beta, d_ff, cuda_stream);
}
