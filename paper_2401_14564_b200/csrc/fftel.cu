// fftel.cu — grid electrostatics of an extended tip charge density (Eq.7):
//     E_el(R) = integral rho_PP(r) V_S(r + R) dr,      F_el(R) = -grad_R E_el = integral grad rho_PP(r) V_S(r + R) dr,
// evaluated with the convolution theorem ("a product in the Fourier space, with an additional complex
// conjugation in the cross-correlation case") on the periodic grid.  Reading S21: the integral is the
// cyclic sum over grid nodes times dV = |det(step)|; rho_PP is a Gaussian multipole (monopole q_s, dipole p_z,
// quadrupole Q_zz) sampled with its analytic gradient at the nodes, minimum image by index.
//
// Path: fill_kernel (V -> FP64, rho and grad rho in FP64) -> cuFFT D2Z, batch 5 -> spectral_kernel
// (conj(rho^_c) V^ dV / N, c = 0..3) -> cuFFT Z2D, batch 4 -> pack_kernel (float4 Fx, Fy, Fz, E).  The FFT itself is
// the library primitive (cuFFT, FP64: V_S spans several orders of magnitude between the atoms and the scan region,
// and B200 runs FP64 at half the FP32 rate, so there is no reason to pay FP32's 1e-6 of max|V| everywhere).
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
fft_fill_kernel(const __grid_constant__ FftJob job, const float *__restrict__ V, double *__restrict__ real5) {
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
    const double v = (double)V[m];
    real5[m] = (job.vpow == 0.0) ? v : pow(fmax(v, 0.0), job.vpow);
    real5[job.N + m] = Pg;
    real5[2 * job.N + m] = dPx * g - Pg * r[0] * is2;
    real5[3 * job.N + m] = dPy * g - Pg * r[1] * is2;
    real5[4 * job.N + m] = dPz * g - Pg * r[2] * is2;
}

// in place on the four tip-field spectra: X_c <- conj(X_c) * V^ * scale
__global__ void __launch_bounds__(256)
fft_spectral_kernel(long long Nc, double scale, const double2 *__restrict__ Vh, double2 *__restrict__ X4) {
    const long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= Nc) return;
    const double2 v = Vh[m];
#pragma unroll
    for (int c = 0; c < 4; c++) {
        const double2 x = X4[c * Nc + m];
        X4[c * Nc + m] = make_double2((x.x * v.x + x.y * v.y) * scale, (x.x * v.y - x.y * v.x) * scale);
    }
}

__global__ void __launch_bounds__(256)
fft_pack_kernel(long long N, const double *__restrict__ real4, float4 *__restrict__ ff) {
    const long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= N) return;
    ff[m] = make_float4((float)real4[N + m], (float)real4[2 * N + m], (float)real4[3 * N + m], (float)real4[m]);
}

// ---- cuFFT plans, cached per (device, nx, ny, nz); destroyed by ppfm_release_scratch() ------------------------------
struct PlanEntry {
    int dev, nx, ny, nz;
    cufftHandle fwd, inv;
};
static std::mutex g_plan_mu;
static std::vector<PlanEntry> g_plans;

static cufftResult get_plans(int nx, int ny, int nz, cufftHandle *fwd, cufftHandle *inv) {
    int dev = 0;
    cudaGetDevice(&dev);
    std::lock_guard<std::mutex> lk(g_plan_mu);
    for (const PlanEntry &p : g_plans)
        if (p.dev == dev && p.nx == nx && p.ny == ny && p.nz == nz) { *fwd = p.fwd; *inv = p.inv; return CUFFT_SUCCESS; }
    PlanEntry e = {dev, nx, ny, nz, 0, 0};
    int dims[3] = {nz, ny, nx};
    const long long N = (long long)nx * ny * nz, Nc = (long long)nz * ny * (nx / 2 + 1);
    if (N > 0x7fffffffLL) return CUFFT_INVALID_SIZE;
    cufftResult r = cufftPlanMany(&e.fwd, 3, dims, nullptr, 1, (int)N, nullptr, 1, (int)Nc, CUFFT_D2Z, 5);
    if (r != CUFFT_SUCCESS) return r;
    r = cufftPlanMany(&e.inv, 3, dims, nullptr, 1, (int)Nc, nullptr, 1, (int)N, CUFFT_Z2D, 4);
    if (r != CUFFT_SUCCESS) { cufftDestroy(e.fwd); return r; }
    g_plans.push_back(e);
    *fwd = e.fwd; *inv = e.inv;
    return CUFFT_SUCCESS;
}

void release_fft_plans() {
    std::lock_guard<std::mutex> lk(g_plan_mu);
    for (const PlanEntry &p : g_plans) { cufftDestroy(p.fwd); cufftDestroy(p.inv); }
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
    cufftHandle fwd, inv;
    cufftResult fr = get_plans(job.nx, job.ny, job.nz, &fwd, &inv);
    if (fr != CUFFT_SUCCESS) { set_cuda_error(cudaErrorUnknown, "cufftPlanMany"); return fr == CUFFT_ALLOC_FAILED ? PPFM_ENOMEM : PPFM_ECUDA; }
    double *d_real = nullptr;
    double2 *d_cplx = nullptr;
    cudaError_t e = scratch_alloc((void **)&d_real, (size_t)5 * job.N * sizeof(double), st);
    if (e != cudaSuccess) { set_cuda_error(e, "scratch_alloc"); return PPFM_ENOMEM; }
    e = scratch_alloc((void **)&d_cplx, (size_t)5 * job.Nc * sizeof(double2), st);
    if (e != cudaSuccess) { set_cuda_error(e, "scratch_alloc"); cudaFreeAsync(d_real, st); return PPFM_ENOMEM; }
    int rc = PPFM_OK;
    const unsigned gN = (unsigned)((job.N + 255) / 256), gC = (unsigned)((job.Nc + 255) / 256);
    {
        KernelTimer kt(PPFM_K_FFT_EL, st);
        fft_fill_kernel<<<gN, 256, 0, st>>>(job, d_V, d_real);
        if (cufftSetStream(fwd, st) != CUFFT_SUCCESS || cufftExecD2Z(fwd, d_real, (cufftDoubleComplex *)d_cplx) != CUFFT_SUCCESS)
            rc = PPFM_ECUDA;
        if (rc == PPFM_OK) {
            fft_spectral_kernel<<<gC, 256, 0, st>>>(job.Nc, job.scale, d_cplx, d_cplx + job.Nc);
            if (cufftSetStream(inv, st) != CUFFT_SUCCESS ||
                cufftExecZ2D(inv, (cufftDoubleComplex *)(d_cplx + job.Nc), d_real) != CUFFT_SUCCESS)
                rc = PPFM_ECUDA;
        }
        if (rc == PPFM_OK) fft_pack_kernel<<<gN, 256, 0, st>>>(job.N, d_real, reinterpret_cast<float4 *>(d_ff));
    }
    e = cudaGetLastError();
    if (rc != PPFM_OK) set_cuda_error(cudaErrorUnknown, "cuFFT exec");
    else if (e != cudaSuccess) { set_cuda_error(e, "fft kernels"); rc = PPFM_ECUDA; }
    else count_launch(3);
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
