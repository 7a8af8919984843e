// df.cu — Fz -> frequency shift: Giessibl's formula, Eq.3,
//   df = -(f0 / 2k) (8 / (pi A^2)) int_{-A/2}^{A/2} q Fz(z + q) / sqrt(A^2/4 - q^2) dq,
// integrated exactly for the piecewise-linear interpolant of the n + 1 = A/dz + 1 samples in each window
// (reading S9).  The n + 1 weights are computed in FP64 on the host and passed by value; the kernel is
// a streaming weighted sum down each pixel column (HBM-bound: every Fz sample is read once).
#include "common.cuh"

#include <algorithm>

namespace ppfm {

constexpr int DF_MAX_N = PPFM_DF_MAX_N;

#define PPFM_CHK_READER df_checks_read
PPFM_CHK_STORAGE
#undef PPFM_CHK_READER
#ifndef PPFM_CHECKS
void df_checks_read(unsigned long long *) {}
#endif

struct DfWeights {
    float w[DF_MAX_N + 1];   // already multiplied by -(f0 / 2 k0) * 16.02176634
};

// Host: exact moments of q / sqrt(a^2 - q^2) against the hat functions of the uniform nodes q_m = -a + m dz.
// With y(q) = sqrt(a^2 - q^2):  int q/y dq = -y,  int q^2/y dq = (a^2/2) asin(q/a) - (q/2) y.
static void df_weights_host(int n, double dz, double *W) {
    const double a = 0.5 * n * dz;
    for (int m = 0; m <= n; m++) W[m] = 0.0;
    double q_lo = -a, y_lo = 0.0, G_lo = -0.25 * M_PI * a * a;
    for (int j = 0; j < n; j++) {
        const double q_hi = (j == n - 1) ? a : -a + (j + 1) * dz;
        const double y_hi = (j == n - 1) ? 0.0 : std::sqrt(std::fmax(a * a - q_hi * q_hi, 0.0));
        const double G_hi = (j == n - 1) ? 0.25 * M_PI * a * a
                                         : 0.5 * a * a * std::asin(q_hi / a) - 0.5 * q_hi * y_hi;
        const double m1 = y_lo - y_hi;   // first moment over the interval
        const double m2 = G_hi - G_lo;   // second moment
        W[j] += (q_hi * m1 - m2) / dz;
        W[j + 1] += (m2 - q_lo * m1) / dz;
        q_lo = q_hi; y_lo = y_hi; G_lo = G_hi;
    }
    const double norm = 2.0 / (M_PI * a * a);   // 8 / (pi A^2)
    for (int m = 0; m <= n; m++) W[m] *= norm;
}

// FZ4: Fz is the .w lane of the float4 (x, y, z, Fz) stack; otherwise a plain float stack (ppfm_scan_host keeps one
// on the device when the float4 stack itself is written straight to mapped host memory).
//
// Column kernel (n + 1 <= DF_RING_MAX): one thread per pixel column and chunk of output planes marches down z with the
// n + 1 samples of the current window in a register ring (slot indices are compile-time constants: the march is
// unrolled NW = n + 1 deep), so every sample is loaded once per chunk instead of n + 1 times and a warp's loads are
// 32 consecutive pixels of one plane.  The sum runs in the same order as the gather kernel below (m = 0 .. n).
constexpr int DF_RING_MAX = 33;
constexpr int DF_COL_THREADS = 128;

template <int NW, bool FZ4>
__global__ void __launch_bounds__(DF_COL_THREADS)
df_column_kernel(const float *__restrict__ fz, long long npix, int nz, int kc, const __grid_constant__ DfWeights W,
                 float *__restrict__ df) {
    constexpr int n = NW - 1;
    constexpr int S = FZ4 ? 4 : 1;
    const long long col = (long long)blockIdx.x * DF_COL_THREADS + threadIdx.x;
    if (col >= npix) return;
    const int nout = nz - n;
    const int k0 = (int)blockIdx.y * kc;
    const int cnt = min(kc, nout - k0);                       // output planes of this chunk
    const long long zs = npix * S;
    const float *src = fz + (((long long)blockIdx.z * nz + k0) * npix + col) * S + (FZ4 ? 3 : 0);
    float *dst = df + ((long long)blockIdx.z * nout + k0) * npix + col;
    float ring[NW];                                           // sample k0 + j lives in slot j % NW
#pragma unroll
    for (int j = 0; j < n; j++) ring[j] = __ldg(src + (long long)j * zs);
    // Each block of NW output planes first loads its NW new samples, unpredicated and back to back (past the chunk's
    // end the index is clamped to the stack's last plane and the value is not used), then forms the NW sums; only the
    // stores are guarded.
    const int jmax = nz - 1 - k0;
    for (int i0 = 0; i0 < cnt; i0 += NW) {
        float nxt[NW];
#pragma unroll
        for (int r = 0; r < NW; r++) {
            PPFM_CHK(PPFM_CHK_DF_LOAD, k0 + min(i0 + r + n, jmax) >= 0 && k0 + min(i0 + r + n, jmax) < nz);
            nxt[r] = __ldg(src + (long long)min(i0 + r + n, jmax) * zs);
        }
#pragma unroll
        for (int r = 0; r < NW; r++) {
            ring[(r + n) % NW] = nxt[r];
            float acc = 0.f;
#pragma unroll
            for (int m = 0; m <= n; m++) acc = fmaf(W.w[m], ring[(r + n - m) % NW], acc);
            PPFM_CHK(PPFM_CHK_DF_STORE, i0 + r >= cnt || k0 + i0 + r < nout);
            if (i0 + r < cnt) dst[(long long)(i0 + r) * npix] = acc;
        }
    }
}

// Gather kernel (any n <= DF_MAX_N): one thread per output sample, n + 1 strided loads each.
template <bool FZ4>
__global__ void __launch_bounds__(256)
df_kernel(const float *__restrict__ fz, long long npix, int nz, int n, int nsys, DfWeights W,
          float *__restrict__ df) {
    const long long nout_per = (long long)(nz - n) * npix;
    const long long total = nout_per * nsys;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long o = (long long)blockIdx.x * blockDim.x + threadIdx.x; o < total; o += stride) {
        const long long s = o / nout_per;
        const long long r = o - s * nout_per;
        const long long k = r / npix, p = r - k * npix;
        const float *src = fz + ((s * nz + k) * npix + p) * (FZ4 ? 4 : 1) + (FZ4 ? 3 : 0);
        float acc = 0.f;
        for (int m = 0; m <= n; m++) acc = fmaf(W.w[m], __ldg(&src[(long long)(n - m) * npix * (FZ4 ? 4 : 1)]), acc);
        df[o] = acc;
    }
}

template <int NW>
static void launch_df_column(int nw, bool fz4, dim3 grid, cudaStream_t st, const float *fz, long long npix, int nz,
                             int kc, const DfWeights &W, float *df) {
    if (nw == NW) {
        if (fz4) df_column_kernel<NW, true><<<grid, DF_COL_THREADS, 0, st>>>(fz, npix, nz, kc, W, df);
        else df_column_kernel<NW, false><<<grid, DF_COL_THREADS, 0, st>>>(fz, npix, nz, kc, W, df);
    } else if constexpr (NW < DF_RING_MAX) {
        launch_df_column<NW + 1>(nw, fz4, grid, st, fz, npix, nz, kc, W, df);
    }
}

static int df_impl(int nsys, const float *d_pos_fz, int npx, int npy, int nz, double dz, double A, double k0,
                   double f0, float *d_df, void *cuda_stream, bool fz4 = true) {
    if (nsys < 1 || !d_pos_fz || !d_df || npx < 1 || npy < 1 || nz < 1) return PPFM_EINVAL;
    if (!(dz > 0) || !(A > 0) || !(k0 > 0) || !std::isfinite(f0) || !std::isfinite(dz) || !std::isfinite(A))
        return PPFM_EINVAL;
    if ((uintptr_t)d_pos_fz & (fz4 ? 15 : 3)) return PPFM_EINVAL;
    const double nn = A / dz;
    const long long n = std::llround(nn);
    if (n < 1 || n > DF_MAX_N || std::fabs(nn - (double)n) > 1e-6 || nz <= n) return PPFM_EINVAL;
    double Wd[DF_MAX_N + 1];
    df_weights_host((int)n, dz, Wd);
    DfWeights W;
    const double pref = -(f0 / (2.0 * k0)) * kEVA2toNm;
    for (int m = 0; m <= DF_MAX_N; m++) W.w[m] = (m <= n) ? (float)(pref * Wd[m]) : 0.f;
    const long long npix = (long long)npx * npy;
    const long long total = (long long)(nz - n) * npix * nsys;
    const int nout = nz - (int)n;
    const long long col_blocks = (npix + DF_COL_THREADS - 1) / DF_COL_THREADS;
    {
        KernelTimer kt(PPFM_K_DF, (cudaStream_t)cuda_stream);
        if (n + 1 <= DF_RING_MAX && nsys <= 65535 && col_blocks <= 0x7fffffffLL) {
            // chunks of output planes per column: one chunk when the columns alone fill the GPU, otherwise enough chunks
            // for ~512 threads per SM, each at least one window long (a chunk re-reads n samples of its neighbour)
            const long long want = 148LL * 512;
            long long nchunks = (want + npix * nsys - 1) / (npix * nsys);
            const long long max_chunks = std::max<long long>(1, nout / std::max<long long>(n + 1, 8));
            nchunks = std::min(std::max<long long>(nchunks, 1), std::min<long long>(max_chunks, 65535));
            const int kc = (int)((nout + nchunks - 1) / nchunks);
            const dim3 grid((unsigned)col_blocks, (unsigned)((nout + kc - 1) / kc), (unsigned)nsys);
            launch_df_column<2>((int)n + 1, fz4, grid, (cudaStream_t)cuda_stream, d_pos_fz, npix, nz, kc, W, d_df);
        } else {
            long long blocks = (total + 255) / 256;
            if (blocks > 148LL * 32) blocks = 148LL * 32;
            if (fz4) df_kernel<true><<<(unsigned)blocks, 256, 0, (cudaStream_t)cuda_stream>>>(d_pos_fz, npix, nz, (int)n, nsys, W, d_df);
            else df_kernel<false><<<(unsigned)blocks, 256, 0, (cudaStream_t)cuda_stream>>>(d_pos_fz, npix, nz, (int)n, nsys, W, d_df);
        }
    }
    PPFM_LAUNCH_CHECK();
    return PPFM_OK;
}

int df_from_fz(int nsys, const float *d_fz, int npx, int npy, int nz, double dz, double A, double k0, double f0,
               float *d_df, void *cuda_stream) {
    return df_impl(nsys, d_fz, npx, npy, nz, dz, A, k0, f0, d_df, cuda_stream, false);
}

}  // namespace ppfm

using namespace ppfm;

extern "C" int ppfm_df(const float *d_pos_fz, int32_t npx, int32_t npy, int32_t nz, double dz, double A, double k0_Nm,
                       double f0_Hz, float *d_df, void *cuda_stream) {
    return df_impl(1, d_pos_fz, npx, npy, nz, dz, A, k0_Nm, f0_Hz, d_df, cuda_stream);
}

extern "C" int ppfm_df_batch(int32_t nsys, const float *d_pos_fz, int32_t npx, int32_t npy, int32_t nz, double dz,
                             double A, double k0_Nm, double f0_Hz, float *d_df, void *cuda_stream) {
    return df_impl(nsys, d_pos_fz, npx, npy, nz, dz, A, k0_Nm, f0_Hz, d_df, cuda_stream);
}

extern "C" int ppfm_df_weights(int32_t n, double dz, double *h_W) {
    if (n < 1 || n > DF_MAX_N || !(dz > 0) || !h_W) return PPFM_EINVAL;
    df_weights_host(n, dz, h_W);
    return PPFM_OK;
}
