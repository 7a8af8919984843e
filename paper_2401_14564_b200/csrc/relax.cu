// relax.cu — per-pixel FIRE relaxation scan: for every lateral tip position the tip
// anchor steps down in z and the probe particle is relaxed under F = F_T + F_S (Eq.1) with the tip
// springs of Eq.2 and F_S from tri-linear interpolation of the float4 grid, using
// FIRE (ref [7]; constants and loop order = DESIGN.md reading S6).  Read-out Fz_tip = -F_R,z
// (PAPER.md:62).
//
// Kernel design: one thread per pixel, the whole z stroke inside the kernel (state carried in registers); a warp
// covers an 8 x 4 pixel patch so that the 8-corner float4 gathers of neighbouring lanes fall into the same
// 128-byte lines (L1/L2 hits) and iteration counts within a warp stay similar; the FIRE loop is warp-converged by
// an __all_sync vote on (converged || max_iter), so the eight LDG.128 of an iteration issue warp-wide.
// FP32 with two precautions that keep |F| < 1e-6 eV/Å reachable:
//   * the state is the displacement u = d - d0 from the spring equilibrium, and the radial extension is
//     |d| - R0 = (|u|^2 + 2 d0.u)/(|d| + R0) (no cancellation);
//   * the fractional grid coordinate is (exact FP64 coordinate of r_TIP + d0, split int + frac once per z-step)
//     + Minv u in FP32.
#include "common.cuh"

namespace ppfm {

constexpr int RX_THREADS = 128;     // 4 warps = 2 x 2 patches of 8 x 4 pixels -> 16 x 8 pixels per CTA
constexpr int RX_TILE_X = 16, RX_TILE_Y = 8;

struct RelaxJob {
    long long ff_offset;     // float4 offset of this system's grid
    long long out_offset;    // pixel-step offset of this system's outputs
    int block_begin;
    int nbx;                 // CTAs along x
    int npx, npy, nzs;
    int n[3], periodic[3];
    double origin[3], Minv[9];
    double p0[3], dx[3], dy[3], dz;
    double d0[3];
    float Minvf[9];
    float d0f[3], R_rest, k_lat[2], k_rad;
};

struct FireParams {
    float dt0, dt_max, finc, fdec, alpha0, falpha, fconv2;
    int n_min, max_iter;
};

__device__ __forceinline__ float rsqrt_fast(float x) {
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float lerp(float a, float b, float t) { return fmaf(t, b - a, a); }

// cell index pair and fraction along one axis; `ib` = integer part of the base coordinate (already wrapped into
// [0, n) on periodic axes), `tf` = fractional base + FP32 offset.
__device__ __forceinline__ bool axis_cell(float tf, int ib, int n, int periodic, int &i0, int &i1, float &f) {
    bool clamped = false;
    if (periodic) {
        tf = fminf(fmaxf(tf, (float)(1 - n)), (float)(n - 1));   // never more than one cell-length away
        const float fl = floorf(tf);
        f = tf - fl;
        int i = ib + (int)fl;
        if (i >= n) i -= n;
        if (i < 0) i += n;
        i0 = i;
        i1 = (i + 1 == n) ? 0 : i + 1;
    } else {
        const float lo = (float)(-ib), hi = (float)(n - 1 - ib);
        clamped = (tf < lo) || (tf > hi);
        tf = fminf(fmaxf(tf, lo), hi);
        int i = ib + (int)floorf(tf);
        i = min(i, n - 2);
        i = max(i, 0);
        f = tf - (float)(i - ib);
        i0 = i;
        i1 = i + 1;
    }
    return clamped;
}

__global__ void __launch_bounds__(RX_THREADS)
relax_kernel(const RelaxJob *__restrict__ jobs, int njobs, FireParams fp, const float4 *__restrict__ ff,
             float4 *__restrict__ pos_fz, uint16_t *__restrict__ iters_out, ppfm_stats *__restrict__ stats) {
    __shared__ RelaxJob s_job;
    const int blk = blockIdx.x;
    int lo = 0, hi = njobs - 1;
    while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (jobs[mid].block_begin <= blk) lo = mid; else hi = mid - 1;
    }
    {
        const int *srcw = reinterpret_cast<const int *>(&jobs[lo]);
        int *dstw = reinterpret_cast<int *>(&s_job);
        for (int w = threadIdx.x; w < (int)(sizeof(RelaxJob) / sizeof(int)); w += RX_THREADS) dstw[w] = srcw[w];
    }
    __syncthreads();
    const RelaxJob &job = s_job;

    const int lb = blk - job.block_begin;
    const int by = lb / job.nbx, bx = lb - by * job.nbx;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int ix = bx * RX_TILE_X + (warp & 1) * 8 + (lane & 7);
    const int iy = by * RX_TILE_Y + (warp >> 1) * 4 + (lane >> 3);
    const bool valid = (ix < job.npx) && (iy < job.npy);
    const int ixc = min(ix, job.npx - 1), iyc = min(iy, job.npy - 1);

    const float4 *__restrict__ g = ff + job.ff_offset;
    const int nx = job.n[0], ny = job.n[1], nz = job.n[2];
    const int perx = job.periodic[0], pery = job.periodic[1], perz = job.periodic[2];
    const float m00 = job.Minvf[0], m01 = job.Minvf[1], m02 = job.Minvf[2];
    const float m10 = job.Minvf[3], m11 = job.Minvf[4], m12 = job.Minvf[5];
    const float m20 = job.Minvf[6], m21 = job.Minvf[7], m22 = job.Minvf[8];
    const float d0x = job.d0f[0], d0y = job.d0f[1], d0z = job.d0f[2];
    const float R_rest = job.R_rest, k_rad = job.k_rad, kx = job.k_lat[0], ky = job.k_lat[1];

    // r_TIP + d0 - origin at iz = 0, FP64
    double rb[3];
#pragma unroll
    for (int c = 0; c < 3; c++)
        rb[c] = job.p0[c] + ixc * job.dx[c] + iyc * job.dy[c] + job.d0[c] - job.origin[c];

    float ux = 0.f, uy = 0.f, uz = 0.f;
    unsigned long long my_iters = 0;
    unsigned int my_notconv = 0, my_clamped = 0, my_max = 0;

    for (int iz = 0; iz < job.nzs; iz++) {
        // a4: exact fractional grid coordinate of the spring equilibrium point, split int + frac
        const double rz = rb[2] - iz * job.dz;
        int ib[3];
        float fb[3];
#pragma unroll
        for (int a = 0; a < 3; a++) {
            const double t = job.Minv[3 * a] * rb[0] + job.Minv[3 * a + 1] * rb[1] + job.Minv[3 * a + 2] * rz;
            const double fl = floor(t);
            fb[a] = (float)(t - fl);
            const int n = job.n[a];
            if (job.periodic[a]) {
                long long m = (long long)fl % n;
                if (m < 0) m += n;
                ib[a] = (int)m;
            } else {
                ib[a] = (int)fmin(fmax(fl, -1.0e9), 1.0e9);
            }
        }

        float vx = 0.f, vy = 0.f, vz = 0.f, dt = fp.dt0, alpha = fp.alpha0;
        int npos = 0, moves = 0;
        bool conv = !valid, clamped = false;
        float ext = 0.f, invL = 0.f, dzc = d0z;

        while (true) {
            // ---- F_S: tri-linear interpolation (8 x LDG.128)
            const float tx = fb[0] + fmaf(m00, ux, fmaf(m01, uy, m02 * uz));
            const float ty = fb[1] + fmaf(m10, ux, fmaf(m11, uy, m12 * uz));
            const float tz = fb[2] + fmaf(m20, ux, fmaf(m21, uy, m22 * uz));
            int i0, i1, j0, j1, k0, k1;
            float fx, fy, fz;
            clamped = axis_cell(tx, ib[0], nx, perx, i0, i1, fx);
            clamped |= axis_cell(ty, ib[1], ny, pery, j0, j1, fy);
            clamped |= axis_cell(tz, ib[2], nz, perz, k0, k1, fz);
            const int r00 = (k0 * ny + j0) * nx, r01 = (k0 * ny + j1) * nx;
            const int r10 = (k1 * ny + j0) * nx, r11 = (k1 * ny + j1) * nx;
            const float4 c000 = __ldg(g + r00 + i0), c001 = __ldg(g + r00 + i1);
            const float4 c010 = __ldg(g + r01 + i0), c011 = __ldg(g + r01 + i1);
            const float4 c100 = __ldg(g + r10 + i0), c101 = __ldg(g + r10 + i1);
            const float4 c110 = __ldg(g + r11 + i0), c111 = __ldg(g + r11 + i1);
            float Fx = lerp(lerp(lerp(c000.x, c001.x, fx), lerp(c010.x, c011.x, fx), fy),
                            lerp(lerp(c100.x, c101.x, fx), lerp(c110.x, c111.x, fx), fy), fz);
            float Fy = lerp(lerp(lerp(c000.y, c001.y, fx), lerp(c010.y, c011.y, fx), fy),
                            lerp(lerp(c100.y, c101.y, fx), lerp(c110.y, c111.y, fx), fy), fz);
            float Fz = lerp(lerp(lerp(c000.z, c001.z, fx), lerp(c010.z, c011.z, fx), fy),
                            lerp(lerp(c100.z, c101.z, fx), lerp(c110.z, c111.z, fx), fy), fz);
            // ---- F_T: radial + lateral springs (Eq.2), d = d0 + u
            const float dxc = d0x + ux, dyc = d0y + uy;
            dzc = d0z + uz;
            const float L2 = fmaf(dxc, dxc, fmaf(dyc, dyc, dzc * dzc));
            invL = rsqrt_fast(L2);
            const float L = L2 * invL;
            const float num = fmaf(ux, ux, fmaf(uy, uy, uz * uz)) + 2.0f * fmaf(d0x, ux, fmaf(d0y, uy, d0z * uz));
            ext = __fdividef(num, L + R_rest);           // |d| - R0
            const float fr = -k_rad * ext * invL;
            Fx = fmaf(fr, dxc, Fx) - kx * ux;
            Fy = fmaf(fr, dyc, Fy) - ky * uy;
            Fz = fmaf(fr, dzc, Fz);
            const float F2 = fmaf(Fx, Fx, fmaf(Fy, Fy, Fz * Fz));
            if (!conv) conv = F2 < fp.fconv2;            // tested before every move (reading S7)
            const bool done = conv || (moves >= fp.max_iter);
            if (__all_sync(0xffffffffu, done)) break;
            if (!done) {
                // ---- FIRE (reading S6)
                const float Pw = fmaf(Fx, vx, fmaf(Fy, vy, Fz * vz));
                if (Pw >= 0.0f) {
                    const float v2 = fmaf(vx, vx, fmaf(vy, vy, vz * vz));
                    const float c = alpha * sqrtf(v2) * rsqrt_fast(F2);
                    const float om = 1.0f - alpha;
                    vx = fmaf(om, vx, c * Fx); vy = fmaf(om, vy, c * Fy); vz = fmaf(om, vz, c * Fz);
                    if (npos > fp.n_min) {
                        dt = fminf(dt * fp.finc, fp.dt_max);
                        alpha *= fp.falpha;
                    }
                    npos++;
                } else {
                    vx = vy = vz = 0.f;
                    dt *= fp.fdec;
                    alpha = fp.alpha0;
                    npos = 0;
                }
                vx = fmaf(Fx, dt, vx); vy = fmaf(Fy, dt, vy); vz = fmaf(Fz, dt, vz);
                ux = fmaf(vx, dt, ux); uy = fmaf(vy, dt, uy); uz = fmaf(vz, dt, uz);
                moves++;
            }
        }

        if (valid) {
            const size_t o = (size_t)job.out_offset + ((size_t)iz * job.npy + iy) * job.npx + ix;
            float4 outv;
            outv.x = (float)(rb[0] + job.origin[0] + (double)ux);
            outv.y = (float)(rb[1] + job.origin[1] + (double)uy);
            outv.z = (float)(rz + job.origin[2] + (double)uz);
            outv.w = k_rad * ext * invL * dzc;            // Fz_tip = -F_R,z
            pos_fz[o] = outv;
            if (iters_out) iters_out[o] = conv ? (uint16_t)min(moves, 0xFFFE) : (uint16_t)0xFFFF;
            my_iters += (unsigned)moves;
            my_notconv += conv ? 0u : 1u;
            my_clamped += clamped ? 1u : 0u;
            my_max = max(my_max, (unsigned)moves);
        }
    }

    if (stats) {
#pragma unroll
        for (int s = 16; s > 0; s >>= 1) {
            my_iters += __shfl_xor_sync(0xffffffffu, my_iters, s);
            my_notconv += __shfl_xor_sync(0xffffffffu, my_notconv, s);
            my_clamped += __shfl_xor_sync(0xffffffffu, my_clamped, s);
            my_max = max(my_max, __shfl_xor_sync(0xffffffffu, my_max, s));
        }
        if (lane == 0) {
            atomicAdd(reinterpret_cast<unsigned long long *>(&stats->total_iters), my_iters);
            if (my_notconv) atomicAdd(reinterpret_cast<unsigned long long *>(&stats->n_not_converged), (unsigned long long)my_notconv);
            if (my_clamped) atomicAdd(reinterpret_cast<unsigned long long *>(&stats->n_clamped), (unsigned long long)my_clamped);
            atomicMax(&stats->max_iters, my_max);
        }
    }
}

static int relax_impl(int nsys, const float *d_ff, const ppfm_grid *grids, const ppfm_tip *tips,
                      const ppfm_fire *fire, const ppfm_scan *scans, float *d_pos_fz, uint16_t *d_iters,
                      ppfm_stats *d_stats, void *cuda_stream) {
    if (nsys < 1 || !d_ff || !grids || !tips || !fire || !scans || !d_pos_fz) return PPFM_EINVAL;
    if (((uintptr_t)d_ff & 15) || ((uintptr_t)d_pos_fz & 15) || ((uintptr_t)d_iters & 1) || ((uintptr_t)d_stats & 7))
        return PPFM_EINVAL;
    if (!(fire->dt > 0) || !(fire->dt_max > 0) || !(fire->finc >= 1.0) || !(fire->fdec > 0 && fire->fdec < 1.0) ||
        !(fire->alpha0 >= 0 && fire->alpha0 <= 1.0) || !(fire->falpha > 0 && fire->falpha <= 1.0) ||
        fire->n_min < 0 || fire->max_iter < 0 || fire->max_iter > 0xFFFE || !(fire->f_conv > 0))
        return PPFM_EINVAL;
    RelaxJob *hj = (RelaxJob *)calloc((size_t)nsys, sizeof(RelaxJob));
    if (!hj) return PPFM_ENOMEM;
    long long blocks = 0, ff_off = 0, out_off = 0;
    for (int m = 0; m < nsys; m++) {
        const ppfm_grid &g = grids[m];
        const ppfm_scan &s = scans[m];
        const ppfm_tip &t = tips[m];
        RelaxJob &j = hj[m];
        bool ok = grid_ok(&g) && g.n[0] >= 2 && g.n[1] >= 2 && g.n[2] >= 2 && s.npx >= 1 && s.npy >= 1 && s.nz >= 1 &&
                  std::isfinite(s.dz) && invert_steps(g.step, j.Minv) && grid_points(&g) <= 0x7fffffffLL;
        const double R0 = std::sqrt(t.d0[0] * t.d0[0] + t.d0[1] * t.d0[1] + t.d0[2] * t.d0[2]);
        ok = ok && (R0 > 0) && std::isfinite(R0) && (t.k_rad >= 0) && (t.k_lat[0] >= 0) && (t.k_lat[1] >= 0) &&
             std::isfinite(t.k_rad) && std::isfinite(t.k_lat[0]) && std::isfinite(t.k_lat[1]);
        if (!ok) { free(hj); return PPFM_EINVAL; }
        j.ff_offset = ff_off;
        j.out_offset = out_off;
        j.block_begin = (int)blocks;
        j.nbx = (s.npx + RX_TILE_X - 1) / RX_TILE_X;
        j.npx = s.npx; j.npy = s.npy; j.nzs = s.nz;
        for (int a = 0; a < 3; a++) {
            j.n[a] = g.n[a];
            j.periodic[a] = g.periodic[a] ? 1 : 0;
            j.origin[a] = g.origin[a];
            j.p0[a] = s.p0[a]; j.dx[a] = s.dx[a]; j.dy[a] = s.dy[a];
            j.d0[a] = t.d0[a];
            j.d0f[a] = (float)t.d0[a];
        }
        for (int i = 0; i < 9; i++) j.Minvf[i] = (float)j.Minv[i];
        j.dz = s.dz;
        j.R_rest = (float)R0;
        j.k_lat[0] = (float)t.k_lat[0]; j.k_lat[1] = (float)t.k_lat[1];
        j.k_rad = (float)t.k_rad;
        blocks += (long long)j.nbx * ((s.npy + RX_TILE_Y - 1) / RX_TILE_Y);
        ff_off += grid_points(&g);
        out_off += (long long)s.npx * s.npy * s.nz;
        if (blocks > 0x7fffffffLL) { free(hj); return PPFM_EINVAL; }
    }
    FireParams fp;
    fp.dt0 = (float)fire->dt; fp.dt_max = (float)fire->dt_max; fp.finc = (float)fire->finc;
    fp.fdec = (float)fire->fdec; fp.alpha0 = (float)fire->alpha0; fp.falpha = (float)fire->falpha;
    fp.fconv2 = (float)(fire->f_conv * fire->f_conv);
    fp.n_min = fire->n_min; fp.max_iter = fire->max_iter;

    cudaStream_t st = (cudaStream_t)cuda_stream;
    RelaxJob *dj = nullptr;
    cudaError_t e = cudaMallocAsync((void **)&dj, (size_t)nsys * sizeof(RelaxJob), st);
    if (e != cudaSuccess) { free(hj); set_cuda_error(e, "cudaMallocAsync"); return PPFM_ENOMEM; }
    e = cudaMemcpyAsync(dj, hj, (size_t)nsys * sizeof(RelaxJob), cudaMemcpyHostToDevice, st);
    free(hj);
    if (e != cudaSuccess) { set_cuda_error(e, "job upload"); cudaFreeAsync(dj, st); return PPFM_ECUDA; }
    relax_kernel<<<(unsigned)blocks, RX_THREADS, 0, st>>>(dj, nsys, fp, reinterpret_cast<const float4 *>(d_ff),
                                                         reinterpret_cast<float4 *>(d_pos_fz), d_iters, d_stats);
    e = cudaGetLastError();
    if (e != cudaSuccess) { set_cuda_error(e, "relax_kernel"); cudaFreeAsync(dj, st); return PPFM_ECUDA; }
    count_launch();
    PPFM_CUDA(cudaFreeAsync(dj, st));
    return PPFM_OK;
}

}  // namespace ppfm

using namespace ppfm;

extern "C" int ppfm_relax_scan(const float *d_ff, const ppfm_grid *grid, const ppfm_tip *tip, const ppfm_fire *fire,
                               const ppfm_scan *scan, float *d_pos_fz, uint16_t *d_iters, ppfm_stats *d_stats,
                               void *cuda_stream) {
    return relax_impl(1, d_ff, grid, tip, fire, scan, d_pos_fz, d_iters, d_stats, cuda_stream);
}

extern "C" int ppfm_relax_scan_batch(int32_t nsys, const float *d_ff, const ppfm_grid *grids, const ppfm_tip *tips,
                                     const ppfm_fire *fire, const ppfm_scan *scans, float *d_pos_fz,
                                     uint16_t *d_iters, ppfm_stats *d_stats, void *cuda_stream) {
    return relax_impl(nsys, d_ff, grids, tips, fire, scans, d_pos_fz, d_iters, d_stats, cuda_stream);
}
