// relax.cu — per-pixel FIRE relaxation scan: for every lateral tip position the tip
// anchor steps down in z and the probe particle is relaxed under F = F_T + F_S (Eq.1) with the tip
// springs of Eq.2 and F_S from tri-linear interpolation of the float4 grid, using
// FIRE (ref [7]; constants and loop order = DESIGN.md reading S6).  Read-out Fz_tip = -F_R,z
// (PAPER.md:62).
//
// Kernel design.  One thread per pixel, the whole z stroke inside the kernel (state in registers);
// a warp covers an 8 x 4 pixel patch so that the gathers of neighbouring lanes fall into the same 128-byte lines.
// A FIRE iteration is a strictly dependent chain (position -> force -> step), so with few pixels the kernel runs at
// the latency of that chain and with many pixels at the speed of instruction issue; both want the fewest
// instructions per iteration:
//   * the lane keeps its current grid cell in registers (per force component the 8 coefficients of the tri-linear
//     polynomial, evaluated by Horner: 7 FFMA, depth 3) and the per-axis offset that turns the position into the
//     in-cell fraction with one FFMA; the probe particle leaves
//     its cell in 2-3 % of iterations, and only then the warp (all lanes, one warp-uniform block entered through
//     __any_sync) re-locates and re-gathers: cell index and fraction by the magic-number trick (t - 0.5 + 1.5*2^23
//     rounds to floor(t) in the low mantissa bits; clamps are two FMNMX in that domain), eight LDG.128 issued back
//     to back;
//   * the interpolation is computed speculatively from the cached cell ahead of that branch; the spring chain's
//     MUFU.SQRT has to issue well ahead of it too, which the stated register budget secures (see RX_MIN_CTAS);
//   * FIRE is branch-free: everything that depends only on the old velocity is computed off the critical path; after
//     F arrives the chain is F.F -> rsqrt -> one select -> two FMA per component;
//   * the convergence vote (__all_sync) is taken every second iteration: finished lanes do not move.
// The same function, templated on the interpolant, serves the tri-cubic energy-only variant: 64
// energies of the 4 x 4 x 4 stencil in registers instead of the 8 corner forces.
// FP32 with two precautions that keep |F| < 1e-6 eV/Å reachable:
//   * the state is the displacement u = d - d0 from the spring equilibrium, and the radial extension is
//     |d| - R0 = (|u|^2 + 2 d0.u)/(|d| + R0) (no cancellation);
//   * the fractional grid coordinate is (exact FP64 coordinate of r_TIP + d0, split int + frac once per z-step)
//     + Minv u in FP32.
#include "common.cuh"

namespace ppfm {

constexpr int RX_THREADS = 128;     // 4 warps = 2 x 2 patches of 8 x 4 pixels -> 16 x 8 pixels per CTA
constexpr int RX_TILE_X = 16, RX_TILE_Y = 8;
// Register budget of the tri-linear kernels: 4 CTAs per SM = up to 128 registers.  Left to itself ptxas cuts some
// instantiations to 96 registers (5 CTAs) and then sinks the spring chain's MUFU.SQRT next to its MUFU.RCP behind the
// stale-cell vote: a lone warp then stalls ~17 cycles per iteration (config 1: 0.74 -> 0.85 ms; with the stiffness map
// folded in, 0.97 ms).  With the budget stated every instantiation gets the schedule with the square root issued
// ~15 instructions ahead of the vote (checked in the SASS, profiles/r02_sass_summary.txt); the fifth CTA was worth
// <= 4 % on the large scans and the larger budget is worth that much there too.
constexpr int RX_MIN_CTAS = 4;
constexpr long long RX_SPARSE_MAX_WARPS = 148LL * 2;   // launches up to this many (dense) warps use 16 pixels per warp
constexpr float RX_MAGIC = 12582912.0f;      // 1.5 * 2^23: floats in [2^23, 2^24) are the integers
constexpr int RX_MAGIC_BITS = 0x4B400000;
constexpr int RX_MAX_N = 1 << 21;            // per-axis grid size limit of the magic-number cell index

struct RelaxJob {
    long long ff_offset;     // float4 offset of this system's grid
    long long out_offset;    // pixel-step offset of this system's outputs
    int block_begin;
    int nbx;                 // CTAs along x
    int sparse;              // 16 pixels per warp (4 x 4 patch on lanes 0-15) instead of 32: see build_relax_jobs
    int npx, npy, nzs;
    int n[3], periodic[3];
    double origin[3], Minv[9];
    double p0[3], dx[3], dy[3], dz;
    double d0[3];
    float Minvf[9];
    float d0f[3], R_rest, k_lat[2], k_rad;
};

#define PPFM_CHK_READER relax_checks_read
PPFM_CHK_STORAGE
#undef PPFM_CHK_READER
#ifndef PPFM_CHECKS
void relax_checks_read(unsigned long long *) {}
#endif

struct FireParams {
    float dt0, dt_max, finc, fdec, alpha0, falpha, fconv2;
    int n_min, max_iter;
};

__device__ __forceinline__ float rsqrt_fast(float x) {
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float rsqrt_refined(float x) {      // MUFU.RSQ + one Newton step: unit vectors to 1 ulp
    const float y = rsqrt_fast(x);
    return y * fmaf(-0.5f * x * y, y, 1.5f);
}
__device__ __forceinline__ float sqrt_fast(float x) {
    float y;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
// The spring chain's two MUFU.  `volatile` keeps the front end from merging or moving them, but ptxas still schedules
// them freely against arithmetic: whether MUFU.SQRT issues ~15 instructions ahead of the stale-cell vote or directly in
// front of its MUFU.RCP changes a lone warp's iteration time by 15-40 %, and it is the register budget (RX_MIN_CTAS)
// that decides it.
__device__ __forceinline__ float sqrt_pinned(float x) {
    float y;
    asm volatile("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float rcp_pinned(float x) {
    float y;
    asm volatile("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float rcp_fast(float x) {
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
// Read-only 16-byte gather.  volatile keeps the eight corner loads of an iteration in program order, all ahead of
// their first use, so they are in flight together (ptxas otherwise sinks them pairwise to save registers).
__device__ __forceinline__ float4 ldg_corner(const float4 *p) {
    float4 v;
    asm volatile("ld.global.nc.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
    return v;
}

// Per z-step constants of one grid axis for the magic-number cell lookup.
struct AxisBase {
    float tb, tbm;     // fractional part of the base coordinate, and the same minus 0.5
    float zlo, zhi;    // clamp bounds in the magic domain
    int K;             // cell index = float_as_int(zc) - K
    float lo, hi;      // non-periodic: coordinate range [lo, hi] (relative to the base cell) outside which S12 clamps
};

__device__ __forceinline__ AxisBase axis_base(double t, int n, int periodic) {
    AxisBase a;
    const double fl = floor(t);
    a.tb = (float)(t - fl);
    a.tbm = a.tb - 0.5f;
    int ib;
    if (periodic) {
        long long m = (long long)fl % n;
        if (m < 0) m += n;
        ib = (int)m;
        a.zlo = RX_MAGIC - (float)(n - 1);
        a.zhi = RX_MAGIC + (float)(n - 1);
        a.lo = -3.0e38f;
        a.hi = 3.0e38f;
    } else {
        ib = (int)fmin(fmax(fl, -(double)(1 << 20)), (double)(1 << 20));
        a.zlo = RX_MAGIC + (float)(-ib);
        a.zhi = RX_MAGIC + (float)(n - 2 - ib);
        a.lo = (float)(-ib);
        a.hi = (float)(n - 1 - ib);
    }
    a.K = RX_MAGIC_BITS - ib;
    return a;
}

// cell offset fl (float, relative to the base cell) and absolute cell index i0 (before periodic wrap) from t, t - 0.5
__device__ __forceinline__ void axis_cell(float t, float tm, const AxisBase &a, int &i0, float &fl) {
    (void)t;
    const float z = tm + RX_MAGIC;                       // nearest integer of t - 0.5 = floor(t) (ties are harmless:
    const float zc = fminf(fmaxf(z, a.zlo), a.zhi);      //   the interpolant is continuous across cell faces)
    fl = zc - RX_MAGIC;
    i0 = __float_as_int(zc) - a.K;
}

// Eigenvalues (ascending) of a symmetric 3 x 3 matrix in FP32, for the stiffness map folded into the relaxation
// (SURVEY 8(f) N2).  The two soft lateral modes (~k_xy) are nearly degenerate next to the stiff radial one (~k_R), and
// any route through all three roots of the characteristic cubic loses the close pair to sqrt(eps).  Instead (the
// deflation scheme of robust 3 x 3 symmetric solvers): with B = (A - q I)/p, q = tr A/3, p^2 = |A - q I|_F^2/6, the
// roots of mu^3 - 3 mu - det B = 0 lie in [-2, 2]; the root on the side of sign(det B) is the ISOLATED one
// (|mu| in [sqrt 3, 2], slope >= 6), found by Newton from |mu| = 2 (monotone: the cubic is convex there).  Its
// eigenvector is the largest cross product of two rows of A - lambda I; the other two eigenvalues are those of A
// projected on the plane orthogonal to it, mean +- sqrt(diff^2 + off^2): no cancellation between close roots.
// Error ~ a few ulp of |A| (2e-7 for k_R = 1.9 eV/A^2; tolerance of the map 1e-5).
__device__ __forceinline__ void sym3_eigenvalues_f32(float a00, float a11, float a22, float a01, float a02, float a12,
                                                     float &e0, float &e1, float &e2) {
    const float q = (a00 + a11 + a22) * (1.0f / 3.0f);
    const float b00 = a00 - q, b11 = a11 - q, b22 = a22 - q;
    const float p2 = (fmaf(b00, b00, fmaf(b11, b11, b22 * b22)) + 2.0f * fmaf(a01, a01, fmaf(a02, a02, a12 * a12))) *
                     (1.0f / 6.0f);
    if (!(p2 > 1.0e-30f)) { e0 = e1 = e2 = q; return; }
    const float ip = rsqrt_fast(p2), p = p2 * ip;
    const float c00 = b00 * ip, c11 = b11 * ip, c22 = b22 * ip, c01 = a01 * ip, c02 = a02 * ip, c12 = a12 * ip;
    const float det = c00 * fmaf(c11, c22, -c12 * c12) - c01 * fmaf(c01, c22, -c12 * c02) + c02 * fmaf(c01, c12, -c11 * c02);
    const float sgn = (det >= 0.0f) ? 1.0f : -1.0f;
    const float ad = fminf(fabsf(det), 2.0f);
    float mu = 2.0f;
    // from mu = 2 the worst case (root sqrt 3) is within 1e-6 after three steps and converged after four; an
    // approximate reciprocal is enough inside a Newton step (the iteration corrects its own rounding)
#pragma unroll
    for (int it = 0; it < 5; it++) {
        const float f = fmaf(mu, fmaf(mu, mu, -3.0f), -ad);
        mu = fmaf(-f, rcp_fast(fmaf(3.0f * mu, mu, -3.0f)), mu);
    }
    const float liso = sgn * mu;                       // isolated eigenvalue of C = B/p
    // eigenvector of liso: largest cross product of two rows of C - liso I
    const float m00 = c00 - liso, m11 = c11 - liso, m22 = c22 - liso;
    const float x0 = fmaf(c01, c12, -c02 * m11), y0 = fmaf(c02, c01, -m00 * c12), z0 = fmaf(m00, m11, -c01 * c01);   // r0 x r1
    const float x1 = fmaf(c01, m22, -c02 * c12), y1 = fmaf(c02, c02, -m00 * m22), z1 = fmaf(m00, c12, -c01 * c02);   // r0 x r2
    const float x2 = fmaf(m11, m22, -c12 * c12), y2 = fmaf(c12, c02, -c01 * m22), z2 = fmaf(c01, c12, -m11 * c02);   // r1 x r2
    const float n0 = fmaf(x0, x0, fmaf(y0, y0, z0 * z0)), n1 = fmaf(x1, x1, fmaf(y1, y1, z1 * z1));
    const float n2 = fmaf(x2, x2, fmaf(y2, y2, z2 * z2));
    float vx = x0, vy = y0, vz = z0, nn = n0;
    if (n1 > nn) { vx = x1; vy = y1; vz = z1; nn = n1; }
    if (n2 > nn) { vx = x2; vy = y2; vz = z2; nn = n2; }
    const float inn = rsqrt_refined(nn);
    vx *= inn; vy *= inn; vz *= inn;
    // orthonormal a, b spanning the plane orthogonal to v: a = e_k x v for the smallest |v_k|
    const float ax_ = fabsf(vx), ay_ = fabsf(vy), az_ = fabsf(vz);
    float ux, uy, uz;
    if (ax_ <= ay_ && ax_ <= az_) { ux = 0.0f; uy = -vz; uz = vy; }
    else if (ay_ <= az_) { ux = vz; uy = 0.0f; uz = -vx; }
    else { ux = -vy; uy = vx; uz = 0.0f; }
    const float iu = rsqrt_refined(fmaf(ux, ux, fmaf(uy, uy, uz * uz)));
    ux *= iu; uy *= iu; uz *= iu;
    const float wx = fmaf(vy, uz, -vz * uy), wy = fmaf(vz, ux, -vx * uz), wz = fmaf(vx, uy, -vy * ux);
    // C u, C w and the projected 2 x 2 matrix
    const float cux = fmaf(c00, ux, fmaf(c01, uy, c02 * uz)), cuy = fmaf(c01, ux, fmaf(c11, uy, c12 * uz));
    const float cuz = fmaf(c02, ux, fmaf(c12, uy, c22 * uz));
    const float cwx = fmaf(c00, wx, fmaf(c01, wy, c02 * wz)), cwy = fmaf(c01, wx, fmaf(c11, wy, c12 * wz));
    const float cwz = fmaf(c02, wx, fmaf(c12, wy, c22 * wz));
    const float muu = fmaf(ux, cux, fmaf(uy, cuy, uz * cuz)), mww = fmaf(wx, cwx, fmaf(wy, cwy, wz * cwz));
    const float muw = fmaf(ux, cwx, fmaf(uy, cwy, uz * cwz));
    const float mean = 0.5f * (muu + mww), hd = 0.5f * (muu - mww);
    const float sq = sqrt_fast(fmaf(hd, hd, muw * muw));
    const float la = fmaf(p, mean - sq, q), lb = fmaf(p, mean + sq, q), li = fmaf(p, liso, q);
    if (sgn > 0.0f) { e0 = la; e1 = lb; e2 = li; }
    else { e0 = li; e1 = la; e2 = lb; }
}

// Inputs of the stiffness map at the end of a z-step: the cached cell (the eight coefficients of the tri-linear
// polynomial per force component, see relax_pixels), the in-cell fractions, d = r_PP - r_TIP and
// fr = -k_R (|d| - R0)/|d|.
struct StiffIn {
    float a[8][3];
    float f[3], d[3], fr;
};

// G[c][a] = dF_c/dt_a of the tri-linear interpolant, J = G Minv, H = H_spring - (J + J^T)/2 with
// H_spring = k_R dd^T/|d|^2 + k_t (I - dd^T/|d|^2) + diag(k_x, k_y, 0), k_t = k_R (|d| - R0)/|d| = -fr; eigenvalues ascending.
template <bool ORTHO>
__device__ __noinline__ float4 stiffness_from_cell(const StiffIn in, const RelaxJob &job) {
    const float fx = in.f[0], fy = in.f[1], fz = in.f[2];
    float G[3][3];               // dF_c/dt_a: derivatives of a0 + a1 x + a2 y + a3 z + a4 xy + a5 xz + a6 yz + a7 xyz
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const float a1 = in.a[1][c], a2 = in.a[2][c], a3 = in.a[3][c], a4 = in.a[4][c], a5 = in.a[5][c], a6 = in.a[6][c],
                    a7 = in.a[7][c];
        G[c][0] = fmaf(fz, fmaf(fy, a7, a5), fmaf(fy, a4, a1));
        G[c][1] = fmaf(fz, fmaf(fx, a7, a6), fmaf(fx, a4, a2));
        G[c][2] = fmaf(fy, fmaf(fx, a7, a6), fmaf(fx, a5, a3));
    }
    const float *m = job.Minvf;
    float J[3][3];
#pragma unroll
    for (int c = 0; c < 3; c++) {
        if (ORTHO) {
            J[c][0] = G[c][0] * m[0]; J[c][1] = G[c][1] * m[4]; J[c][2] = G[c][2] * m[8];
        } else {
            J[c][0] = fmaf(G[c][2], m[6], fmaf(G[c][1], m[3], G[c][0] * m[0]));
            J[c][1] = fmaf(G[c][2], m[7], fmaf(G[c][1], m[4], G[c][0] * m[1]));
            J[c][2] = fmaf(G[c][2], m[8], fmaf(G[c][1], m[5], G[c][0] * m[2]));
        }
    }
    const float ddx = in.d[0], ddy = in.d[1], ddz = in.d[2];
    const float L2 = fmaf(ddx, ddx, fmaf(ddy, ddy, ddz * ddz));
    const float kt = -in.fr;
    const float kd = (L2 > 0.0f) ? (job.k_rad - kt) * rcp_fast(L2) : 0.0f;
    const float h00 = fmaf(kd * ddx, ddx, kt) - J[0][0] + job.k_lat[0];
    const float h11 = fmaf(kd * ddy, ddy, kt) - J[1][1] + job.k_lat[1];
    const float h22 = fmaf(kd * ddz, ddz, kt) - J[2][2];
    const float h01 = fmaf(kd * ddx, ddy, -0.5f * (J[0][1] + J[1][0]));
    const float h02 = fmaf(kd * ddx, ddz, -0.5f * (J[0][2] + J[2][0]));
    const float h12 = fmaf(kd * ddy, ddz, -0.5f * (J[1][2] + J[2][1]));
    float l0, l1, l2;
    sym3_eigenvalues_f32(h00, h11, h22, h01, h02, h12, l0, l1, l2);
    return make_float4(l0, l1, l2, 0.0f);
}

template <bool ORTHO, bool ANYPER, bool SYMTIP, bool TRICUBIC, bool STIFF = false>
__device__ __forceinline__ void relax_pixels(const RelaxJob &job, const FireParams &fp, int lb,
                                             const void *__restrict__ ff, float4 *__restrict__ pos_fz,
                                             uint16_t *__restrict__ iters_out, ppfm_stats *__restrict__ stats,
                                             float *__restrict__ fz_out, float4 *__restrict__ eig_out) {
    const int by = lb / job.nbx, bx = lb - by * job.nbx;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const bool sparse = job.sparse != 0;
    const int ix = sparse ? bx * (RX_TILE_X / 2) + (warp & 1) * 4 + (lane & 3) : bx * RX_TILE_X + (warp & 1) * 8 + (lane & 7);
    const int iy = sparse ? by * RX_TILE_Y + (warp >> 1) * 4 + ((lane >> 2) & 3) : by * RX_TILE_Y + (warp >> 1) * 4 + (lane >> 3);
    const bool valid = (ix < job.npx) && (iy < job.npy) && (!sparse || lane < 16);
    const int ixc = min(ix, job.npx - 1), iyc = min(iy, job.npy - 1);

    // tri-linear: float4 (Fx,Fy,Fz,E) grid; TRICUBIC: energy-only float grid
    const float4 *__restrict__ g = reinterpret_cast<const float4 *>(ff) + (TRICUBIC ? 0 : job.ff_offset);
    const float *__restrict__ ge = reinterpret_cast<const float *>(ff) + (TRICUBIC ? job.ff_offset : 0);
    const int nx = job.n[0], ny = job.n[1], nz = job.n[2];
    const int perx = job.periodic[0], pery = job.periodic[1], perz = job.periodic[2];
    const float m00 = job.Minvf[0], m01 = job.Minvf[1], m02 = job.Minvf[2];
    const float m10 = job.Minvf[3], m11 = job.Minvf[4], m12 = job.Minvf[5];
    const float m20 = job.Minvf[6], m21 = job.Minvf[7], m22 = job.Minvf[8];
    const float d0x = job.d0f[0], d0y = job.d0f[1], d0z = job.d0f[2];
    const float d0x2 = 2.0f * d0x, d0y2 = 2.0f * d0y, d0z2 = 2.0f * d0z;
    const float R_rest = job.R_rest, nk_rad = -job.k_rad, nkx = -job.k_lat[0], nky = -job.k_lat[1];
    const long long sy = nx, sz = (long long)nx * ny;       // float4 strides

    // r_TIP + d0 - origin at iz = 0, FP64
    double rb[3];
#pragma unroll
    for (int c = 0; c < 3; c++)
        rb[c] = job.p0[c] + ixc * job.dx[c] + iyc * job.dy[c] + job.d0[c] - job.origin[c];

    float ux = 0.f, uy = 0.f, uz = 0.f;
    unsigned long long my_iters = 0;
    unsigned int my_notconv = 0, my_clamped = 0, my_max = 0, my_reloads = 0, my_witers = 0, my_wreloads = 0;

    // per z-step state (set by begin_step): axis bases of the spring equilibrium point, FIRE state
    AxisBase ax = {}, ay = {}, az = {};
    float vx = 0.f, vy = 0.f, vz = 0.f, dt = fp.dt0, alpha = fp.alpha0;
    int npos = 0, moves = 0;
    bool conv = !valid;
    float fr = 0.f, dzc = d0z, fx = 0.f, fy = 0.f, fz = 0.f;
    // cached cell: per force component the eight coefficients of the tri-linear polynomial in the in-cell fractions,
    //   F = a0 + a1 x + a2 y + a3 z + a4 xy + a5 xz + a6 yz + a7 xyz
    // (formed from the eight corners when the cell is gathered; evaluated by Horner in 7 FFMA of depth 3, where nested
    // lerps on the corners take 10 operations of depth 5), and per axis tbf = (fraction of the z-step's base point) -
    // (offset of the cached cell from the base cell), so that the position inside the cell is one FFMA:
    // f = Minv u + tbf.  An impossible offset makes the first iteration gather.
    float tbfx = -1.0e30f, tbfy = -1.0e30f, tbfz = -1.0e30f;
    float ca[8][3];
#pragma unroll
    for (int e = 0; e < 8; e++)
#pragma unroll
        for (int c = 0; c < 3; c++) ca[e][c] = 0.0f;
    // TRICUBIC: the 4 x 4 x 4 energies around the cell, [z][y][x], minus the value at the cell's own node (the
    // gradient does not see a constant, and differences of ~|F| h keep FP32 rounding far below f_conv)
    float en[TRICUBIC ? 4 : 1][TRICUBIC ? 4 : 1][TRICUBIC ? 4 : 1];
    if (TRICUBIC) {
#pragma unroll
        for (int a = 0; a < (TRICUBIC ? 4 : 1); a++)
#pragma unroll
            for (int b = 0; b < (TRICUBIC ? 4 : 1); b++)
#pragma unroll
                for (int c = 0; c < (TRICUBIC ? 4 : 1); c++) en[a][b][c] = 0.0f;
    }

    auto interp = [&](float (&S)[3]) {     // Horner in x, y, z on the cached coefficients: 7 FFMA per component, depth 3
        if (TRICUBIC) {
            // F_S = -grad of the tri-cubic (Catmull-Rom per axis, reading S22) interpolant of the energies:
            // weights w and their derivatives d per axis (Horner), x pass per (z,y) row, y pass per z plane, z pass
            float w[3][4], d[3][4];
            const float fa[3] = {fx, fy, fz};
#pragma unroll
            for (int a = 0; a < 3; a++) {
                const float f = fa[a], f2 = f * f;
                w[a][0] = fmaf(fmaf(-0.5f, f, 1.0f), f, -0.5f) * f;
                w[a][1] = fmaf(fmaf(1.5f, f, -2.5f), f2, 1.0f);
                w[a][2] = fmaf(fmaf(-1.5f, f, 2.0f), f, 0.5f) * f;
                w[a][3] = fmaf(0.5f, f, -0.5f) * f2;
                d[a][0] = fmaf(fmaf(-1.5f, f, 2.0f), f, -0.5f);
                d[a][1] = fmaf(4.5f, f, -5.0f) * f;
                d[a][2] = fmaf(fmaf(-4.5f, f, 4.0f), f, 0.5f);
                d[a][3] = fmaf(1.5f, f, -1.0f) * f;
            }
            float Ex = 0.f, Ey = 0.f, Ez = 0.f;            // dE/dt along the three grid axes
#pragma unroll
            for (int k = 0; k < (TRICUBIC ? 4 : 1); k++) {
                float V = 0.f, DX = 0.f, DY = 0.f;
#pragma unroll
                for (int j = 0; j < (TRICUBIC ? 4 : 1); j++) {
                    const float *r = en[k][j];
                    const float v = fmaf(w[0][3], r[TRICUBIC ? 3 : 0], fmaf(w[0][2], r[TRICUBIC ? 2 : 0], fmaf(w[0][1], r[TRICUBIC ? 1 : 0], w[0][0] * r[0])));
                    const float dxv = fmaf(d[0][3], r[TRICUBIC ? 3 : 0], fmaf(d[0][2], r[TRICUBIC ? 2 : 0], fmaf(d[0][1], r[TRICUBIC ? 1 : 0], d[0][0] * r[0])));
                    V = fmaf(w[1][j], v, V);
                    DX = fmaf(w[1][j], dxv, DX);
                    DY = fmaf(d[1][j], v, DY);
                }
                Ex = fmaf(w[2][k], DX, Ex);
                Ey = fmaf(w[2][k], DY, Ey);
                Ez = fmaf(d[2][k], V, Ez);
            }
            if (ORTHO) {
                S[0] = -m00 * Ex; S[1] = -m11 * Ey; S[2] = -m22 * Ez;
            } else {                                         // F_c = -sum_a dE/dt_a Minv[a][c]
                S[0] = -fmaf(m20, Ez, fmaf(m10, Ey, m00 * Ex));
                S[1] = -fmaf(m21, Ez, fmaf(m11, Ey, m01 * Ex));
                S[2] = -fmaf(m22, Ez, fmaf(m12, Ey, m02 * Ex));
            }
        }
#pragma unroll
        for (int c = 0; c < (TRICUBIC ? 0 : 3); c++) {
            const float p0 = fmaf(fx, ca[1][c], ca[0][c]);
            const float p1 = fmaf(fx, ca[4][c], ca[2][c]);
            const float p2 = fmaf(fx, ca[5][c], ca[3][c]);
            const float p3 = fmaf(fx, ca[7][c], ca[6][c]);
            S[c] = fmaf(fz, fmaf(fy, p3, p2), fmaf(fy, p1, p0));
        }
    };

    auto fire_iteration = [&]() -> bool {
        // ---- position inside the cached cell
        if (ORTHO) {
            fx = fmaf(m00, ux, tbfx);
            fy = fmaf(m11, uy, tbfy);
            fz = fmaf(m22, uz, tbfz);
        } else {
            fx = fmaf(m00, ux, fmaf(m01, uy, fmaf(m02, uz, tbfx)));
            fy = fmaf(m10, ux, fmaf(m11, uy, fmaf(m12, uz, tbfy)));
            fz = fmaf(m20, ux, fmaf(m21, uy, fmaf(m22, uz, tbfz)));
        }
        // outside [0,1] on any axis?  As unsigned integers, negative floats and floats > 1 both exceed bits(1.0f).
        const unsigned worst = max(max(__float_as_uint(fx), __float_as_uint(fy)), __float_as_uint(fz));
        // ---- F_T first (the longest dependency chain: two MUFU): radial + lateral springs (Eq.2) with d = d0 + u;
        // (|d| - R0)/|d| = (|u|^2 + 2 d0.u)/(|d|(|d| + R0))
        float dxc = ux, dyc = uy, frk;
        dzc = d0z + uz;
        if (SYMTIP) {                      // d0 = (0, 0, d0z) and k_x = k_y: the usual symmetric tip
            const float w = fmaf(ux, ux, uy * uy);
            const float L2 = fmaf(dzc, dzc, w);
            const float num = fmaf(uz, uz + d0z2, w);                                    // |u|^2 + 2 d0.u
            const float L = sqrt_pinned(L2);
            fr = (nk_rad * num) * rcp_pinned(fmaf(R_rest, L, L2));                       // -k_R (|d| - R0)/|d|
            frk = fr + nkx;
        } else {
            dxc = d0x + ux; dyc = d0y + uy;
            const float L2 = fmaf(dxc, dxc, fmaf(dyc, dyc, dzc * dzc));
            const float num = fmaf(ux, ux + d0x2, fmaf(uy, uy + d0y2, uz * (uz + d0z2)));
            const float L = sqrt_pinned(L2);
            fr = (nk_rad * num) * rcp_pinned(fmaf(R_rest, L, L2));
            frk = fr;
        }
        // ---- F_S, speculatively from the cached cell (redone below in the rare case that a lane left its cell)
        // (the tri-cubic field is 233 instructions: not worth computing twice, it waits for the vote instead)
        float S[3];
        if (!TRICUBIC) interp(S);
        if (__any_sync(0xffffffffu, worst > 0x3F800000u)) {
            // ---- some lane's PP left its cell.  The block is warp-uniform (no reconvergence barrier on the hot
            // path): every lane locates its cell again (magic-number floor, S12 clamp) and gathers it; lanes
            // that had not moved get the cell they already hold, from L1.
            float tx, ty, tz;
            if (ORTHO) {
                tx = fmaf(m00, ux, ax.tb);
                ty = fmaf(m11, uy, ay.tb);
                tz = fmaf(m22, uz, az.tb);
            } else {
                tx = fmaf(m00, ux, fmaf(m01, uy, fmaf(m02, uz, ax.tb)));
                ty = fmaf(m10, ux, fmaf(m11, uy, fmaf(m12, uz, ay.tb)));
                tz = fmaf(m20, ux, fmaf(m21, uy, fmaf(m22, uz, az.tb)));
            }
            int i0, j0, k0;
            float flx, fly, flz;
            axis_cell(tx, tx - 0.5f, ax, i0, flx);
            axis_cell(ty, ty - 0.5f, ay, j0, fly);
            axis_cell(tz, tz - 0.5f, az, k0, flz);
            float4 c000, c001, c010, c011, c100, c101, c110, c111;
            if (TRICUBIC) {
                // 4 x 4 x 4 stencil i0-1 .. i0+2 (reading S22).  Interior cells of the whole warp: 16 row bases and
                // immediate offsets.  Otherwise per-axis index lists: wrap on periodic axes, clamp to [0, n-1] on
                // the others.
                const bool inside = (i0 >= 1) & (i0 + 2 <= nx - 1) & (j0 >= 1) & (j0 + 2 <= ny - 1) & (k0 >= 1) &
                                    (k0 + 2 <= nz - 1);
                if (__all_sync(0xffffffffu, inside)) {
                    PPFM_CHK(PPFM_CHK_RELAX_GATHER, i0 >= 1 && i0 + 2 <= nx - 1 && j0 >= 1 && j0 + 2 <= ny - 1 && k0 >= 1 && k0 + 2 <= nz - 1);
                    const int base = (int)((k0 - 1) * ny + (j0 - 1)) * nx + (i0 - 1);
#pragma unroll
                    for (int kk = 0; kk < (TRICUBIC ? 4 : 1); kk++)
#pragma unroll
                        for (int jj = 0; jj < (TRICUBIC ? 4 : 1); jj++) {
                            const float *row = ge + (base + (kk * ny + jj) * nx);
#pragma unroll
                            for (int m = 0; m < (TRICUBIC ? 4 : 1); m++) en[kk][jj][m] = __ldg(row + m);
                        }
                } else {
                    int xi[4], yo[4], zo[4];
                    int iw = i0, jw = j0, kw = k0;              // periodic: |index - [0,n)| < n after axis_cell
                    if (perx) { iw -= (iw >= nx) ? nx : 0; iw += (iw < 0) ? nx : 0; }
                    if (pery) { jw -= (jw >= ny) ? ny : 0; jw += (jw < 0) ? ny : 0; }
                    if (perz) { kw -= (kw >= nz) ? nz : 0; kw += (kw < 0) ? nz : 0; }
#pragma unroll
                    for (int m = 0; m < 4; m++) {
                        int a = iw + m - 1, b = jw + m - 1, c = kw + m - 1;
                        if (perx) { a -= (a >= nx) ? nx : 0; a += (a < 0) ? nx : 0; } else a = min(max(a, 0), nx - 1);
                        if (pery) { b -= (b >= ny) ? ny : 0; b += (b < 0) ? ny : 0; } else b = min(max(b, 0), ny - 1);
                        if (perz) { c -= (c >= nz) ? nz : 0; c += (c < 0) ? nz : 0; } else c = min(max(c, 0), nz - 1);
                        PPFM_CHK(PPFM_CHK_RELAX_GATHER, a >= 0 && a < nx && b >= 0 && b < ny && c >= 0 && c < nz);
                        xi[m] = a; yo[m] = b * nx; zo[m] = c * ny * nx;
                    }
#pragma unroll
                    for (int kk = 0; kk < (TRICUBIC ? 4 : 1); kk++)
#pragma unroll
                        for (int jj = 0; jj < (TRICUBIC ? 4 : 1); jj++) {
                            const int ro = zo[kk] + yo[jj];
#pragma unroll
                            for (int m = 0; m < (TRICUBIC ? 4 : 1); m++) en[kk][jj][m] = __ldg(ge + (ro + xi[m]));
                        }
                }
                const float ref = en[TRICUBIC ? 1 : 0][TRICUBIC ? 1 : 0][TRICUBIC ? 1 : 0];
#pragma unroll
                for (int kk = 0; kk < (TRICUBIC ? 4 : 1); kk++)
#pragma unroll
                    for (int jj = 0; jj < (TRICUBIC ? 4 : 1); jj++)
#pragma unroll
                        for (int m = 0; m < (TRICUBIC ? 4 : 1); m++) en[kk][jj][m] -= ref;
            } else if (!ANYPER) {
                PPFM_CHK(PPFM_CHK_RELAX_GATHER, i0 >= 0 && i0 <= nx - 2 && j0 >= 0 && j0 <= ny - 2 && k0 >= 0 && k0 <= nz - 2);
                const float4 *p = g + ((long long)(k0 * ny + j0) * nx + i0);
                c000 = ldg_corner(p);           c001 = ldg_corner(p + 1);
                c010 = ldg_corner(p + sy);      c011 = ldg_corner(p + sy + 1);
                c100 = ldg_corner(p + sz);      c101 = ldg_corner(p + sz + 1);
                c110 = ldg_corner(p + sz + sy); c111 = ldg_corner(p + sz + sy + 1);
            } else {
                if (perx) { i0 -= (i0 >= nx) ? nx : 0; i0 += (i0 < 0) ? nx : 0; }
                if (pery) { j0 -= (j0 >= ny) ? ny : 0; j0 += (j0 < 0) ? ny : 0; }
                if (perz) { k0 -= (k0 >= nz) ? nz : 0; k0 += (k0 < 0) ? nz : 0; }
                const int i1 = (i0 + 1 == nx) ? 0 : i0 + 1;       // non-periodic axes never reach n - 1
                const int j1 = (j0 + 1 == ny) ? 0 : j0 + 1;
                const int k1 = (k0 + 1 == nz) ? 0 : k0 + 1;
                PPFM_CHK(PPFM_CHK_RELAX_GATHER, i0 >= 0 && i0 < nx && j0 >= 0 && j0 < ny && k0 >= 0 && k0 < nz &&
                                                    i1 < nx && j1 < ny && k1 < nz);
                const float4 *r00 = g + (long long)(k0 * ny + j0) * nx, *r01 = g + (long long)(k0 * ny + j1) * nx;
                const float4 *r10 = g + (long long)(k1 * ny + j0) * nx, *r11 = g + (long long)(k1 * ny + j1) * nx;
                c000 = ldg_corner(r00 + i0); c001 = ldg_corner(r00 + i1);
                c010 = ldg_corner(r01 + i0); c011 = ldg_corner(r01 + i1);
                c100 = ldg_corner(r10 + i0); c101 = ldg_corner(r10 + i1);
                c110 = ldg_corner(r11 + i0); c111 = ldg_corner(r11 + i1);
            }
            tbfx = ax.tb - flx; tbfy = ay.tb - fly; tbfz = az.tb - flz;
            if (ORTHO) {
                fx = __saturatef(fmaf(m00, ux, tbfx));
                fy = __saturatef(fmaf(m11, uy, tbfy));
                fz = __saturatef(fmaf(m22, uz, tbfz));
            } else {
                fx = __saturatef(fmaf(m00, ux, fmaf(m01, uy, fmaf(m02, uz, tbfx))));
                fy = __saturatef(fmaf(m10, ux, fmaf(m11, uy, fmaf(m12, uz, tbfy))));
                fz = __saturatef(fmaf(m20, ux, fmaf(m21, uy, fmaf(m22, uz, tbfz))));
            }
            if (!TRICUBIC) {
#define PPFM_COEF(C, I)                                                              \
    {                                                                                \
        const float d0 = c001.C - c000.C, d1 = c011.C - c010.C, d2 = c101.C - c100.C, d3 = c111.C - c110.C; \
        const float e2 = c010.C - c000.C, e6 = c110.C - c100.C;                      \
        ca[0][I] = c000.C; ca[1][I] = d0; ca[2][I] = e2; ca[3][I] = c100.C - c000.C; \
        ca[4][I] = d1 - d0; ca[5][I] = d2 - d0; ca[6][I] = e6 - e2;                  \
        ca[7][I] = (d3 - d2) - (d1 - d0);                                            \
    }
            PPFM_COEF(x, 0) PPFM_COEF(y, 1) PPFM_COEF(z, 2)
#undef PPFM_COEF
            }
            my_reloads += (worst > 0x3F800000u) ? 1u : 0u;
            my_wreloads++;
            if (!TRICUBIC) interp(S);
        }
        if (TRICUBIC) interp(S);
        float Fx, Fy, Fz;
        if (SYMTIP) {
            Fx = fmaf(frk, ux, S[0]);
            Fy = fmaf(frk, uy, S[1]);
        } else {
            Fx = fmaf(fr, dxc, fmaf(nkx, ux, S[0]));
            Fy = fmaf(fr, dyc, fmaf(nky, uy, S[1]));
        }
        Fz = fmaf(fr, dzc, S[2]);
        // ---- the part of FIRE that needs only the old velocity (reading S6), off the critical path
        const float vn = sqrt_fast(fmaf(vx, vx, fmaf(vy, vy, vz * vz)));
        const float av = alpha * vn, om = 1.0f - alpha;
        const bool grow = npos > fp.n_min;
        const float dt_pos = grow ? fminf(dt * fp.finc, fp.dt_max) : dt;
        const float al_pos = grow ? alpha * fp.falpha : alpha;
        const float dt_neg = dt * fp.fdec;
        const float F2 = fmaf(Fx, Fx, fmaf(Fy, Fy, Fz * Fz));
        const float Pw = fmaf(Fx, vx, fmaf(Fy, vy, Fz * vz));
        conv = conv || (F2 < fp.fconv2);                     // tested before every move (reading S7)
        const bool done = conv || (moves >= fp.max_iter);
        // ---- FIRE step, branch-free; P >= 0 counts as downhill
        const bool down = Pw >= 0.0f;
        const float omv = down ? om : 0.0f;
        const float s = down ? fmaf(av, rsqrt_fast(F2), dt_pos) : dt_neg;
        vx = fmaf(s, Fx, omv * vx);
        vy = fmaf(s, Fy, omv * vy);
        vz = fmaf(s, Fz, omv * vz);
        dt = down ? dt_pos : dt_neg;
        alpha = down ? al_pos : fp.alpha0;
        npos = down ? npos + 1 : 0;
        if (!done) {                                         // finished lanes stay where they are
            ux = fmaf(vx, dt, ux); uy = fmaf(vy, dt, uy); uz = fmaf(vz, dt, uz);
            moves++;
        }
        return done;
    };

    // start of a z-step (O7): FIRE state reset, the displacement u is carried over; the cached cell is dropped
    auto reset_step = [&]() {
        vx = vy = vz = 0.f; dt = fp.dt0; alpha = fp.alpha0;
        npos = 0; moves = 0;
        conv = !valid;
        tbfx = tbfy = tbfz = -1.0e30f;
    };
    // end of a z-step (O8): outputs of this pixel at tip height index iz
    auto finish_step = [&](int iz) {
        const double rz = rb[2] - iz * job.dz;
        const size_t o = (size_t)job.out_offset + ((size_t)iz * job.npy + iy) * job.npx + ix;
        float4 outv;
        outv.x = (float)(rb[0] + job.origin[0] + (double)ux);
        outv.y = (float)(rb[1] + job.origin[1] + (double)uy);
        outv.z = (float)(rz + job.origin[2] + (double)uz);
        outv.w = -fr * dzc;                           // Fz_tip = -F_R,z
        PPFM_CHK(PPFM_CHK_RELAX_STORE, o < (size_t)job.out_offset + (size_t)job.nzs * job.npy * job.npx);
        pos_fz[o] = outv;
        if (fz_out) fz_out[o] = outv.w;
        if (iters_out) iters_out[o] = conv ? (uint16_t)min(moves, 0xFFFE) : (uint16_t)0xFFFF;
        if (STIFF && !TRICUBIC) {
            // Stiffness map from the cell this lane still holds: the last FIRE
            // iteration of a finished lane does not move it, so (c0, cd, fx, fy, fz, fr, dzc) belong to the relaxed
            // point.  Done in a function that is NOT inlined: the FIRE loop's instruction schedule and register
            // allocation then stay those of the plain kernel (inlined, the ~200 extra instructions per z-step cost
            // config 1 a quarter of its speed through the loop's schedule, DESIGN.md §7 "schedule sensitivity").
            StiffIn in;
#pragma unroll
            for (int e = 0; e < 8; e++)
#pragma unroll
                for (int c = 0; c < 3; c++) in.a[e][c] = ca[e][c];
            in.f[0] = fx; in.f[1] = fy; in.f[2] = fz;
            in.d[0] = SYMTIP ? ux : d0x + ux; in.d[1] = SYMTIP ? uy : d0y + uy; in.d[2] = dzc;
            in.fr = fr;
            eig_out[o] = stiffness_from_cell<ORTHO>(in, job);
        }
        float tx, ty, tz;
        if (ORTHO) {
            tx = fmaf(m00, ux, ax.tb); ty = fmaf(m11, uy, ay.tb); tz = fmaf(m22, uz, az.tb);
        } else {
            tx = fmaf(m00, ux, fmaf(m01, uy, fmaf(m02, uz, ax.tb)));
            ty = fmaf(m10, ux, fmaf(m11, uy, fmaf(m12, uz, ay.tb)));
            tz = fmaf(m20, ux, fmaf(m21, uy, fmaf(m22, uz, az.tb)));
        }
        const bool clamped = (tx < ax.lo) | (tx > ax.hi) | (ty < ay.lo) | (ty > ay.hi) | (tz < az.lo) | (tz > az.hi);
        my_iters += (unsigned)moves;
        my_notconv += conv ? 0u : 1u;
        my_clamped += clamped ? 1u : 0u;
        my_max = max(my_max, (unsigned)moves);
    };

    for (int iz = 0; iz < job.nzs; iz++) {
        // a4: exact fractional grid coordinate of the spring equilibrium point, split int + frac
        const double rz = rb[2] - iz * job.dz;
        ax = axis_base(job.Minv[0] * rb[0] + job.Minv[1] * rb[1] + job.Minv[2] * rz, nx, perx);
        ay = axis_base(job.Minv[3] * rb[0] + job.Minv[4] * rb[1] + job.Minv[5] * rz, ny, pery);
        az = axis_base(job.Minv[6] * rb[0] + job.Minv[7] * rb[1] + job.Minv[8] * rz, nz, perz);
        reset_step();
        // the convergence vote is taken every second iteration: finished lanes do not move, so an extra iteration
        // changes nothing but saves one VOTE + branch per iteration
        while (true) {
            fire_iteration();
            const bool done = fire_iteration();
            my_witers += 2;
            if (__all_sync(0xffffffffu, done)) break;
        }
        if (valid) finish_step(iz);
    }

    if (stats) {
#pragma unroll
        for (int s = 16; s > 0; s >>= 1) {
            my_iters += __shfl_xor_sync(0xffffffffu, my_iters, s);
            my_notconv += __shfl_xor_sync(0xffffffffu, my_notconv, s);
            my_clamped += __shfl_xor_sync(0xffffffffu, my_clamped, s);
            my_max = max(my_max, __shfl_xor_sync(0xffffffffu, my_max, s));
        }
        unsigned long long rel = my_reloads;
#pragma unroll
        for (int s = 16; s > 0; s >>= 1) rel += __shfl_xor_sync(0xffffffffu, rel, s);
        if (lane == 0) {
            atomicAdd(reinterpret_cast<unsigned long long *>(&stats->warp_iters), (unsigned long long)my_witers);
            atomicAdd(reinterpret_cast<unsigned long long *>(&stats->cell_gathers), rel);
            atomicAdd(reinterpret_cast<unsigned long long *>(&stats->warp_gathers), (unsigned long long)my_wreloads);
            atomicAdd(reinterpret_cast<unsigned long long *>(&stats->total_iters), my_iters);
            if (my_notconv) atomicAdd(reinterpret_cast<unsigned long long *>(&stats->n_not_converged), (unsigned long long)my_notconv);
            if (my_clamped) atomicAdd(reinterpret_cast<unsigned long long *>(&stats->n_clamped), (unsigned long long)my_clamped);
            atomicMax(&stats->max_iters, my_max);
        }
    }
}

// One system: the job travels as a kernel parameter (constant bank), no scratch and no copy.
template <bool ORTHO, bool ANYPER, bool SYMTIP, bool TRICUBIC, bool STIFF>
__global__ void __launch_bounds__(RX_THREADS, TRICUBIC ? 3 : RX_MIN_CTAS)
relax_kernel(const __grid_constant__ RelaxJob job, const __grid_constant__ FireParams fp,
             const void *__restrict__ ff, float4 *__restrict__ pos_fz, uint16_t *__restrict__ iters_out,
             ppfm_stats *__restrict__ stats, float *__restrict__ fz_out, float4 *__restrict__ eig_out) {
    relax_pixels<ORTHO, ANYPER, SYMTIP, TRICUBIC, STIFF>(job, fp, blockIdx.x, ff, pos_fz, iters_out, stats, fz_out,
                                                         eig_out);
}

// Batch: the CTA finds its system in a device array and keeps a copy in shared memory.
template <bool ORTHO, bool ANYPER, bool SYMTIP, bool TRICUBIC, bool STIFF>
__global__ void __launch_bounds__(RX_THREADS, TRICUBIC ? 3 : RX_MIN_CTAS)
relax_batch_kernel(const RelaxJob *__restrict__ jobs, int njobs, const __grid_constant__ FireParams fp,
                   const void *__restrict__ ff, float4 *__restrict__ pos_fz, uint16_t *__restrict__ iters_out,
                   ppfm_stats *__restrict__ stats, float *__restrict__ fz_out, float4 *__restrict__ eig_out) {
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
    relax_pixels<ORTHO, ANYPER, SYMTIP, TRICUBIC, STIFF>(s_job, fp, blk - s_job.block_begin, ff, pos_fz, iters_out,
                                                         stats, fz_out, eig_out);
}

template <bool ORTHO, bool ANYPER, bool SYMTIP, bool TRICUBIC, bool STIFF>
static void launch_relax(int nsys, long long blocks, cudaStream_t st, const RelaxJob *hj, const RelaxJob *dj,
                         const FireParams &fp, const void *ff, float4 *pos, uint16_t *it, ppfm_stats *stats,
                         float *fz, float4 *eig) {
    if (nsys == 1)
        relax_kernel<ORTHO, ANYPER, SYMTIP, TRICUBIC, STIFF><<<(unsigned)blocks, RX_THREADS, 0, st>>>(
            hj[0], fp, ff, pos, it, stats, fz, eig);
    else
        relax_batch_kernel<ORTHO, ANYPER, SYMTIP, TRICUBIC, STIFF><<<(unsigned)blocks, RX_THREADS, 0, st>>>(
            dj, nsys, fp, ff, pos, it, stats, fz, eig);
}

// Host side shared by the relaxation and the stiffness map: validate and pack one RelaxJob per system.
static int build_relax_jobs(int nsys, const ppfm_grid *grids, const ppfm_tip *tips, const ppfm_scan *scans,
                            RelaxJob **hj_out, long long *blocks_out, long long *samples_out, bool *ortho_out,
                            bool *anyper_out, bool *symtip_out, bool shared_grid = false) {
    RelaxJob *hj = (RelaxJob *)calloc((size_t)nsys, sizeof(RelaxJob));
    if (!hj) return PPFM_ENOMEM;
    long long blocks = 0, ff_off = 0, out_off = 0;
    bool ortho = true, anyper = false, symtip = true;
    for (int m = 0; m < nsys; m++) {
        const ppfm_grid &g = grids[shared_grid ? 0 : m];     // sweep form: every scan reads the ONE grid at offset 0
        const ppfm_scan &s = scans[m];
        const ppfm_tip &t = tips[m];
        RelaxJob &j = hj[m];
        bool ok = grid_ok(&g) && g.n[0] >= 2 && g.n[1] >= 2 && g.n[2] >= 2 && g.n[0] <= RX_MAX_N && g.n[1] <= RX_MAX_N &&
                  g.n[2] <= RX_MAX_N && s.npx >= 1 && s.npy >= 1 && s.nz >= 1 && std::isfinite(s.dz) &&
                  invert_steps(g.step, j.Minv) && grid_points(&g) <= 0x7fffffffLL;
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
            anyper = anyper || (g.periodic[a] != 0);
            j.origin[a] = g.origin[a];
            j.p0[a] = s.p0[a]; j.dx[a] = s.dx[a]; j.dy[a] = s.dy[a];
            j.d0[a] = t.d0[a];
            j.d0f[a] = (float)t.d0[a];
            for (int c = 0; c < 3; c++)
                if (a != c && g.step[a][c] != 0.0) ortho = false;
        }
        for (int i = 0; i < 9; i++) j.Minvf[i] = (float)j.Minv[i];
        j.dz = s.dz;
        j.R_rest = (float)R0;
        j.k_lat[0] = (float)t.k_lat[0]; j.k_lat[1] = (float)t.k_lat[1];
        j.k_rad = (float)t.k_rad;
        if (t.d0[0] != 0.0 || t.d0[1] != 0.0 || j.k_lat[0] != j.k_lat[1]) symtip = false;
        blocks += (long long)j.nbx * ((s.npy + RX_TILE_Y - 1) / RX_TILE_Y);
        if (!shared_grid) ff_off += grid_points(&g);
        out_off += (long long)s.npx * s.npy * s.nz;
        if (blocks > 0x7fffffffLL) { free(hj); return PPFM_EINVAL; }
    }
    // Tiny launches (at most half a warp per SM sub-partition, so that even with twice the warps every warp has a
    // sub-partition to itself) run at the latency of the slowest warp's chain of FIRE iterations: give each warp 16
    // pixels instead of 32 (lanes 16-31 idle).  A warp then waits for the slowest of 16 pixels instead of 32 and
    // re-gathers (a warp-wide trip whenever ANY lane leaves its cell) about half as often: config 0 0.506 -> 0.473 ms.
    // Beyond that size the doubled instruction count costs more than it saves (config 1, 704 warps: 0.745 -> 1.00 ms).
    if (blocks * (RX_THREADS / 32) <= RX_SPARSE_MAX_WARPS) {
        blocks = 0;
        for (int m = 0; m < nsys; m++) {
            RelaxJob &j = hj[m];
            j.sparse = 1;
            j.block_begin = (int)blocks;
            j.nbx = (scans[m].npx + RX_TILE_X / 2 - 1) / (RX_TILE_X / 2);
            blocks += (long long)j.nbx * ((scans[m].npy + RX_TILE_Y - 1) / RX_TILE_Y);
        }
    }
    *hj_out = hj;
    *blocks_out = blocks;
    *samples_out = out_off;
    *ortho_out = ortho; *anyper_out = anyper; *symtip_out = symtip;
    return PPFM_OK;
}

static int relax_impl(int nsys, const float *d_ff, const ppfm_grid *grids, const ppfm_tip *tips,
                      const ppfm_fire *fire, const ppfm_scan *scans, float *d_pos_fz, uint16_t *d_iters,
                      ppfm_stats *d_stats, void *cuda_stream, bool tricubic = false, float *d_fz = nullptr,
                      float *d_eig = nullptr, bool shared_grid = false) {
    if (nsys < 1 || !d_ff || !grids || !tips || !fire || !scans || !d_pos_fz) return PPFM_EINVAL;
    if (d_eig && (tricubic || ((uintptr_t)d_eig & 15))) return PPFM_EINVAL;
    if (((uintptr_t)d_ff & (tricubic ? 3 : 15)) || ((uintptr_t)d_pos_fz & 15) || ((uintptr_t)d_iters & 1) || ((uintptr_t)d_stats & 7))
        return PPFM_EINVAL;
    if (!(fire->dt > 0) || !(fire->dt_max > 0) || !(fire->finc >= 1.0) || !(fire->fdec > 0 && fire->fdec < 1.0) ||
        !(fire->alpha0 >= 0 && fire->alpha0 <= 1.0) || !(fire->falpha > 0 && fire->falpha <= 1.0) ||
        fire->n_min < 0 || fire->max_iter < 0 || fire->max_iter > 0xFFFE || !(fire->f_conv > 0))
        return PPFM_EINVAL;
    RelaxJob *hj = nullptr;
    long long blocks = 0, samples = 0;
    bool ortho = true, anyper = false, symtip = true;
    {
        const int rc = build_relax_jobs(nsys, grids, tips, scans, &hj, &blocks, &samples, &ortho, &anyper, &symtip,
                                        shared_grid);
        if (rc != PPFM_OK) return rc;
    }
    FireParams fp;
    fp.dt0 = (float)fire->dt; fp.dt_max = (float)fire->dt_max; fp.finc = (float)fire->finc;
    fp.fdec = (float)fire->fdec; fp.alpha0 = (float)fire->alpha0; fp.falpha = (float)fire->falpha;
    fp.fconv2 = (float)(fire->f_conv * fire->f_conv);
    fp.n_min = fire->n_min; fp.max_iter = fire->max_iter;

    cudaStream_t st = (cudaStream_t)cuda_stream;
    RelaxJob *dj = nullptr;
    cudaError_t e;
    if (nsys > 1) {
        e = scratch_alloc((void **)&dj, (size_t)nsys * sizeof(RelaxJob), st);
        if (e != cudaSuccess) { free(hj); set_cuda_error(e, "scratch_alloc"); return PPFM_ENOMEM; }
        e = cudaMemcpyAsync(dj, hj, (size_t)nsys * sizeof(RelaxJob), cudaMemcpyHostToDevice, st);   // pageable: staged
        if (e != cudaSuccess) { free(hj); set_cuda_error(e, "job upload"); cudaFreeAsync(dj, st); return PPFM_ECUDA; }
    }
    float4 *pos4 = reinterpret_cast<float4 *>(d_pos_fz);
    {
        KernelTimer kt(tricubic ? PPFM_K_RELAX_TRICUBIC : PPFM_K_RELAX, st);
    float4 *eig4 = reinterpret_cast<float4 *>(d_eig);
#define PPFM_RX(O, A, S) \
    do { \
        if (tricubic) launch_relax<O, A, S, true, false>(nsys, blocks, st, hj, dj, fp, d_ff, pos4, d_iters, d_stats, d_fz, nullptr); \
        else if (eig4) launch_relax<O, A, S, false, true>(nsys, blocks, st, hj, dj, fp, d_ff, pos4, d_iters, d_stats, d_fz, eig4); \
        else launch_relax<O, A, S, false, false>(nsys, blocks, st, hj, dj, fp, d_ff, pos4, d_iters, d_stats, d_fz, nullptr); \
    } while (0)
        if (symtip) {
            if (ortho && !anyper) PPFM_RX(true, false, true);
            else if (ortho) PPFM_RX(true, true, true);
            else if (!anyper) PPFM_RX(false, false, true);
            else PPFM_RX(false, true, true);
        } else {
            if (ortho && !anyper) PPFM_RX(true, false, false);
            else if (ortho) PPFM_RX(true, true, false);
            else if (!anyper) PPFM_RX(false, false, false);
            else PPFM_RX(false, true, false);
        }
#undef PPFM_RX
    }
    free(hj);
    e = cudaGetLastError();
    if (e != cudaSuccess) { set_cuda_error(e, "relax_kernel"); if (dj) cudaFreeAsync(dj, st); return PPFM_ECUDA; }
    count_launch();
    if (dj) PPFM_CUDA(cudaFreeAsync(dj, st));
    return PPFM_OK;
}

// ---------------------------------------------------------------------------------------------------- stiffness map
// SURVEY.md 8(f) N2, PAPER.md:202-216 (IETS module): "the change of the stiffness of lateral vibration modes" of the
// probe particle caused by the curvature of the tip-sample potential.  At every relaxed point the total Hessian of
// the PP's potential is H = H_spring - (J + J^T)/2, with J = dF_S/dr the analytic Jacobian of the tri-linear
// interpolant inside the current cell (reading S14: the interpolant is not a gradient field, so J is symmetrised)
// and H_spring the second derivative of the tip springs of Eq.2.  Output: the three eigenvalues, ascending.
//
// One thread per (pixel, z-step) sample, x fastest so that reads, gathers and the float4 store are coalesced.  Cell
// lookup and the spring Hessian are FP64 (once per sample); the Jacobian is formed in FP32 from the FP32 grid; the
// eigenvalues come from the FP32 deflation solver above (the eigenvalues of interest, ~k_xy = 0.016 eV/A^2, sit next to
// one of ~k_R = 1.9: a route through all three roots of the characteristic cubic would need FP64 trigonometry).
struct StiffCell {
    int i0, i1;
    float f;
};

__device__ __forceinline__ StiffCell stiff_axis(double t, int n, int periodic) {
    StiffCell c;
    if (periodic) {
        const double fl = floor(t);
        long long m = (long long)fl % n;
        if (m < 0) m += n;
        c.i0 = (int)m;
        c.i1 = (c.i0 + 1 == n) ? 0 : c.i0 + 1;
        c.f = (float)(t - fl);
    } else {
        const double tc = fmin(fmax(t, 0.0), (double)(n - 1));          // S12: clamp the coordinate
        int i = (int)floor(tc);
        if (i > n - 2) i = n - 2;
        c.i0 = i;
        c.i1 = i + 1;
        c.f = (float)(tc - (double)i);
    }
    return c;
}

__global__ void __launch_bounds__(256)
stiffness_kernel(const RelaxJob *__restrict__ jobs, int njobs, long long nsamples, const float4 *__restrict__ ff,
                 const float4 *__restrict__ pos_fz, float4 *__restrict__ eig) {
    const long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= nsamples) return;
    int lo = 0, hi = njobs - 1;
    while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (jobs[mid].out_offset <= s) lo = mid; else hi = mid - 1;
    }
    const RelaxJob &job = jobs[lo];
    const long long ls = s - job.out_offset;
    const int npix = job.npx * job.npy;
    const int iz = (int)(ls / npix);
    const int pix = (int)(ls - (long long)iz * npix);
    const int iy = pix / job.npx, ix = pix - iy * job.npx;

    const float4 pp = pos_fz[s];
    const double r[3] = {(double)pp.x, (double)pp.y, (double)pp.z};
    double d[3], t[3];
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const double rtip = job.p0[c] + ix * job.dx[c] + iy * job.dy[c] - (c == 2 ? iz * job.dz : 0.0);
        d[c] = r[c] - rtip;
    }
#pragma unroll
    for (int a = 0; a < 3; a++)
        t[a] = job.Minv[3 * a] * (r[0] - job.origin[0]) + job.Minv[3 * a + 1] * (r[1] - job.origin[1]) +
               job.Minv[3 * a + 2] * (r[2] - job.origin[2]);
    const StiffCell cx = stiff_axis(t[0], job.n[0], job.periodic[0]);
    const StiffCell cy = stiff_axis(t[1], job.n[1], job.periodic[1]);
    const StiffCell cz = stiff_axis(t[2], job.n[2], job.periodic[2]);
    const float4 *g = ff + job.ff_offset;
    const long long nx = job.n[0], nxy = (long long)job.n[0] * job.n[1];
    const float4 *r00 = g + cz.i0 * nxy + cy.i0 * nx, *r01 = g + cz.i0 * nxy + cy.i1 * nx;
    const float4 *r10 = g + cz.i1 * nxy + cy.i0 * nx, *r11 = g + cz.i1 * nxy + cy.i1 * nx;
    PPFM_CHK(PPFM_CHK_RELAX_GATHER, cx.i0 >= 0 && cx.i0 < job.n[0] && cx.i1 >= 0 && cx.i1 < job.n[0] && cy.i0 >= 0 &&
                                        cy.i0 < job.n[1] && cy.i1 >= 0 && cy.i1 < job.n[1] && cz.i0 >= 0 && cz.i0 < job.n[2] &&
                                        cz.i1 >= 0 && cz.i1 < job.n[2]);
    const float4 c000 = __ldg(r00 + cx.i0), c001 = __ldg(r00 + cx.i1), c010 = __ldg(r01 + cx.i0), c011 = __ldg(r01 + cx.i1);
    const float4 c100 = __ldg(r10 + cx.i0), c101 = __ldg(r10 + cx.i1), c110 = __ldg(r11 + cx.i0), c111 = __ldg(r11 + cx.i1);
    // G[c][a] = dF_c/dt_a inside the cell (FP32): difference along axis a, tri-linear weights on the other two
    const float fx = cx.f, fy = cy.f, fz = cz.f, gx = 1.0f - fx, gy = 1.0f - fy, gz = 1.0f - fz;
    float G[3][3];
#define PPFM_G(C)                                                                                                  \
    {                                                                                                              \
        const float v000 = c000.C, v001 = c001.C, v010 = c010.C, v011 = c011.C;                                    \
        const float v100 = c100.C, v101 = c101.C, v110 = c110.C, v111 = c111.C;                                    \
        row[0] = gz * (gy * (v001 - v000) + fy * (v011 - v010)) + fz * (gy * (v101 - v100) + fy * (v111 - v110));   \
        row[1] = gz * (gx * (v010 - v000) + fx * (v011 - v001)) + fz * (gx * (v110 - v100) + fx * (v111 - v101));   \
        row[2] = gy * (gx * (v100 - v000) + fx * (v101 - v001)) + fy * (gx * (v110 - v010) + fx * (v111 - v011));   \
    }
    { float *row = G[0]; PPFM_G(x) }
    { float *row = G[1]; PPFM_G(y) }
    { float *row = G[2]; PPFM_G(z) }
#undef PPFM_G
    // J = G Minv (chain rule through t = Minv (r - origin))
    double J[3][3];
#pragma unroll
    for (int c = 0; c < 3; c++)
#pragma unroll
        for (int a = 0; a < 3; a++)
            J[c][a] = (double)(G[c][0] * job.Minvf[a] + G[c][1] * job.Minvf[3 + a] + G[c][2] * job.Minvf[6 + a]);
    // H_spring = k_R dd^T/|d|^2 + k_R (|d| - R0)/|d| (I - dd^T/|d|^2) + diag(k_x, k_y, 0)
    const double L2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
    const double L = sqrt(L2);
    const double kR = (double)job.k_rad;
    const double R0 = sqrt(job.d0[0] * job.d0[0] + job.d0[1] * job.d0[1] + job.d0[2] * job.d0[2]);
    const double kt = (L > 0.0) ? kR * (L - R0) / L : 0.0;                // transverse stiffness of the radial spring
    const double iL2 = (L2 > 0.0) ? 1.0 / L2 : 0.0;
    double H[3][3];
#pragma unroll
    for (int a = 0; a < 3; a++)
#pragma unroll
        for (int b = 0; b < 3; b++) {
            const double dd = d[a] * d[b] * iL2;
            H[a][b] = kR * dd + kt * ((a == b ? 1.0 : 0.0) - dd) - 0.5 * (J[a][b] + J[b][a]);
        }
    H[0][0] += (double)job.k_lat[0];
    H[1][1] += (double)job.k_lat[1];
    float e0, e1, e2;
    sym3_eigenvalues_f32((float)H[0][0], (float)H[1][1], (float)H[2][2], (float)H[0][1], (float)H[0][2], (float)H[1][2],
                         e0, e1, e2);
    eig[s] = make_float4(e0, e1, e2, 0.0f);
}

static int stiffness_impl(int nsys, const float *d_ff, const ppfm_grid *grids, const ppfm_tip *tips,
                          const ppfm_scan *scans, const float *d_pos_fz, float *d_eig, void *cuda_stream) {
    if (nsys < 1 || !d_ff || !grids || !tips || !scans || !d_pos_fz || !d_eig) return PPFM_EINVAL;
    if (((uintptr_t)d_ff & 15) || ((uintptr_t)d_pos_fz & 15) || ((uintptr_t)d_eig & 15)) return PPFM_EINVAL;
    RelaxJob *hj = nullptr;
    long long blocks = 0, samples = 0;
    bool ortho, anyper, symtip;
    const int rc = build_relax_jobs(nsys, grids, tips, scans, &hj, &blocks, &samples, &ortho, &anyper, &symtip);
    if (rc != PPFM_OK) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    RelaxJob *dj = nullptr;
    cudaError_t e = scratch_alloc((void **)&dj, (size_t)nsys * sizeof(RelaxJob), st);
    if (e != cudaSuccess) { free(hj); set_cuda_error(e, "scratch_alloc"); return PPFM_ENOMEM; }
    e = cudaMemcpyAsync(dj, hj, (size_t)nsys * sizeof(RelaxJob), cudaMemcpyHostToDevice, st);   // pageable: staged
    free(hj);
    if (e != cudaSuccess) { set_cuda_error(e, "job upload"); cudaFreeAsync(dj, st); return PPFM_ECUDA; }
    const long long nblk = (samples + 255) / 256;
    if (nblk > 0x7fffffffLL) { cudaFreeAsync(dj, st); return PPFM_EINVAL; }
    {
        KernelTimer kt(PPFM_K_STIFFNESS, st);
        stiffness_kernel<<<(unsigned)nblk, 256, 0, st>>>(dj, nsys, samples, reinterpret_cast<const float4 *>(d_ff),
                                                         reinterpret_cast<const float4 *>(d_pos_fz),
                                                         reinterpret_cast<float4 *>(d_eig));
    }
    e = cudaGetLastError();
    if (e != cudaSuccess) { set_cuda_error(e, "stiffness_kernel"); cudaFreeAsync(dj, st); return PPFM_ECUDA; }
    count_launch();
    PPFM_CUDA(cudaFreeAsync(dj, st));
    return PPFM_OK;
}

int relax_scan_fz(int nsys, const float *d_ff, const ppfm_grid *grids, const ppfm_tip *tips, const ppfm_fire *fire,
                  const ppfm_scan *scans, float *d_pos_fz, uint16_t *d_iters, ppfm_stats *d_stats, float *d_fz,
                  void *cuda_stream) {
    return relax_impl(nsys, d_ff, grids, tips, fire, scans, d_pos_fz, d_iters, d_stats, cuda_stream, false, d_fz);
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

// Parameter sweep on ONE resident grid ("so the tip ... can change without
// recomputation"): nscan scans with their own tip (k_x, k_y, k_R, d0) and scan geometry in one launch, all gathering
// from the same grid.  The batch kernel is used as is; every job's grid offset is 0.
extern "C" int ppfm_relax_scan_sweep(int32_t nscan, const float *d_ff, const ppfm_grid *grid, const ppfm_tip *tips,
                                     const ppfm_fire *fire, const ppfm_scan *scans, float *d_pos_fz,
                                     uint16_t *d_iters, ppfm_stats *d_stats, void *cuda_stream) {
    return relax_impl(nscan, d_ff, grid, tips, fire, scans, d_pos_fz, d_iters, d_stats, cuda_stream, false, nullptr,
                      nullptr, true);
}

// relaxation with the stiffness map folded into the end of every z-step: the eigenvalues come
// from the cell the lane already holds in registers, so the map costs no second gather and no second launch
extern "C" int ppfm_relax_scan_stiffness(const float *d_ff, const ppfm_grid *grid, const ppfm_tip *tip,
                                         const ppfm_fire *fire, const ppfm_scan *scan, float *d_pos_fz,
                                         uint16_t *d_iters, float *d_eig, ppfm_stats *d_stats, void *cuda_stream) {
    if (!d_eig) return PPFM_EINVAL;
    return relax_impl(1, d_ff, grid, tip, fire, scan, d_pos_fz, d_iters, d_stats, cuda_stream, false, nullptr, d_eig);
}

extern "C" int ppfm_relax_scan_stiffness_batch(int32_t nsys, const float *d_ff, const ppfm_grid *grids,
                                               const ppfm_tip *tips, const ppfm_fire *fire, const ppfm_scan *scans,
                                               float *d_pos_fz, uint16_t *d_iters, float *d_eig, ppfm_stats *d_stats,
                                               void *cuda_stream) {
    if (!d_eig) return PPFM_EINVAL;
    return relax_impl(nsys, d_ff, grids, tips, fire, scans, d_pos_fz, d_iters, d_stats, cuda_stream, false, nullptr,
                      d_eig);
}

extern "C" int ppfm_stiffness(const float *d_ff, const ppfm_grid *grid, const ppfm_tip *tip, const ppfm_scan *scan,
                              const float *d_pos_fz, float *d_eig, void *cuda_stream) {
    return stiffness_impl(1, d_ff, grid, tip, scan, d_pos_fz, d_eig, cuda_stream);
}

extern "C" int ppfm_stiffness_batch(int32_t nsys, const float *d_ff, const ppfm_grid *grids, const ppfm_tip *tips,
                                    const ppfm_scan *scans, const float *d_pos_fz, float *d_eig, void *cuda_stream) {
    return stiffness_impl(nsys, d_ff, grids, tips, scans, d_pos_fz, d_eig, cuda_stream);
}

// ---- relaxation on an energy-only grid with tri-cubic interpolation of the potential
extern "C" int ppfm_relax_scan_tricubic(const float *d_E, const ppfm_grid *grid, const ppfm_tip *tip,
                                        const ppfm_fire *fire, const ppfm_scan *scan, float *d_pos_fz,
                                        uint16_t *d_iters, ppfm_stats *d_stats, void *cuda_stream) {
    return relax_impl(1, d_E, grid, tip, fire, scan, d_pos_fz, d_iters, d_stats, cuda_stream, true);
}

extern "C" int ppfm_relax_scan_tricubic_batch(int32_t nsys, const float *d_E, const ppfm_grid *grids,
                                              const ppfm_tip *tips, const ppfm_fire *fire, const ppfm_scan *scans,
                                              float *d_pos_fz, uint16_t *d_iters, ppfm_stats *d_stats,
                                              void *cuda_stream) {
    return relax_impl(nsys, d_E, grids, tips, fire, scans, d_pos_fz, d_iters, d_stats, cuda_stream, true);
}

namespace ppfm {
__global__ void energy_grid_kernel(const float4 *__restrict__ ff, long long n, float *__restrict__ E) {
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) E[i] = ff[i].w;
}
}  // namespace ppfm

extern "C" int ppfm_energy_grid(const float *d_ff, int64_t n_points, float *d_E, void *cuda_stream) {
    if (!d_ff || !d_E || n_points < 0 || ((uintptr_t)d_ff & 15) || ((uintptr_t)d_E & 3)) return PPFM_EINVAL;
    if (n_points == 0) return PPFM_OK;
    long long blocks = (n_points + 255) / 256;
    if (blocks > 148LL * 16) blocks = 148LL * 16;
    energy_grid_kernel<<<(unsigned)blocks, 256, 0, (cudaStream_t)cuda_stream>>>(
        reinterpret_cast<const float4 *>(d_ff), n_points, d_E);
    PPFM_LAUNCH_CHECK();
    return PPFM_OK;
}
