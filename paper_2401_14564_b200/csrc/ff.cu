// ff.cu — force-field grid sampling: Lennard-Jones (Eq.5, mixing
// rules PAPER.md:85) plus point-charge Coulomb (Eq.6) summed over all sample atoms and their periodic
// images at every point of a uniform grid, forces as F = -grad E.
//
// Kernel design (B200 / sm_100a; nothing here is a dense contraction, so no tensor cores):
//   * a1  `ff_prep_kernel` (one CTA per system) packs one 48-byte record per atom (x, y, z, - | c12, c12, -c6, -c6 |
//         6 c6, 6 c6, kq, kq: the pair coefficients twice, so that LDS.128 yields aligned FP32x2 operand pairs) and
//         stable-partitions the records: atoms with a Coulomb factor first, LJ-only atoms behind them.
//   * a2  `ff_kernel`: one CTA = 128 columns (FF_THREADS) (consecutive x-fastest (i,j) indices, so a warp's float4 stores are
//         512 contiguous bytes) x P consecutive z planes held in registers as P/2 FP32x2 pairs.  Atom records stream
//         through a 3-stage shared-memory ring filled by 1-D TMA bulk copies (cp.async.bulk + mbarrier complete_tx),
//         one elected thread producing two chunks ahead; every warp reads records as uniform (broadcast) LDS.128.
//         Images are the outer loop and are applied as a shift of the grid point; the shifted point is formed in
//         FP64 once per image and split hi+lo so that dx = (p_hi - a) + p_lo carries no coordinate rounding.
//         The inner loop is sm_100's packed FP32x2 arithmetic (FFMA2 / FMUL2 / FADD2): per pair of grid points and
//         atom 15 packed instructions + 2 MUFU.RSQ (13 + 2 for an LJ-only atom; +2 FMNMX when the r_min clamp is
//         live, which the prep kernel decides from the atoms' distance to the grid's bounding box).
//   * a3  `combine_kernel`: F = F_LJ + Q F_el, float4 streaming.
#include "common.cuh"

#include <type_traits>

namespace ppfm {

#ifndef PPFM_FF_THREADS
#define PPFM_FF_THREADS 128
#endif
constexpr int FF_THREADS = PPFM_FF_THREADS;  // columns per CTA
constexpr int FF_CHUNK = 256;   // atoms per pipeline stage
constexpr int FF_STAGES = 3;
constexpr int FF_AHEAD = 2;     // chunks in flight ahead of the consumer

// 48-byte record.  The pair coefficients are stored twice so that one LDS.128 yields the aligned 64-bit register
// pairs the packed FP32x2 instructions (FFMA2 / FMUL2 / FADD2, new on sm_100) take as operands, with no MOVs.
struct __align__(16) AtomRec {
    float x, y, z, pad;
    float c12[2], nc6[2];       // c12 = E0 R0^12, nc6 = -2 E0 R0^6
    float c6x6[2], kq[2];       // 6 c6;  kq = k_e q_PP q_i (eV*Angstrom), or k_e q_i (unit probe charge) in split mode
};
static_assert(sizeof(AtomRec) == 48, "AtomRec must be 48 bytes");

struct FFJob {
    long long tile_begin;   // first tile (CTA) of this system in the launch
    long long out_offset;   // float4 offset of this system's grid in the output buffer(s)
    int atom_begin, natoms;
    int nx, ny, nz, nxy;
    int n_xy_tiles, n_z_groups;
    int nimg[3];
    int table_offset;       // first entry of this system's per-type table
    double origin[3], step[3][3], cell[3][3];
    double bb_lo[3], bb_hi[3];   // Cartesian bounding box of the grid points
    float keQ;              // k_e q_PP
    float rmin2;
    int ntypes;
    int split;              // records carry the unit-charge Coulomb factor
};

struct TypeEntry {
    float c6, c12;
};

#define PPFM_CHK_READER ff_checks_read
PPFM_CHK_STORAGE
#undef PPFM_CHK_READER
#ifndef PPFM_CHECKS
void ff_checks_read(unsigned long long *) {}
#endif

// ---------------------------------------------------------------------------------------------------- a1 prep
struct FFSingle {               // one system: job and per-type table travel as a kernel parameter (constant bank)
    FFJob job;
    TypeEntry table[PPFM_MAX_TYPES];
};

// Per-system flags written by the prep kernel and read by every tile of that system.
struct FFFlags {
    int clamp;      // some atom image lies within r_min of the grid's bounding box: the tile applies the S3 clamp
    int ncharged;   // records [0, ncharged) carry a Coulomb factor != 0; the rest are LJ-only (e.g. a neutral slab)
};
constexpr int PREP_THREADS = 256;

__device__ __forceinline__ AtomRec make_record(const FFJob &job, const TypeEntry *__restrict__ table, float4 a, int t) {
    AtomRec r;
    r.x = a.x; r.y = a.y; r.z = a.z;
    r.pad = 0.0f;
    if (t >= 0 && t < job.ntypes) {
        const TypeEntry te = table[job.table_offset + t];
        r.c12[0] = r.c12[1] = te.c12;
        r.nc6[0] = r.nc6[1] = -te.c6;
        r.c6x6[0] = r.c6x6[1] = 6.0f * te.c6;
        r.kq[0] = r.kq[1] = job.split ? (float)(kCoulomb * (double)a.w) : (float)((double)job.keQ * (double)a.w);
    } else {   // out-of-range type index: the atom contributes nothing
        r.c12[0] = r.c12[1] = r.nc6[0] = r.nc6[1] = r.c6x6[0] = r.c6x6[1] = r.kq[0] = r.kq[1] = 0.0f;
    }
    return r;
}

// r_min clamp needed?  distance of every image of this atom to the grid's bounding box
__device__ __forceinline__ bool atom_near_grid(const FFJob &job, float4 a) {
    const double rmin = sqrt((double)job.rmin2) * 1.0001 + 1e-6;
    bool near = false;
    for (int ia = -job.nimg[0]; ia <= job.nimg[0]; ia++)
        for (int ib = -job.nimg[1]; ib <= job.nimg[1]; ib++)
            for (int ic = -job.nimg[2]; ic <= job.nimg[2]; ic++) {
                double d2 = 0.0;
                const double p[3] = {a.x, a.y, a.z};
                for (int c = 0; c < 3; c++) {
                    const double x = p[c] + ia * job.cell[0][c] + ib * job.cell[1][c] + ic * job.cell[2][c];
                    const double d = fmax(fmax(job.bb_lo[c] - x, x - job.bb_hi[c]), 0.0);
                    d2 += d * d;
                }
                near |= (d2 < rmin * rmin);
            }
    return near;
}

// One CTA per system.  Packs the records and stable-partitions them (block scan, so the order and therefore the
// summation order is fixed): atoms with a Coulomb factor first, LJ-only atoms after them.
__device__ __forceinline__ void prep_system(const FFJob &job, const TypeEntry *__restrict__ table, int job_index,
                                            const float4 *__restrict__ xyzq, const int *__restrict__ type,
                                            AtomRec *__restrict__ recs, FFFlags *__restrict__ flags,
                                            ppfm_ff_status *__restrict__ status) {
    __shared__ int s_warp[PREP_THREADS / 32];
    __shared__ int s_total, s_near, s_bad;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int n = job.natoms;
    // pass 1: number of charged atoms
    int cnt = 0, bad = 0;
    for (int i = tid; i < n; i += PREP_THREADS) {
        const int t = type[job.atom_begin + i];
        const AtomRec r = make_record(job, table, xyzq[job.atom_begin + i], t);
        cnt += (r.kq[0] != 0.0f) ? 1 : 0;
        bad += (t < 0 || t >= job.ntypes) ? 1 : 0;
    }
#pragma unroll
    for (int s = 16; s > 0; s >>= 1) {
        cnt += __shfl_xor_sync(0xffffffffu, cnt, s);
        bad += __shfl_xor_sync(0xffffffffu, bad, s);
    }
    if (tid == 0) { s_total = 0; s_near = 0; s_bad = 0; }
    __syncthreads();
    if (lane == 0 && cnt) atomicAdd(&s_total, cnt);      // integer sums: order does not matter
    if (lane == 0 && bad) atomicAdd(&s_bad, bad);
    __syncthreads();
    const int nq = s_total;
    // pass 2: stable partition, PREP_THREADS atoms at a time
    int run_q = 0;
    bool near = false;
    for (int base = 0; base < n; base += PREP_THREADS) {
        const int i = base + tid;
        const bool live = i < n;
        AtomRec r;
        bool charged = false;
        if (live) {
            const float4 a = xyzq[job.atom_begin + i];
            r = make_record(job, table, a, type[job.atom_begin + i]);
            charged = r.kq[0] != 0.0f;
            near |= atom_near_grid(job, a);
        }
        const unsigned ballot = __ballot_sync(0xffffffffu, charged);
        const int in_warp = __popc(ballot & ((1u << lane) - 1u));
        __syncthreads();                                   // s_warp reuse
        if (lane == 0) s_warp[wid] = __popc(ballot);
        __syncthreads();
        int before = 0, chunk_total = 0;
#pragma unroll
        for (int w = 0; w < PREP_THREADS / 32; w++) {
            const int c = s_warp[w];
            before += (w < wid) ? c : 0;
            chunk_total += c;
        }
        if (live) {
            const int q_before = run_q + before + in_warp;             // charged atoms ahead of atom i
            const int pos = charged ? q_before : nq + (i - q_before);
            PPFM_CHK(PPFM_CHK_FF_STORE, pos >= 0 && pos < n);
            recs[job.atom_begin + pos] = r;
        }
        run_q += chunk_total;
    }
    if (near) atomicOr(&s_near, 1);
    __syncthreads();
    if (tid == 0) {
        flags[job_index].clamp = s_near; flags[job_index].ncharged = nq;
        if (status) {                                   // zeroed by the host on the same stream before this launch
            if (s_bad) atomicAdd(&status->n_bad_type, (unsigned)s_bad);
            if (s_near) atomicAdd(&status->n_clamped, 1u);
        }
    }
}

__global__ void __launch_bounds__(PREP_THREADS)
ff_prep_kernel(const __grid_constant__ FFSingle one, const float4 *__restrict__ xyzq, const int *__restrict__ type,
               AtomRec *__restrict__ recs, FFFlags *__restrict__ flags, ppfm_ff_status *__restrict__ status) {
    prep_system(one.job, one.table, 0, xyzq, type, recs, flags, status);
}

__global__ void __launch_bounds__(PREP_THREADS)
ff_prep_batch_kernel(const FFJob *__restrict__ jobs, const TypeEntry *__restrict__ table,
                     const float4 *__restrict__ xyzq, const int *__restrict__ type, AtomRec *__restrict__ recs,
                     FFFlags *__restrict__ flags, ppfm_ff_status *__restrict__ status) {
    prep_system(jobs[blockIdx.x], table, blockIdx.x, xyzq, type, recs, flags, status);
}

// ---------------------------------------------------------------------------------------------------- PTX helpers
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra DONE;\n"
        "bra LAB_WAIT;\n"
        "DONE:\n"
        "}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// 1-D TMA bulk copy global -> shared, completion counted in bytes on an mbarrier (SASS: UBLKCP).
__device__ __forceinline__ void tma_load_1d(void *dst, const void *src, uint32_t bytes, uint64_t *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ float rsqrt_approx(float x) {
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// ---------------------------------------------------------------------------------------------------- a2 tile body
// P      grid points per thread along step[2]
// SPLIT  false: one grid (LJ + Coulomb with q_PP);  true: two grids (LJ | Coulomb of a unit probe charge)
// CLAMP  apply s = max(r^2, r_min^2)
// ZCOL   step[2] is parallel to z (dx, dy shared by the P points of a column)
template <int P, bool SPLIT, bool CLAMP, bool ZCOL>
__device__ __forceinline__ void ff_tile(const FFJob &job, int ncharged, const AtomRec *__restrict__ recs,
                                        float4 *__restrict__ out_a,
                                        float4 *__restrict__ out_b, AtomRec *s_rec, uint64_t *full_bar,
                                        uint64_t *empty_bar, long long local_tile) {
    const int tid = threadIdx.x;
    const int zg = (int)(local_tile / job.n_xy_tiles);
    const int xyt = (int)(local_tile - (long long)zg * job.n_xy_tiles);
    const int col = xyt * FF_THREADS + tid;
    const bool valid = col < job.nxy;
    const int colc = valid ? col : job.nxy - 1;
    const int j = colc / job.nx, i = colc - j * job.nx;
    const int k0 = zg * P;

    // base point of the column, FP64
    double pb[3];
#pragma unroll
    for (int c = 0; c < 3; c++)
        pb[c] = job.origin[c] + i * job.step[0][c] + j * job.step[1][c] + k0 * job.step[2][c];
    // P points along step[2], held as P/2 packed pairs (lo = point 2h, hi = point 2h + 1)
    constexpr int H = P / 2;
    static_assert(P % 2 == 0, "P must be even: points are processed as FP32x2 pairs");
    float2 off[ZCOL ? 1 : 3][H];   // offsets of the points along step[2]
#pragma unroll
    for (int h = 0; h < H; h++) {
#pragma unroll
        for (int c = 0; c < (ZCOL ? 1 : 3); c++) {
            const int cc = ZCOL ? 2 : c;
            off[c][h] = make_float2((float)((2 * h) * job.step[2][cc]), (float)((2 * h + 1) * job.step[2][cc]));
        }
    }

    float2 Fx[H], Fy[H], Fz[H], E[H];
    float2 Gx[SPLIT ? H : 1], Gy[SPLIT ? H : 1], Gz[SPLIT ? H : 1], Ge[SPLIT ? H : 1];
    // energies are accumulated per chunk and folded into a running total at every chunk boundary: the 1/r and
    // 1/r^6 tails of tens of thousands of atom images otherwise lose ~1e-5 eV to FP32 accumulation rounding
    float2 Etot[H], Getot[SPLIT ? H : 1];
    const float2 zero2 = make_float2(0.0f, 0.0f);
#pragma unroll
    for (int h = 0; h < H; h++) {
        Fx[h] = Fy[h] = Fz[h] = E[h] = Etot[h] = zero2;
        if (SPLIT) Gx[h] = Gy[h] = Gz[h] = Ge[h] = Getot[h] = zero2;
    }

    // chunks [0, nch_q) hold atoms with a Coulomb factor, chunks [nch_q, nchunks) the LJ-only atoms behind them
    const int natoms = job.natoms;
    const int nq = min(max(ncharged, 0), natoms);
    const int nch_q = (nq + FF_CHUNK - 1) / FF_CHUNK;
    const int nchunks = nch_q + (natoms - nq + FF_CHUNK - 1) / FF_CHUNK;
    auto chunk_begin = [&](int c) { return c < nch_q ? c * FF_CHUNK : nq + (c - nch_q) * FF_CHUNK; };
    auto chunk_count = [&](int c) {
        return c < nch_q ? min(FF_CHUNK, nq - c * FF_CHUNK) : min(FF_CHUNK, natoms - nq - (c - nch_q) * FF_CHUNK);
    };
    const int nimages = (2 * job.nimg[0] + 1) * (2 * job.nimg[1] + 1) * (2 * job.nimg[2] + 1);
    const int nsteps = nimages * nchunks;
    const AtomRec *src = recs + job.atom_begin;
    const float rmin2 = job.rmin2;

    auto issue = [&](int t) {   // producer: fill stage t % STAGES with chunk t % nchunks
        const int st = t % FF_STAGES;
        const int use = t / FF_STAGES;
        if (use > 0) mbar_wait(&empty_bar[st], (use - 1) & 1);
        const int c = t % nchunks;
        const uint32_t bytes = (uint32_t)chunk_count(c) * (uint32_t)sizeof(AtomRec);
        mbar_expect_tx(&full_bar[st], bytes);
        tma_load_1d(s_rec + st * FF_CHUNK, src + chunk_begin(c), bytes, &full_bar[st]);
    };
    if (tid == 0) {
        for (int t = 0; t < FF_AHEAD && t < nsteps; t++) issue(t);
    }

    // shifted point p' = p - image shift, split hi + lo; set once per image
    float ph[3], pl[3];
    const float2 twelve = make_float2(12.0f, 12.0f);

    // The pair body is written in two stages so that the MUFU of atom a + 1 is in flight while the polynomial of
    // atom a runs (software pipelining), and every stage loops over the H point pairs of the column, which gives
    // ptxas H independent dependency chains side by side instead of one chain after the other (ncu, round 1: the
    // serial schedule left the FMA pipe 79 % busy with `wait` and `short_scoreboard` stalls on every link).
    //   stage A (atom record -> displacement, r^2, 1/r):   per pair of points 1 FADD2 + 1 FFMA2 + 2 MUFU.RSQ
    //   stage B (1/r -> energy and force accumulation):    13 packed instructions (11 for an LJ-only atom)
    struct Stage {
        float2 dx[ZCOL ? 1 : H], dy[ZCOL ? 1 : H], dz[H], ir[H];
        float2 c12, nc6, c6x6, kq;
    };
    auto stage_a = [&](const float4 *s4, int a, Stage &S) {
        const float4 r0 = s4[3 * a];          // x, y, z, -
        const float4 r1 = s4[3 * a + 1];      // c12, c12, -c6, -c6
        const float4 r2_ = s4[3 * a + 2];     // 6 c6, 6 c6, kq, kq
        S.c12 = make_float2(r1.x, r1.y); S.nc6 = make_float2(r1.z, r1.w);
        S.c6x6 = make_float2(r2_.x, r2_.y); S.kq = make_float2(r2_.z, r2_.w);
        const float dx0 = (ph[0] - r0.x) + pl[0];
        const float dy0 = (ph[1] - r0.y) + pl[1];
        const float dz0 = (ph[2] - r0.z) + pl[2];
        const float2 dxx = make_float2(dx0, dx0), dyy = make_float2(dy0, dy0), dzz = make_float2(dz0, dz0);
        float2 r2[H];
        if (ZCOL) {
            const float rxy2s = fmaf(dy0, dy0, dx0 * dx0);
            const float2 rxy2 = make_float2(rxy2s, rxy2s);
            S.dx[0] = dxx; S.dy[0] = dyy;
#pragma unroll
            for (int h = 0; h < H; h++) S.dz[h] = __fadd2_rn(dzz, off[0][h]);
#pragma unroll
            for (int h = 0; h < H; h++) r2[h] = __ffma2_rn(S.dz[h], S.dz[h], rxy2);
        } else {
#pragma unroll
            for (int h = 0; h < H; h++) {
                S.dx[ZCOL ? 0 : h] = __fadd2_rn(dxx, off[0][h]);
                S.dy[ZCOL ? 0 : h] = __fadd2_rn(dyy, off[1 % (ZCOL ? 1 : 3)][h]);
                S.dz[h] = __fadd2_rn(dzz, off[2 % (ZCOL ? 1 : 3)][h]);
                r2[h] = __ffma2_rn(S.dz[h], S.dz[h], __ffma2_rn(S.dy[ZCOL ? 0 : h], S.dy[ZCOL ? 0 : h],
                                                                 __fmul2_rn(S.dx[ZCOL ? 0 : h], S.dx[ZCOL ? 0 : h])));
            }
        }
#pragma unroll
        for (int h = 0; h < H; h++) {
            if (CLAMP) { r2[h].x = fmaxf(r2[h].x, rmin2); r2[h].y = fmaxf(r2[h].y, rmin2); }
            S.ir[h].x = rsqrt_approx(r2[h].x);
            S.ir[h].y = rsqrt_approx(r2[h].y);
        }
    };
    auto stage_b = [&](const Stage &S, auto neutral_tag) {
        constexpr bool NEUTRAL = decltype(neutral_tag)::value;
        float2 ir2[H], ir6[H], t[H], g[H];
#pragma unroll
        for (int h = 0; h < H; h++) ir2[h] = __fmul2_rn(S.ir[h], S.ir[h]);
#pragma unroll
        for (int h = 0; h < H; h++) ir6[h] = __fmul2_rn(ir2[h], ir2[h]);
#pragma unroll
        for (int h = 0; h < H; h++) ir6[h] = __fmul2_rn(ir6[h], ir2[h]);
#pragma unroll
        for (int h = 0; h < H; h++) t[h] = __ffma2_rn(S.c12, ir6[h], S.nc6);            // c12/r^6 - c6
#pragma unroll
        for (int h = 0; h < H; h++) E[h] = __ffma2_rn(t[h], ir6[h], E[h]);              // E_LJ = c12/r^12 - c6/r^6
#pragma unroll
        for (int h = 0; h < H; h++) t[h] = __ffma2_rn(t[h], twelve, S.c6x6);            // 12 c12/r^6 - 6 c6
#pragma unroll
        for (int h = 0; h < H; h++) g[h] = __fmul2_rn(t[h], ir6[h]);
        if (!SPLIT) {
            if (!NEUTRAL) {
#pragma unroll
                for (int h = 0; h < H; h++) E[h] = __ffma2_rn(S.kq, S.ir[h], E[h]);     // E_C = kq / r
#pragma unroll
                for (int h = 0; h < H; h++) g[h] = __ffma2_rn(S.kq, S.ir[h], g[h]);
            }
#pragma unroll
            for (int h = 0; h < H; h++) g[h] = __fmul2_rn(g[h], ir2[h]);                // (12c12/r^12 - 6c6/r^6 + kq/r)/r^2
        } else {
#pragma unroll
            for (int h = 0; h < H; h++) g[h] = __fmul2_rn(g[h], ir2[h]);
        }
#pragma unroll
        for (int h = 0; h < H; h++) Fx[h] = __ffma2_rn(g[h], S.dx[ZCOL ? 0 : h], Fx[h]);
#pragma unroll
        for (int h = 0; h < H; h++) Fy[h] = __ffma2_rn(g[h], S.dy[ZCOL ? 0 : h], Fy[h]);
#pragma unroll
        for (int h = 0; h < H; h++) Fz[h] = __ffma2_rn(g[h], S.dz[h], Fz[h]);
        if (SPLIT && !NEUTRAL) {
            float2 ec[SPLIT ? H : 1];
#pragma unroll
            for (int h = 0; h < (SPLIT ? H : 0); h++) ec[h] = __fmul2_rn(S.kq, S.ir[h]);
#pragma unroll
            for (int h = 0; h < (SPLIT ? H : 0); h++) Ge[h] = __fadd2_rn(Ge[h], ec[h]);
#pragma unroll
            for (int h = 0; h < (SPLIT ? H : 0); h++) ec[h] = __fmul2_rn(ec[h], ir2[h]);
#pragma unroll
            for (int h = 0; h < (SPLIT ? H : 0); h++) Gx[h] = __ffma2_rn(ec[h], S.dx[ZCOL ? 0 : h], Gx[h]);
#pragma unroll
            for (int h = 0; h < (SPLIT ? H : 0); h++) Gy[h] = __ffma2_rn(ec[h], S.dy[ZCOL ? 0 : h], Gy[h]);
#pragma unroll
            for (int h = 0; h < (SPLIT ? H : 0); h++) Gz[h] = __ffma2_rn(ec[h], S.dz[h], Gz[h]);
        }
    };
    // one chunk of atom records against the thread's P points; NEUTRAL: the records carry no Coulomb factor
    auto run_chunk = [&](const float4 *s4, int n, auto neutral_tag) {
        Stage S0, S1;
        stage_a(s4, 0, S0);
        int a = 0;
#pragma unroll 1
        for (; a + 2 <= n; a += 2) {
            stage_a(s4, a + 1, S1);
            stage_b(S0, neutral_tag);
            stage_a(s4, min(a + 2, n - 1), S0);      // past the end: the last atom again, not used
            stage_b(S1, neutral_tag);
        }
        if (a < n) stage_b(S0, neutral_tag);
    };

    int step = 0;
    for (int ia = -job.nimg[0]; ia <= job.nimg[0]; ia++)
        for (int ib = -job.nimg[1]; ib <= job.nimg[1]; ib++)
            for (int ic = -job.nimg[2]; ic <= job.nimg[2]; ic++) {
                // shifted point p' = p - shift, split hi + lo (FP64 once per image)
#pragma unroll
                for (int c = 0; c < 3; c++) {
                    const double s = pb[c] - (ia * job.cell[0][c] + ib * job.cell[1][c] + ic * job.cell[2][c]);
                    ph[c] = (float)s;
                    pl[c] = (float)(s - (double)ph[c]);
                }
                for (int ch = 0; ch < nchunks; ch++, step++) {
                    if (tid == 0 && step + FF_AHEAD < nsteps) issue(step + FF_AHEAD);
                    const int st = step % FF_STAGES;
                    mbar_wait(&full_bar[st], (step / FF_STAGES) & 1);
                    const float4 *s4 = reinterpret_cast<const float4 *>(s_rec + st * FF_CHUNK);
                    const int n = chunk_count(ch);
#ifdef PPFM_CHECKS
                    auto ring_matches = [&]() {      // this thread's record of the stage against the global copy
                        const int a = tid % n;
                        const float4 *gsrc = reinterpret_cast<const float4 *>(src + chunk_begin(ch) + a);
                        bool same = true;
                        for (int q = 0; q < 3; q++) {
                            const float4 x = s4[3 * a + q], y = gsrc[q];
                            same = same && __float_as_uint(x.x) == __float_as_uint(y.x) && __float_as_uint(x.y) == __float_as_uint(y.y) &&
                                   __float_as_uint(x.z) == __float_as_uint(y.z) && __float_as_uint(x.w) == __float_as_uint(y.w);
                        }
                        return same;
                    };
                    PPFM_CHK(PPFM_CHK_RING_ACQUIRE, ring_matches());
#endif
                    if (ch < nch_q) run_chunk(s4, n, std::false_type{});
                    else run_chunk(s4, n, std::true_type{});
#ifdef PPFM_CHECKS
                    PPFM_CHK(PPFM_CHK_RING_RELEASE, ring_matches());
#endif
                    __syncwarp();
                    if ((tid & 31) == 0) mbar_arrive(&empty_bar[st]);
#pragma unroll
                    for (int h = 0; h < H; h++) {
                        Etot[h] = __fadd2_rn(Etot[h], E[h]); E[h] = zero2;
                        if (SPLIT) { Getot[h] = __fadd2_rn(Getot[h], Ge[h]); Ge[h] = zero2; }
                    }
                }
            }

    if (valid) {
#pragma unroll
        for (int h = 0; h < H; h++) {
            const size_t o = (size_t)job.out_offset + (size_t)(k0 + 2 * h) * job.nxy + col;
            PPFM_CHK(PPFM_CHK_FF_STORE, k0 + 2 * h >= job.nz ||
                                            o + (k0 + 2 * h + 1 < job.nz ? job.nxy : 0) <
                                                (size_t)job.out_offset + (size_t)job.nz * job.nxy);
            if (k0 + 2 * h < job.nz) {
                out_a[o] = make_float4(Fx[h].x, Fy[h].x, Fz[h].x, Etot[h].x);
                if (SPLIT) out_b[o] = make_float4(Gx[h].x, Gy[h].x, Gz[h].x, Getot[h].x);
            }
            if (k0 + 2 * h + 1 < job.nz) {
                out_a[o + job.nxy] = make_float4(Fx[h].y, Fy[h].y, Fz[h].y, Etot[h].y);
                if (SPLIT) out_b[o + job.nxy] = make_float4(Gx[h].y, Gy[h].y, Gz[h].y, Getot[h].y);
            }
        }
    }
}

__device__ __forceinline__ void ff_init_barriers(uint64_t *full_bar, uint64_t *empty_bar) {
    if (threadIdx.x == 0) {
        for (int s = 0; s < FF_STAGES; s++) {
            mbar_init(&full_bar[s], 1);
            mbar_init(&empty_bar[s], FF_THREADS / 32);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
}

// CTAs per SM the register budget is cut for.  The software-pipelined body keeps ~(18 + 4) registers per point pair
// plus ~40 (two accumulator sets in split mode: ~28 per pair): P = 20 needs the full 255 registers (2 CTAs of 128
// threads per SM), P <= 10 fits 168 (3 CTAs).  More warps do not help: the loop is bound by issue slots, not latency.
template <int P, bool SPLIT>
constexpr int ff_min_ctas() { return (SPLIT ? (P >= 10 ? 2 : 3) : (P >= 16 ? 2 : 3)) * (128 / FF_THREADS); }

// One system: job in the constant bank (kernel parameter).
template <int P, bool SPLIT, bool ZCOL>
__global__ void __launch_bounds__(FF_THREADS, ff_min_ctas<P, SPLIT>())
ff_kernel(const __grid_constant__ FFJob job, const FFFlags *__restrict__ flags, const AtomRec *__restrict__ recs,
          float4 *__restrict__ out_a, float4 *__restrict__ out_b) {
    __shared__ __align__(128) AtomRec s_rec[FF_STAGES * FF_CHUNK];
    __shared__ __align__(8) uint64_t full_bar[FF_STAGES];
    __shared__ __align__(8) uint64_t empty_bar[FF_STAGES];
    __shared__ FFFlags s_flags;
    if (threadIdx.x == 0) s_flags = flags[0];
    ff_init_barriers(full_bar, empty_bar);
    __syncthreads();
    if (s_flags.clamp)
        ff_tile<P, SPLIT, true, ZCOL>(job, s_flags.ncharged, recs, out_a, out_b, s_rec, full_bar, empty_bar,
                                      (long long)blockIdx.x);
    else
        ff_tile<P, SPLIT, false, ZCOL>(job, s_flags.ncharged, recs, out_a, out_b, s_rec, full_bar, empty_bar,
                                       (long long)blockIdx.x);
}

// Batch: the CTA finds its system in a device array and keeps a copy in shared memory.
template <int P, bool SPLIT, bool ZCOL>
__global__ void __launch_bounds__(FF_THREADS, ff_min_ctas<P, SPLIT>())
ff_batch_kernel(const FFJob *__restrict__ jobs, int njobs, const FFFlags *__restrict__ flags,
                const AtomRec *__restrict__ recs, float4 *__restrict__ out_a, float4 *__restrict__ out_b) {
    __shared__ __align__(128) AtomRec s_rec[FF_STAGES * FF_CHUNK];
    __shared__ __align__(8) uint64_t full_bar[FF_STAGES];
    __shared__ __align__(8) uint64_t empty_bar[FF_STAGES];
    __shared__ FFJob s_job;
    __shared__ FFFlags s_flags;

    const long long tile = blockIdx.x;
    // the system this tile belongs to: with equal tile counts per system (the usual batch) it is tile * njobs / ntiles,
    // checked with two independent loads; otherwise a binary search (log2(njobs) dependent loads, ~0.3 us each from
    // L2, which a CTA of a 35-atom molecule would spend a fifth of its life on)
    int lo = (int)((tile * njobs) / gridDim.x);
    {
        const long long b0 = jobs[lo].tile_begin;
        const long long b1 = (lo + 1 < njobs) ? jobs[lo + 1].tile_begin : (long long)gridDim.x;
        if (!(b0 <= tile && tile < b1)) {
            int hi = njobs - 1;
            lo = 0;
            while (lo < hi) {
                const int mid = (lo + hi + 1) >> 1;
                if (jobs[mid].tile_begin <= tile) lo = mid; else hi = mid - 1;
            }
        }
    }
    {
        const int *srcw = reinterpret_cast<const int *>(&jobs[lo]);
        int *dstw = reinterpret_cast<int *>(&s_job);
        for (int w = threadIdx.x; w < (int)(sizeof(FFJob) / sizeof(int)); w += FF_THREADS) dstw[w] = srcw[w];
    }
    if (threadIdx.x == 0) s_flags = flags[lo];
    ff_init_barriers(full_bar, empty_bar);
    __syncthreads();
    const long long local_tile = tile - s_job.tile_begin;
    if (s_flags.clamp)
        ff_tile<P, SPLIT, true, ZCOL>(s_job, s_flags.ncharged, recs, out_a, out_b, s_rec, full_bar, empty_bar, local_tile);
    else
        ff_tile<P, SPLIT, false, ZCOL>(s_job, s_flags.ncharged, recs, out_a, out_b, s_rec, full_bar, empty_bar, local_tile);
}

// ------------------------------------------------------------------------------------------- energy-only pass (N4)
// SURVEY 8(f) N4, PAPER.md:264 ("tri-cubic interpolation of the potential ... avoid storage of forces (i.e. improve
// memory efficiency)"): the same sum as a2 but only E = E_LJ + E_C per grid point, 4 bytes per point instead of 16,
// for ppfm_relax_scan_tricubic.  Same tile shape, atom records and TMA ring as ff_tile; the pair body shrinks to
// 8 packed FP32x2 instructions + 2 MUFU.RSQ per pair of points (no force factor, no three accumulating FMAs), which
// puts the XU (MUFU) pipe level with the FMA pipe.  The derivative stencil of the tri-cubic interpolant amplifies
// node-to-node noise, so the per-chunk FP32 partial sums are folded into FP64 totals (P DADDs per 256 atoms).
template <int P, bool CLAMP, bool ZCOL>
__device__ __forceinline__ void ffe_tile(const FFJob &job, int ncharged, const AtomRec *__restrict__ recs,
                                         float *__restrict__ out, AtomRec *s_rec, uint64_t *full_bar,
                                         uint64_t *empty_bar, long long local_tile) {
    const int tid = threadIdx.x;
    const int zg = (int)(local_tile / job.n_xy_tiles);
    const int xyt = (int)(local_tile - (long long)zg * job.n_xy_tiles);
    const int col = xyt * FF_THREADS + tid;
    const bool valid = col < job.nxy;
    const int colc = valid ? col : job.nxy - 1;
    const int j = colc / job.nx, i = colc - j * job.nx;
    const int k0 = zg * P;
    double pb[3];
#pragma unroll
    for (int c = 0; c < 3; c++)
        pb[c] = job.origin[c] + i * job.step[0][c] + j * job.step[1][c] + k0 * job.step[2][c];
    constexpr int H = P / 2;
    static_assert(P % 2 == 0, "P must be even: points are processed as FP32x2 pairs");
    float2 off[ZCOL ? 1 : 3][H];   // offsets of the points along step[2] (ZCOL: step[2] is parallel to z)
#pragma unroll
    for (int h = 0; h < H; h++)
#pragma unroll
        for (int c = 0; c < (ZCOL ? 1 : 3); c++) {
            const int cc = ZCOL ? 2 : c;
            off[c][h] = make_float2((float)((2 * h) * job.step[2][cc]), (float)((2 * h + 1) * job.step[2][cc]));
        }

    float2 E[H];
    double Etot[P];
    const float2 zero2 = make_float2(0.0f, 0.0f);
#pragma unroll
    for (int h = 0; h < H; h++) { E[h] = zero2; Etot[2 * h] = 0.0; Etot[2 * h + 1] = 0.0; }

    const int natoms = job.natoms;
    const int nq = min(max(ncharged, 0), natoms);
    const int nch_q = (nq + FF_CHUNK - 1) / FF_CHUNK;
    const int nchunks = nch_q + (natoms - nq + FF_CHUNK - 1) / FF_CHUNK;
    auto chunk_begin = [&](int c) { return c < nch_q ? c * FF_CHUNK : nq + (c - nch_q) * FF_CHUNK; };
    auto chunk_count = [&](int c) {
        return c < nch_q ? min(FF_CHUNK, nq - c * FF_CHUNK) : min(FF_CHUNK, natoms - nq - (c - nch_q) * FF_CHUNK);
    };
    const int nimages = (2 * job.nimg[0] + 1) * (2 * job.nimg[1] + 1) * (2 * job.nimg[2] + 1);
    const int nsteps = nimages * nchunks;
    const AtomRec *src = recs + job.atom_begin;
    const float rmin2 = job.rmin2;
    auto issue = [&](int t) {
        const int st = t % FF_STAGES;
        const int use = t / FF_STAGES;
        if (use > 0) mbar_wait(&empty_bar[st], (use - 1) & 1);
        const int c = t % nchunks;
        const uint32_t bytes = (uint32_t)chunk_count(c) * (uint32_t)sizeof(AtomRec);
        mbar_expect_tx(&full_bar[st], bytes);
        tma_load_1d(s_rec + st * FF_CHUNK, src + chunk_begin(c), bytes, &full_bar[st]);
    };
    if (tid == 0)
        for (int t = 0; t < FF_AHEAD && t < nsteps; t++) issue(t);

    float ph[3], pl[3];
    // two atoms per trip so that one atom's MUFU results are in flight while the other's polynomial runs
    auto pair_energy = [&](const float4 *s4, int a, auto neutral_tag) {
        constexpr bool NEUTRAL = decltype(neutral_tag)::value;
        const float4 r0 = s4[3 * a];
        const float4 r1 = s4[3 * a + 1];
        const float4 r2_ = s4[3 * a + 2];
        const float2 c12 = make_float2(r1.x, r1.y), nc6 = make_float2(r1.z, r1.w), kq = make_float2(r2_.z, r2_.w);
        const float dx0 = (ph[0] - r0.x) + pl[0];
        const float dy0 = (ph[1] - r0.y) + pl[1];
        const float dz0 = (ph[2] - r0.z) + pl[2];
        const float2 dxx = make_float2(dx0, dx0), dyy = make_float2(dy0, dy0), dzz = make_float2(dz0, dz0);
        float2 r2[H], ir[H];
        if (ZCOL) {
            const float rxy2s = fmaf(dy0, dy0, dx0 * dx0);
            const float2 rxy2 = make_float2(rxy2s, rxy2s);
#pragma unroll
            for (int h = 0; h < H; h++) {
                const float2 dz = __fadd2_rn(dzz, off[0][h]);
                r2[h] = __ffma2_rn(dz, dz, rxy2);
            }
        } else {
#pragma unroll
            for (int h = 0; h < H; h++) {
                const float2 dx = __fadd2_rn(dxx, off[0][h]), dy = __fadd2_rn(dyy, off[1 % (ZCOL ? 1 : 3)][h]),
                             dz = __fadd2_rn(dzz, off[2 % (ZCOL ? 1 : 3)][h]);
                r2[h] = __ffma2_rn(dz, dz, __ffma2_rn(dy, dy, __fmul2_rn(dx, dx)));
            }
        }
#pragma unroll
        for (int h = 0; h < H; h++) {
            if (CLAMP) { r2[h].x = fmaxf(r2[h].x, rmin2); r2[h].y = fmaxf(r2[h].y, rmin2); }
            ir[h].x = rsqrt_approx(r2[h].x);
            ir[h].y = rsqrt_approx(r2[h].y);
        }
        // (A Newton step on 1/r^2 was measured, round 3: config 1's worst |dE| near E = 0 went 1.97e-7 -> 1.42e-7 eV for
        // 2 more instructions per pair; what remains is the FP32 rounding of ~60-256 signed Coulomb terms inside a
        // chunk, so the step was dropped.)
        float2 ir2[H], ir6[H], t[H];
#pragma unroll
        for (int h = 0; h < H; h++) ir2[h] = __fmul2_rn(ir[h], ir[h]);
#pragma unroll
        for (int h = 0; h < H; h++) ir6[h] = __fmul2_rn(ir2[h], ir2[h]);
#pragma unroll
        for (int h = 0; h < H; h++) ir6[h] = __fmul2_rn(ir6[h], ir2[h]);
#pragma unroll
        for (int h = 0; h < H; h++) t[h] = __ffma2_rn(c12, ir6[h], nc6);              // c12/r^6 - c6
#pragma unroll
        for (int h = 0; h < H; h++) E[h] = __ffma2_rn(t[h], ir6[h], E[h]);            // E_LJ (Eq.5)
        if (!NEUTRAL) {
#pragma unroll
            for (int h = 0; h < H; h++) E[h] = __ffma2_rn(kq, ir[h], E[h]);           // E_C = kq / r (Eq.6)
        }
    };
    auto run_chunk = [&](const float4 *s4, int n, auto neutral_tag) {
#pragma unroll 2
        for (int a = 0; a < n; a++) pair_energy(s4, a, neutral_tag);
    };

    int step = 0;
    for (int ia = -job.nimg[0]; ia <= job.nimg[0]; ia++)
        for (int ib = -job.nimg[1]; ib <= job.nimg[1]; ib++)
            for (int ic = -job.nimg[2]; ic <= job.nimg[2]; ic++) {
#pragma unroll
                for (int c = 0; c < 3; c++) {
                    const double s = pb[c] - (ia * job.cell[0][c] + ib * job.cell[1][c] + ic * job.cell[2][c]);
                    ph[c] = (float)s;
                    pl[c] = (float)(s - (double)ph[c]);
                }
                for (int ch = 0; ch < nchunks; ch++, step++) {
                    if (tid == 0 && step + FF_AHEAD < nsteps) issue(step + FF_AHEAD);
                    const int st = step % FF_STAGES;
                    mbar_wait(&full_bar[st], (step / FF_STAGES) & 1);
                    const float4 *s4 = reinterpret_cast<const float4 *>(s_rec + st * FF_CHUNK);
                    const int n = chunk_count(ch);
                    if (ch < nch_q) run_chunk(s4, n, std::false_type{});
                    else run_chunk(s4, n, std::true_type{});
                    __syncwarp();
                    if ((tid & 31) == 0) mbar_arrive(&empty_bar[st]);
#pragma unroll
                    for (int h = 0; h < H; h++) {          // fold the chunk's FP32 partial sums into the FP64 totals
                        Etot[2 * h] += (double)E[h].x;
                        Etot[2 * h + 1] += (double)E[h].y;
                        E[h] = zero2;
                    }
                }
            }
    if (valid) {
#pragma unroll
        for (int p = 0; p < P; p++) {
            const size_t o = (size_t)job.out_offset + (size_t)(k0 + p) * job.nxy + col;
            PPFM_CHK(PPFM_CHK_FF_STORE, k0 + p >= job.nz || o < (size_t)job.out_offset + (size_t)job.nz * job.nxy);
            if (k0 + p < job.nz) out[o] = (float)Etot[p];
        }
    }
}

template <int P, bool ZCOL>
__global__ void __launch_bounds__(FF_THREADS, 2)
ffe_kernel(const __grid_constant__ FFJob job, const FFFlags *__restrict__ flags, const AtomRec *__restrict__ recs,
           float *__restrict__ out) {
    __shared__ __align__(128) AtomRec s_rec[FF_STAGES * FF_CHUNK];
    __shared__ __align__(8) uint64_t full_bar[FF_STAGES];
    __shared__ __align__(8) uint64_t empty_bar[FF_STAGES];
    __shared__ FFFlags s_flags;
    if (threadIdx.x == 0) s_flags = flags[0];
    ff_init_barriers(full_bar, empty_bar);
    __syncthreads();
    if (s_flags.clamp)
        ffe_tile<P, true, ZCOL>(job, s_flags.ncharged, recs, out, s_rec, full_bar, empty_bar, (long long)blockIdx.x);
    else
        ffe_tile<P, false, ZCOL>(job, s_flags.ncharged, recs, out, s_rec, full_bar, empty_bar, (long long)blockIdx.x);
}

// ---------------------------------------------------------------------------------------------------- a3 combine
__global__ void combine_kernel(const float4 *__restrict__ lj, const float4 *__restrict__ el, float Q, long long n,
                               float4 *__restrict__ out) {
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const float4 a = lj[i], b = el[i];
        out[i] = make_float4(fmaf(Q, b.x, a.x), fmaf(Q, b.y, a.y), fmaf(Q, b.z, a.z), fmaf(Q, b.w, a.w));
    }
}

// ---------------------------------------------------------------------------------------------------- host side
static int pick_P(int nz, long long nxy_tiles, bool split) {
    // padded work ~ ceil(nz/P) * (P + per-atom overhead shared by the column, ~1.2 points: 8 scalar FP32 + 3 LDS +
    // loop control against ~16 issue slots per point).  The split kernel keeps two accumulator sets per point, so
    // it takes fewer points per thread.  Small grids take the smallest P that still gives every SM two CTAs.
    const int cand_one[4] = {20, 16, 10, 8}, cand_two[4] = {10, 8, 6, 6};
    const int *cand = split ? cand_two : cand_one;
    int best = cand[0];
    double best_cost = 1e300;
    for (int c = 0; c < 4; c++) {
        const int P = cand[c];
        const long long ctas = nxy_tiles * ((nz + P - 1) / P);
        double cost = (double)((nz + P - 1) / P) * (P + 1.2);
        if (ctas < 2 * 148) cost *= 2.0 * 148.0 / (double)(ctas > 0 ? ctas : 1);      // idle SMs
        if (cost < best_cost - 1e-9) { best_cost = cost; best = P; }
    }
    return best;
}

template <bool SPLIT, int P, bool ZCOL>
static void launch_ff_one(long long ntiles, cudaStream_t st, const FFJob *hj, const FFJob *dj, int njobs,
                          const FFFlags *flags, const AtomRec *recs, float4 *a, float4 *b) {
    const dim3 grid((unsigned)ntiles), block(FF_THREADS);
    if (njobs == 1) ff_kernel<P, SPLIT, ZCOL><<<grid, block, 0, st>>>(hj[0], flags, recs, a, b);
    else ff_batch_kernel<P, SPLIT, ZCOL><<<grid, block, 0, st>>>(dj, njobs, flags, recs, a, b);
}

template <bool SPLIT>
static cudaError_t launch_ff(int P, bool zcol, long long ntiles, cudaStream_t st, const FFJob *hj, const FFJob *dj,
                             int njobs, const FFFlags *flags, const AtomRec *recs, float4 *a, float4 *b) {
    KernelTimer kt(PPFM_K_FF, st);
    if (!zcol) launch_ff_one<SPLIT, 4, false>(ntiles, st, hj, dj, njobs, flags, recs, a, b);
    else if (P == 8) launch_ff_one<SPLIT, 8, true>(ntiles, st, hj, dj, njobs, flags, recs, a, b);
    else if (P == 10) launch_ff_one<SPLIT, 10, true>(ntiles, st, hj, dj, njobs, flags, recs, a, b);
    else if constexpr (SPLIT) launch_ff_one<true, 6, true>(ntiles, st, hj, dj, njobs, flags, recs, a, b);
#ifdef PPFM_EXPERIMENT
    else if (P == 12) launch_ff_one<false, 12, true>(ntiles, st, hj, dj, njobs, flags, recs, a, b);
    else if (P == 14) launch_ff_one<false, 14, true>(ntiles, st, hj, dj, njobs, flags, recs, a, b);
#endif
    else if (P == 16) launch_ff_one<false, 16, true>(ntiles, st, hj, dj, njobs, flags, recs, a, b);
    else launch_ff_one<false, 20, true>(ntiles, st, hj, dj, njobs, flags, recs, a, b);
    return cudaGetLastError();
}

static int forcefield_impl(int nsys, const int32_t *h_atom_offset, const float *d_xyzq, const int32_t *d_type,
                           int32_t ntypes, const double *h_R, const double *h_e, const ppfm_lattice *lattices,
                           const ppfm_probe *probes, const ppfm_grid *grids, double r_min, float *d_a, float *d_b,
                           bool split, ppfm_ff_status *d_status, void *cuda_stream) {
    if (nsys < 1 || !h_atom_offset || !h_R || !h_e || !lattices || !probes || !grids || !d_a) return PPFM_EINVAL;
    if (h_atom_offset[nsys] > 0 && (!d_xyzq || !d_type)) return PPFM_EINVAL;   // an empty atom list may be NULL
    if (split && !d_b) return PPFM_EINVAL;
    if (ntypes < 1 || ntypes > PPFM_MAX_TYPES) return PPFM_EINVAL;
    if (!(r_min >= 0.0) || !std::isfinite(r_min)) return PPFM_EINVAL;
    if (((uintptr_t)d_xyzq & 15) || ((uintptr_t)d_a & 15) || (d_b && ((uintptr_t)d_b & 15)) || ((uintptr_t)d_status & 3))
        return PPFM_EINVAL;
    for (int t = 0; t < ntypes; t++)
        if (!(h_R[t] >= 0.0) || !(h_e[t] >= 0.0) || !std::isfinite(h_R[t]) || !std::isfinite(h_e[t])) return PPFM_EINVAL;
    if (h_atom_offset[0] != 0) return PPFM_EINVAL;

    // choose one P / column mode for the launch
    bool zcol = true;
    int nz_common = grids[0].n[2];
    for (int m = 0; m < nsys; m++) {
        const ppfm_grid &g = grids[m];
        if (!grid_ok(&g)) return PPFM_EINVAL;
        if (h_atom_offset[m + 1] < h_atom_offset[m]) return PPFM_EINVAL;
        const ppfm_probe &pr = probes[m];
        if (!(pr.R >= 0.0) || !(pr.e >= 0.0) || !std::isfinite(pr.R) || !std::isfinite(pr.e) || !std::isfinite(pr.Q))
            return PPFM_EINVAL;
        for (int a = 0; a < 3; a++)
            if (lattices[m].nimg[a] < 0 || lattices[m].nimg[a] > 64) return PPFM_EINVAL;
        if (g.step[2][0] != 0.0 || g.step[2][1] != 0.0) zcol = false;
        if (g.n[2] != nz_common) nz_common = -1;
    }
    long long nxy_tiles_total = 0;
    for (int m = 0; m < nsys; m++)
        nxy_tiles_total += ((long long)grids[m].n[0] * grids[m].n[1] + FF_THREADS - 1) / FF_THREADS;
    int P = zcol ? pick_P(nz_common > 0 ? nz_common : grids[0].n[2], nxy_tiles_total, split) : 4;
#ifdef PPFM_EXPERIMENT
    if (zcol && !split && getenv("PPFM_FF_FORCE_P")) P = atoi(getenv("PPFM_FF_FORCE_P"));
#endif

    const bool single = (nsys == 1);
    const size_t jobs_bytes = (size_t)nsys * sizeof(FFJob);
    const size_t table_bytes = (size_t)nsys * ntypes * sizeof(TypeEntry);
    const size_t host_bytes = (jobs_bytes + table_bytes + 15) & ~(size_t)15;
    // device scratch: [jobs | tables] (batch only) [clamp flags] [atom records]
    const size_t flags_off = single ? 0 : host_bytes;
    const size_t flags_bytes = ((size_t)nsys * sizeof(FFFlags) + 15) & ~(size_t)15;
    const size_t recs_off = flags_off + flags_bytes;
    const int natoms_total = h_atom_offset[nsys];
    const size_t recs_bytes = (size_t)(natoms_total > 0 ? natoms_total : 1) * sizeof(AtomRec);
    const size_t total_bytes = recs_off + recs_bytes;

    unsigned char *h_buf = (unsigned char *)malloc(host_bytes);
    if (!h_buf) return PPFM_ENOMEM;
    memset(h_buf, 0, host_bytes);
    FFJob *hj = reinterpret_cast<FFJob *>(h_buf);
    TypeEntry *ht = reinterpret_cast<TypeEntry *>(h_buf + jobs_bytes);
    long long tile = 0, out_off = 0;
    for (int m = 0; m < nsys; m++) {
        const ppfm_grid &g = grids[m];
        FFJob &j = hj[m];
        j.tile_begin = tile;
        j.out_offset = out_off;
        j.atom_begin = h_atom_offset[m];
        j.natoms = h_atom_offset[m + 1] - h_atom_offset[m];
        j.nx = g.n[0]; j.ny = g.n[1]; j.nz = g.n[2]; j.nxy = g.n[0] * g.n[1];
        j.n_xy_tiles = (j.nxy + FF_THREADS - 1) / FF_THREADS;
        j.n_z_groups = (j.nz + P - 1) / P;
        j.table_offset = m * ntypes;
        j.ntypes = ntypes;
        j.split = split ? 1 : 0;
        for (int a = 0; a < 3; a++) {
            j.nimg[a] = lattices[m].nimg[a];
            j.origin[a] = g.origin[a];
            for (int c = 0; c < 3; c++) j.step[a][c] = g.step[a][c];
            j.cell[0][a] = lattices[m].a[a];
            j.cell[1][a] = lattices[m].b[a];
            j.cell[2][a] = lattices[m].c[a];
        }
        for (int c = 0; c < 3; c++) {
            double lo = g.origin[c], hi = g.origin[c];
            for (int corner = 1; corner < 8; corner++) {
                double x = g.origin[c];
                for (int a = 0; a < 3; a++)
                    if (corner & (1 << a)) x += (g.n[a] - 1) * g.step[a][c];
                lo = std::fmin(lo, x); hi = std::fmax(hi, x);
            }
            j.bb_lo[c] = lo; j.bb_hi[c] = hi;
        }
        j.keQ = (float)(kCoulomb * probes[m].Q);
        j.rmin2 = (float)(r_min * r_min);
        for (int t = 0; t < ntypes; t++) {   // mixing rules
            const double R0 = h_R[t] + probes[m].R;
            const double E0 = std::sqrt(h_e[t] * probes[m].e);
            const double R6 = R0 * R0 * R0 * R0 * R0 * R0;
            ht[m * ntypes + t].c6 = (float)(2.0 * E0 * R6);
            ht[m * ntypes + t].c12 = (float)(E0 * R6 * R6);
        }
        tile += (long long)j.n_xy_tiles * j.n_z_groups;
        out_off += grid_points(&g);
    }
    if (tile > 0x7fffffffLL) { free(h_buf); return PPFM_EINVAL; }

    cudaStream_t st = (cudaStream_t)cuda_stream;
    unsigned char *d_buf = nullptr;
    cudaError_t e = scratch_alloc((void **)&d_buf, total_bytes, st);
    if (e != cudaSuccess) { free(h_buf); set_cuda_error(e, "scratch_alloc"); return PPFM_ENOMEM; }
    if (!single) e = cudaMemcpyAsync(d_buf, h_buf, host_bytes, cudaMemcpyHostToDevice, st);   // pageable: staged before return
    if (e == cudaSuccess) e = cudaMemsetAsync(d_buf + flags_off, 0, flags_bytes, st);
    if (e == cudaSuccess && d_status) e = cudaMemsetAsync(d_status, 0, sizeof(ppfm_ff_status), st);
    if (e != cudaSuccess) { free(h_buf); set_cuda_error(e, "scratch upload"); cudaFreeAsync(d_buf, st); return PPFM_ECUDA; }
    const FFJob *dj = reinterpret_cast<const FFJob *>(d_buf);
    const TypeEntry *dt = reinterpret_cast<const TypeEntry *>(d_buf + jobs_bytes);
    FFFlags *dflags = reinterpret_cast<FFFlags *>(d_buf + flags_off);
    AtomRec *drecs = reinterpret_cast<AtomRec *>(d_buf + recs_off);
    if (natoms_total > 0) {
        {
            KernelTimer kt(PPFM_K_FF_PREP, st);
            if (single) {
                FFSingle one;
                memset(&one, 0, sizeof(one));
                one.job = hj[0];
                memcpy(one.table, ht, (size_t)ntypes * sizeof(TypeEntry));
                ff_prep_kernel<<<1, PREP_THREADS, 0, st>>>(one, reinterpret_cast<const float4 *>(d_xyzq), d_type, drecs,
                                                           dflags, d_status);
            } else {
                ff_prep_batch_kernel<<<nsys, PREP_THREADS, 0, st>>>(
                    dj, dt, reinterpret_cast<const float4 *>(d_xyzq), d_type, drecs, dflags, d_status);
            }
        }
        e = cudaGetLastError();
        if (e != cudaSuccess) { free(h_buf); set_cuda_error(e, "ff_prep_kernel"); cudaFreeAsync(d_buf, st); return PPFM_ECUDA; }
        count_launch();
    }
    if (tile > 0) {
        e = split ? launch_ff<true>(P, zcol, tile, st, hj, dj, nsys, dflags, drecs, reinterpret_cast<float4 *>(d_a),
                                    reinterpret_cast<float4 *>(d_b))
                  : launch_ff<false>(P, zcol, tile, st, hj, dj, nsys, dflags, drecs, reinterpret_cast<float4 *>(d_a),
                                     nullptr);
        if (e != cudaSuccess) { free(h_buf); set_cuda_error(e, "ff_kernel"); cudaFreeAsync(d_buf, st); return PPFM_ECUDA; }
        count_launch();
    }
    free(h_buf);
    PPFM_CUDA(cudaFreeAsync(d_buf, st));
    return PPFM_OK;
}

}  // namespace ppfm

using namespace ppfm;

extern "C" int ppfm_forcefield(int32_t natoms, const float *d_xyzq, const int32_t *d_type, int32_t ntypes,
                               const double *h_R, const double *h_e, const ppfm_lattice *lattice,
                               const ppfm_probe *probe, const ppfm_grid *grid, double r_min, float *d_ff,
                               ppfm_ff_status *d_status, void *cuda_stream) {
    if (natoms < 0) return PPFM_EINVAL;
    const int32_t off[2] = {0, natoms};
    return forcefield_impl(1, off, d_xyzq, d_type, ntypes, h_R, h_e, lattice, probe, grid, r_min, d_ff, nullptr,
                           false, d_status, cuda_stream);
}

extern "C" int ppfm_forcefield_split(int32_t natoms, const float *d_xyzq, const int32_t *d_type, int32_t ntypes,
                                     const double *h_R, const double *h_e, const ppfm_lattice *lattice,
                                     const ppfm_probe *probe, const ppfm_grid *grid, double r_min, float *d_ff_lj,
                                     float *d_ff_el, ppfm_ff_status *d_status, void *cuda_stream) {
    if (natoms < 0) return PPFM_EINVAL;
    const int32_t off[2] = {0, natoms};
    return forcefield_impl(1, off, d_xyzq, d_type, ntypes, h_R, h_e, lattice, probe, grid, r_min, d_ff_lj, d_ff_el,
                           true, d_status, cuda_stream);
}

extern "C" int ppfm_forcefield_batch(int32_t nsys, const int32_t *h_atom_offset, const float *d_xyzq,
                                     const int32_t *d_type, int32_t ntypes, const double *h_R, const double *h_e,
                                     const ppfm_lattice *lattices, const ppfm_probe *probes, const ppfm_grid *grids,
                                     double r_min, float *d_ff, ppfm_ff_status *d_status, void *cuda_stream) {
    return forcefield_impl(nsys, h_atom_offset, d_xyzq, d_type, ntypes, h_R, h_e, lattices, probes, grids, r_min,
                           d_ff, nullptr, false, d_status, cuda_stream);
}

extern "C" int ppfm_combine(const float *d_ff_lj, const float *d_ff_el, double Q, int64_t n_points, float *d_out,
                            void *cuda_stream) {
    if (!d_ff_lj || !d_ff_el || !d_out || n_points < 0 || !std::isfinite(Q)) return PPFM_EINVAL;
    if (((uintptr_t)d_ff_lj & 15) || ((uintptr_t)d_ff_el & 15) || ((uintptr_t)d_out & 15)) return PPFM_EINVAL;
    if (n_points == 0) return PPFM_OK;
    long long blocks = (n_points + 255) / 256;
    if (blocks > 148LL * 16) blocks = 148LL * 16;
    {
        KernelTimer kt(PPFM_K_COMBINE, (cudaStream_t)cuda_stream);
        combine_kernel<<<(unsigned)blocks, 256, 0, (cudaStream_t)cuda_stream>>>(
            reinterpret_cast<const float4 *>(d_ff_lj), reinterpret_cast<const float4 *>(d_ff_el), (float)Q, n_points,
            reinterpret_cast<float4 *>(d_out));
    }
    PPFM_LAUNCH_CHECK();
    return PPFM_OK;
}

// ------------------------------------------------------------------------- (1') the pass without any allocation
// ppfm_forcefield_noalloc (include/ppfm.h): for callers that may not allocate after start-up (a pre-carved device
// arena, a real-time loop, an allocator hook that forbids cudaMalloc*).  It runs ff_prep_kernel and ff_kernel, the
// kernels of ppfm_forcefield, but the scratch those two share — the FFFlags the prep kernel writes and the packed
// AtomRec array — lives in the file-scope device array below instead of a pool allocation.  Every GPU that loads this
// library's device code holds the array until the process exits.
//
// `g_noalloc_scratch` names device memory only inside device code.  In host code the same identifier is a host-side
// handle of the symbol, NOT a device address: handing it to a kernel would fault (or, on a system where the GPU can
// reach host memory, quietly read and write the wrong bytes).  The host gets the real address from
// cudaGetSymbolAddress, once per device with that device current (noalloc_scratch_ptr), and passes that to the kernels.
namespace ppfm {

constexpr size_t NOALLOC_RECS_OFF = 256;      // [FFFlags, padding to 256 B][AtomRec x PPFM_NOALLOC_MAX_ATOMS]
static_assert(sizeof(FFFlags) <= NOALLOC_RECS_OFF, "flags must fit ahead of the records");
static_assert(PPFM_NOALLOC_SCRATCH_BYTES == NOALLOC_RECS_OFF + sizeof(AtomRec) * PPFM_NOALLOC_MAX_ATOMS,
              "PPFM_NOALLOC_SCRATCH_BYTES (ppfm.h) must describe this layout");
static __device__ __align__(256) unsigned char g_noalloc_scratch[PPFM_NOALLOC_SCRATCH_BYTES];

static std::atomic<unsigned char *> g_noalloc_ptr[64];      // per device ordinal; zero-initialised (static storage)

// Device address of g_noalloc_scratch on the CURRENT device.  The first call on a device asks the runtime (which may
// load this library's device code on that device: do it before any stream capture); later calls read the cached
// pointer.  Two threads racing through the first call both get the same answer from the runtime, so a plain atomic
// store is enough and no lock is taken on the steady-state path.
static cudaError_t noalloc_scratch_ptr(unsigned char **out) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
    unsigned char *p = g_noalloc_ptr[dev].load(std::memory_order_acquire);
    if (!p) {
        void *sym = nullptr;
        e = cudaGetSymbolAddress(&sym, g_noalloc_scratch);
        if (e != cudaSuccess) return e;
        if (!sym) return cudaErrorInvalidSymbol;
        p = static_cast<unsigned char *>(sym);
        g_noalloc_ptr[dev].store(p, std::memory_order_release);
    }
    *out = p;
    return cudaSuccess;
}

// launch_ff's dispatch for one system and one output grid, without its KernelTimer (which creates CUDA events when
// the ppfm_bench.h timers are on — an allocation this path must not make)
static cudaError_t launch_ff_noalloc(int P, bool zcol, long long ntiles, cudaStream_t st, const FFJob *hj,
                                     const FFFlags *flags, const AtomRec *recs, float4 *out) {
    if (!zcol) launch_ff_one<false, 4, false>(ntiles, st, hj, nullptr, 1, flags, recs, out, nullptr);
    else if (P == 8) launch_ff_one<false, 8, true>(ntiles, st, hj, nullptr, 1, flags, recs, out, nullptr);
    else if (P == 10) launch_ff_one<false, 10, true>(ntiles, st, hj, nullptr, 1, flags, recs, out, nullptr);
    else if (P == 16) launch_ff_one<false, 16, true>(ntiles, st, hj, nullptr, 1, flags, recs, out, nullptr);
    else launch_ff_one<false, 20, true>(ntiles, st, hj, nullptr, 1, flags, recs, out, nullptr);
    return cudaGetLastError();
}

}  // namespace ppfm

namespace ppfm {
// Validation and job description of ONE system on one grid, for the single-system entry points added in round 3
// (ppfm_forcefield_noalloc, ppfm_forcefield_energy): the checks and the FFJob / per-type table that forcefield_impl
// builds for nsys = 1, on the caller's stack (no heap).  P and the column mode are chosen as ppfm_forcefield does.
static int fill_single_job(FFSingle &one, int *P_out, bool *zcol_out, long long *ntiles_out, int32_t natoms,
                           int32_t ntypes, const double *h_R, const double *h_e, const ppfm_lattice *lattice,
                           const ppfm_probe *probe, const ppfm_grid *grid, double r_min) {
    if (natoms < 0 || !h_R || !h_e || !lattice || !probe || !grid) return PPFM_EINVAL;
    if (ntypes < 1 || ntypes > PPFM_MAX_TYPES) return PPFM_EINVAL;
    if (!(r_min >= 0.0) || !std::isfinite(r_min)) return PPFM_EINVAL;
    for (int t = 0; t < ntypes; t++)
        if (!(h_R[t] >= 0.0) || !(h_e[t] >= 0.0) || !std::isfinite(h_R[t]) || !std::isfinite(h_e[t])) return PPFM_EINVAL;
    if (!grid_ok(grid)) return PPFM_EINVAL;
    if (!(probe->R >= 0.0) || !(probe->e >= 0.0) || !std::isfinite(probe->R) || !std::isfinite(probe->e) ||
        !std::isfinite(probe->Q))
        return PPFM_EINVAL;
    for (int a = 0; a < 3; a++)
        if (lattice->nimg[a] < 0 || lattice->nimg[a] > 64) return PPFM_EINVAL;
    const ppfm_grid &g = *grid;
    const bool zcol = (g.step[2][0] == 0.0 && g.step[2][1] == 0.0);
    const long long nxy_tiles = ((long long)g.n[0] * g.n[1] + FF_THREADS - 1) / FF_THREADS;
    const int P = zcol ? pick_P(g.n[2], nxy_tiles, false) : 4;      // the choice ppfm_forcefield makes: same bits
    memset(&one, 0, sizeof(one));
    FFJob &j = one.job;
    j.natoms = natoms;
    j.nx = g.n[0]; j.ny = g.n[1]; j.nz = g.n[2]; j.nxy = g.n[0] * g.n[1];
    j.n_xy_tiles = (j.nxy + FF_THREADS - 1) / FF_THREADS;
    j.n_z_groups = (j.nz + P - 1) / P;
    j.ntypes = ntypes;
    for (int a = 0; a < 3; a++) {
        j.nimg[a] = lattice->nimg[a];
        j.origin[a] = g.origin[a];
        for (int c = 0; c < 3; c++) j.step[a][c] = g.step[a][c];
        j.cell[0][a] = lattice->a[a];
        j.cell[1][a] = lattice->b[a];
        j.cell[2][a] = lattice->c[a];
    }
    for (int c = 0; c < 3; c++) {      // Cartesian bounding box of the grid (decides whether the r_min clamp is live)
        double lo = g.origin[c], hi = g.origin[c];
        for (int corner = 1; corner < 8; corner++) {
            double x = g.origin[c];
            for (int a = 0; a < 3; a++)
                if (corner & (1 << a)) x += (g.n[a] - 1) * g.step[a][c];
            lo = std::fmin(lo, x); hi = std::fmax(hi, x);
        }
        j.bb_lo[c] = lo; j.bb_hi[c] = hi;
    }
    j.keQ = (float)(kCoulomb * probe->Q);
    j.rmin2 = (float)(r_min * r_min);
    for (int t = 0; t < ntypes; t++) {   // mixing rules
        const double R0 = h_R[t] + probe->R;
        const double E0 = std::sqrt(h_e[t] * probe->e);
        const double R6 = R0 * R0 * R0 * R0 * R0 * R0;
        one.table[t].c6 = (float)(2.0 * E0 * R6);
        one.table[t].c12 = (float)(E0 * R6 * R6);
    }
    const long long ntiles = (long long)j.n_xy_tiles * j.n_z_groups;
    if (ntiles > 0x7fffffffLL) return PPFM_EINVAL;
    *P_out = P; *zcol_out = zcol; *ntiles_out = ntiles;
    return PPFM_OK;
}
}  // namespace ppfm

extern "C" int ppfm_forcefield_noalloc(int32_t natoms, const float *d_xyzq, const int32_t *d_type, int32_t ntypes,
                                       const double *h_R, const double *h_e, const ppfm_lattice *lattice,
                                       const ppfm_probe *probe, const ppfm_grid *grid, double r_min, float *d_ff,
                                       ppfm_ff_status *d_status, void *cuda_stream) {
    // the argument checks of ppfm_forcefield (pointers here, the rest in fill_single_job)
    if (!d_ff || (natoms > 0 && (!d_xyzq || !d_type))) return PPFM_EINVAL;
    if (((uintptr_t)d_xyzq & 15) || ((uintptr_t)d_ff & 15) || ((uintptr_t)d_status & 3)) return PPFM_EINVAL;
    FFSingle one;      // the system's description travels as a kernel parameter: it lives on this stack frame
    int P = 0;
    bool zcol = true;
    long long ntiles = 0;
    {
        const int rc = fill_single_job(one, &P, &zcol, &ntiles, natoms, ntypes, h_R, h_e, lattice, probe, grid, r_min);
        if (rc != PPFM_OK) return rc;
    }
    // the one limit this entry point adds: the records must fit the fixed array
    if (natoms > PPFM_NOALLOC_MAX_ATOMS) return PPFM_ELIMIT;

    unsigned char *d_scratch = nullptr;
    cudaError_t e = noalloc_scratch_ptr(&d_scratch);
    if (e != cudaSuccess) { set_cuda_error(e, "cudaGetSymbolAddress(g_noalloc_scratch)"); return PPFM_ECUDA; }
    FFFlags *dflags = reinterpret_cast<FFFlags *>(d_scratch);
    AtomRec *drecs = reinterpret_cast<AtomRec *>(d_scratch + NOALLOC_RECS_OFF);

    cudaStream_t st = (cudaStream_t)cuda_stream;
    // The array still holds the previous call's flags and records.  The flags must read zero when no prep kernel runs
    // (natoms = 0), so they are cleared every call; records [0, natoms) are all rewritten by the prep kernel and no
    // record beyond natoms is ever read.
    e = cudaMemsetAsync(dflags, 0, sizeof(FFFlags), st);
    if (e == cudaSuccess && d_status) e = cudaMemsetAsync(d_status, 0, sizeof(ppfm_ff_status), st);
    if (e != cudaSuccess) { set_cuda_error(e, "noalloc flag reset"); return PPFM_ECUDA; }
    if (natoms > 0) {
        ff_prep_kernel<<<1, PREP_THREADS, 0, st>>>(one, reinterpret_cast<const float4 *>(d_xyzq), d_type, drecs, dflags,
                                                   d_status);
        e = cudaGetLastError();
        if (e != cudaSuccess) { set_cuda_error(e, "ff_prep_kernel (noalloc)"); return PPFM_ECUDA; }
        count_launch();
    }
    if (ntiles > 0) {
        e = launch_ff_noalloc(P, zcol, ntiles, st, &one.job, dflags, drecs, reinterpret_cast<float4 *>(d_ff));
        if (e != cudaSuccess) { set_cuda_error(e, "ff_kernel (noalloc)"); return PPFM_ECUDA; }
        count_launch();
    }
    return PPFM_OK;
}

// ------------------------------------------------------------------------------------------- (1e) energy-only grid
// ppfm_forcefield_energy (include/ppfm.h): E = E_LJ + E_C on the grid, float[nz][ny][nx],
// for ppfm_relax_scan_tricubic.  Set-up (records, flags, scratch) is ppfm_forcefield's; the grid kernel is ffe_kernel.
extern "C" int ppfm_forcefield_energy(int32_t natoms, const float *d_xyzq, const int32_t *d_type, int32_t ntypes,
                                      const double *h_R, const double *h_e, const ppfm_lattice *lattice,
                                      const ppfm_probe *probe, const ppfm_grid *grid, double r_min, float *d_E,
                                      ppfm_ff_status *d_status, void *cuda_stream) {
    if (!d_E || (natoms > 0 && (!d_xyzq || !d_type))) return PPFM_EINVAL;
    if (((uintptr_t)d_xyzq & 15) || ((uintptr_t)d_E & 3) || ((uintptr_t)d_status & 3)) return PPFM_EINVAL;
    FFSingle one;
    int P = 0;
    bool zcol = true;
    long long ntiles = 0;
    {
        const int rc = fill_single_job(one, &P, &zcol, &ntiles, natoms, ntypes, h_R, h_e, lattice, probe, grid, r_min);
        if (rc != PPFM_OK) return rc;
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t recs_off = 16;       // [FFFlags, padded to 16 B][AtomRec x natoms]
    const size_t total_bytes = recs_off + (size_t)(natoms > 0 ? natoms : 1) * sizeof(AtomRec);
    unsigned char *d_buf = nullptr;
    cudaError_t e = scratch_alloc((void **)&d_buf, total_bytes, st);
    if (e != cudaSuccess) { set_cuda_error(e, "scratch_alloc"); return PPFM_ENOMEM; }
    FFFlags *dflags = reinterpret_cast<FFFlags *>(d_buf);
    AtomRec *drecs = reinterpret_cast<AtomRec *>(d_buf + recs_off);
    e = cudaMemsetAsync(dflags, 0, sizeof(FFFlags), st);
    if (e == cudaSuccess && d_status) e = cudaMemsetAsync(d_status, 0, sizeof(ppfm_ff_status), st);
    if (e != cudaSuccess) { set_cuda_error(e, "scratch reset"); cudaFreeAsync(d_buf, st); return PPFM_ECUDA; }
    if (natoms > 0) {
        {
            KernelTimer kt(PPFM_K_FF_PREP, st);
            ff_prep_kernel<<<1, PREP_THREADS, 0, st>>>(one, reinterpret_cast<const float4 *>(d_xyzq), d_type, drecs,
                                                       dflags, d_status);
        }
        e = cudaGetLastError();
        if (e != cudaSuccess) { set_cuda_error(e, "ff_prep_kernel"); cudaFreeAsync(d_buf, st); return PPFM_ECUDA; }
        count_launch();
    }
    if (ntiles > 0) {
        const dim3 gridDim3((unsigned)ntiles), block(FF_THREADS);
        {
            KernelTimer kt(PPFM_K_FF_ENERGY, st);
            if (!zcol) ffe_kernel<4, false><<<gridDim3, block, 0, st>>>(one.job, dflags, drecs, d_E);
            else if (P == 8) ffe_kernel<8, true><<<gridDim3, block, 0, st>>>(one.job, dflags, drecs, d_E);
            else if (P == 10) ffe_kernel<10, true><<<gridDim3, block, 0, st>>>(one.job, dflags, drecs, d_E);
            else if (P == 16) ffe_kernel<16, true><<<gridDim3, block, 0, st>>>(one.job, dflags, drecs, d_E);
            else ffe_kernel<20, true><<<gridDim3, block, 0, st>>>(one.job, dflags, drecs, d_E);
        }
        e = cudaGetLastError();
        if (e != cudaSuccess) { set_cuda_error(e, "ffe_kernel"); cudaFreeAsync(d_buf, st); return PPFM_ECUDA; }
        count_launch();
    }
    PPFM_CUDA(cudaFreeAsync(d_buf, st));
    return PPFM_OK;
}
