// api.cu — the rest of the C ABI: status text, defaults, the one-call host-buffer simulation and the
// two measurement probes that define the roofline denominators on the box.
#include "common.cuh"

#include <mutex>
#include <vector>

namespace ppfm {

std::atomic<long long> g_launches{0};
std::atomic<int> g_timing_on{0};
static thread_local char g_cuda_msg[256] = "no CUDA error recorded";

void set_cuda_error(cudaError_t e, const char *where) {
    snprintf(g_cuda_msg, sizeof(g_cuda_msg), "CUDA error %d (%s) in %s", (int)e, cudaGetErrorString(e), where);
}

// ---- private scratch pool (one per device, created on first use) ---------------------------------------------------
static std::mutex g_pool_mu;
static cudaMemPool_t g_pools[64] = {};

static cudaError_t get_pool(cudaMemPool_t *out) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lk(g_pool_mu);
    if (!g_pools[dev]) {
        cudaMemPoolProps props = {};
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        e = cudaMemPoolCreate(&g_pools[dev], &props);
        if (e != cudaSuccess) { g_pools[dev] = nullptr; return e; }
        unsigned long long keep = ~0ull;          // keep freed blocks until ppfm_release_scratch()
        cudaMemPoolSetAttribute(g_pools[dev], cudaMemPoolAttrReleaseThreshold, &keep);
    }
    *out = g_pools[dev];
    return cudaSuccess;
}

cudaError_t scratch_alloc(void **ptr, size_t bytes, cudaStream_t st) {
    cudaMemPool_t pool;
    cudaError_t e = get_pool(&pool);
    if (e != cudaSuccess) return e;
    return cudaMallocFromPoolAsync(ptr, bytes ? bytes : 1, pool, st);
}

// ---- per-kernel timing ---------------------------------------------------------------------------------------------
struct PendingTiming { int id; cudaEvent_t e0, e1; };
static std::mutex g_tm_mu;
static std::vector<PendingTiming> g_tm_pending;
static double g_tm_ms[PPFM_K_COUNT] = {};
static long long g_tm_n[PPFM_K_COUNT] = {};

void timing_begin(int, cudaStream_t st, cudaEvent_t *e0) {
    if (cudaEventCreate(e0) != cudaSuccess) { *e0 = nullptr; return; }
    cudaEventRecord(*e0, st);
}

void timing_end(int kernel_id, cudaStream_t st, cudaEvent_t e0) {
    if (!e0) return;
    cudaEvent_t e1;
    if (cudaEventCreate(&e1) != cudaSuccess) { cudaEventDestroy(e0); return; }
    cudaEventRecord(e1, st);
    std::lock_guard<std::mutex> lk(g_tm_mu);
    g_tm_pending.push_back({kernel_id, e0, e1});
}

static void timing_drain(bool accumulate) {
    std::lock_guard<std::mutex> lk(g_tm_mu);
    for (auto &p : g_tm_pending) {
        if (accumulate && cudaEventSynchronize(p.e1) == cudaSuccess) {
            float ms = 0.f;
            if (cudaEventElapsedTime(&ms, p.e0, p.e1) == cudaSuccess && p.id >= 0 && p.id < PPFM_K_COUNT) {
                g_tm_ms[p.id] += ms;
                g_tm_n[p.id] += 1;
            }
        }
        cudaEventDestroy(p.e0);
        cudaEventDestroy(p.e1);
    }
    g_tm_pending.clear();
}

// ---- probe 1: FP32 FMA issue rate (the denominator of the force-field kernel's pipe utilisation) ----------------
__global__ void __launch_bounds__(256) probe_fma_kernel(float *out, int iters, float a, float b) {
    float x[16];
#pragma unroll
    for (int i = 0; i < 16; i++) x[i] = (float)(threadIdx.x + i);
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int r = 0; r < 8; r++) {
#pragma unroll
            for (int i = 0; i < 16; i++) x[i] = fmaf(x[i], a, b);
        }
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 16; i++) s += x[i];
    if (s == 123.456f) out[0] = s;   // never true for the arguments used; defeats dead-code elimination
}

// ---- probe 2: the relaxation's gather pattern with no dependent math ("achievable L2 bandwidth") ------------------
// A warp covers an 8 x 4 pixel patch (as relax_kernel does); each step it gathers the 8 corners of a cell of an
// nx x ny x nz float4 volume and moves to a pseudo-random neighbouring cell that does NOT depend on loaded data.
template <bool BYPASS_L1>
__global__ void __launch_bounds__(128) probe_gather_kernel(const float4 *__restrict__ g, int nx, int ny, int nz,
                                                           int steps, float *out) {
    const int warp_global = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    unsigned s = 0x9E3779B9u * (warp_global + 1);
    float acc = 0.f;
    for (int it = 0; it < steps; it++) {
        s = s * 1664525u + 1013904223u;
        const int bx = (int)((s >> 8) % (unsigned)(nx - 9));
        const int by = (int)((s >> 4) % (unsigned)(ny - 5));
        const int bz = (int)((s >> 16) % (unsigned)(nz - 1));
        const int i0 = bx + (lane & 7), j0 = by + (lane >> 3), k0 = bz;
#pragma unroll
        for (int c = 0; c < 8; c++) {
            const int i = i0 + (c & 1), j = j0 + ((c >> 1) & 1), k = k0 + (c >> 2);
            const float4 *p = g + ((size_t)k * ny + j) * nx + i;
            float4 v;
            if (BYPASS_L1) {
                asm volatile("ld.global.cg.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
            } else {
                v = __ldg(p);
            }
            acc += v.x + v.w;
        }
    }
    if (acc == 123.456f) out[0] = acc;
}

__global__ void probe_fill_kernel(float4 *g, long long n) {
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride)
        g[i] = make_float4(1e-3f * (float)(i & 1023), 0.f, 1.f, 2.f);
}

}  // namespace ppfm

using namespace ppfm;

extern "C" int ppfm_version(void) { return PPFM_VERSION; }

extern "C" const char *ppfm_strerror(int code) {
    switch (code) {
        case PPFM_OK: return "ok";
        case PPFM_EINVAL: return "invalid argument";
        case PPFM_ECUDA: return g_cuda_msg;
        case PPFM_ENOMEM: return "device scratch allocation failed";
        default: return "unknown status";
    }
}

extern "C" void ppfm_fire_default(ppfm_fire *out) {
    if (!out) return;
    out->dt = 0.5; out->dt_max = 0.5; out->finc = 1.1; out->fdec = 0.5; out->alpha0 = 0.1; out->falpha = 0.99;
    out->n_min = 5; out->max_iter = 1000; out->f_conv = 1e-6;
}

extern "C" double ppfm_Nm_to_eVA2(double k_Nm) { return k_Nm / kEVA2toNm; }

extern "C" int64_t ppfm_launch_count(void) { return (int64_t)g_launches.load(); }

extern "C" int ppfm_timing_enable(int on) {
    timing_drain(false);
    {
        std::lock_guard<std::mutex> lk(g_tm_mu);
        for (int k = 0; k < PPFM_K_COUNT; k++) { g_tm_ms[k] = 0.0; g_tm_n[k] = 0; }
    }
    g_timing_on.store(on ? 1 : 0);
    return PPFM_OK;
}

extern "C" int ppfm_timing_read(int kernel_id, double *h_ms_total, int64_t *h_launches) {
    if (kernel_id < 0 || kernel_id >= PPFM_K_COUNT || !h_ms_total || !h_launches) return PPFM_EINVAL;
    timing_drain(true);
    std::lock_guard<std::mutex> lk(g_tm_mu);
    *h_ms_total = g_tm_ms[kernel_id];
    *h_launches = (int64_t)g_tm_n[kernel_id];
    return PPFM_OK;
}

extern "C" int ppfm_release_scratch(void) {
    release_fft_plans();
    int dev = 0;
    PPFM_CUDA(cudaGetDevice(&dev));
    std::lock_guard<std::mutex> lk(g_pool_mu);
    if (dev >= 0 && dev < 64 && g_pools[dev]) PPFM_CUDA(cudaMemPoolTrimTo(g_pools[dev], 0));
    return PPFM_OK;
}

// Device-side alias of a host buffer, if it is pinned/registered (UVA-mapped) memory; nullptr for pageable memory.
static void *mapped_alias(const void *h) {
    if (!h) return nullptr;
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, h) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    return (a.type == cudaMemoryTypeHost) ? a.devicePointer : nullptr;
}

// One call, host buffers ("run the whole simulation in one step").  When the output buffers are pinned
// host memory the kernels store straight into them (posted PCIe writes that overlap the computation: no
// device-to-host copy of the float4 stack and of df after the scan); the relaxation then also keeps a plain Fz stack on
// the device for the df kernel.  The uint16 iteration counts go through a device buffer and one DMA copy: written in
// place they are 16-byte PCIe writes, which slow the relaxation more than the 2 bytes per sample are worth.
// Pageable outputs take staged cudaMemcpyAsync copies.
static int scan_host_impl(int nsys, const int32_t *h_atom_offset, const float *h_xyzq, const int32_t *h_type,
                          int32_t ntypes, const double *h_R, const double *h_e, const ppfm_lattice *lattices,
                          const ppfm_probe *probes, const ppfm_grid *grids, double r_min, const ppfm_tip *tips,
                          const ppfm_fire *fire, const ppfm_scan *scans, double A, double k0_Nm, double f0_Hz,
                          float *h_pos_fz, uint16_t *h_iters, float *h_df, ppfm_stats *h_stats, void *cuda_stream,
                          int nQ = 0, const double *h_Q = nullptr) {
    if (nsys < 1 || !h_atom_offset || !grids || !scans || !tips || !fire || !lattices || !probes) return PPFM_EINVAL;
    if (nQ < 0 || (nQ > 0 && (!h_Q || nsys != 1))) return PPFM_EINVAL;      // the Q sweep is a single-system form
    const int nrun = nQ > 0 ? nQ : 1;
    const int natoms = h_atom_offset[nsys];
    if (natoms < 0 || h_atom_offset[0] != 0 || (natoms > 0 && (!h_xyzq || !h_type))) return PPFM_EINVAL;
    size_t npts = 0, nps = 0;
    for (int m = 0; m < nsys; m++) {
        if (!grid_ok(&grids[m]) || scans[m].npx < 1 || scans[m].npy < 1 || scans[m].nz < 1) return PPFM_EINVAL;
        if (h_df && (scans[m].npx != scans[0].npx || scans[m].npy != scans[0].npy || scans[m].nz != scans[0].nz ||
                     scans[m].dz != scans[0].dz))
            return PPFM_EINVAL;                        // the df batch takes stacks of one shape
        npts += (size_t)grid_points(&grids[m]);
        nps += (size_t)scans[m].npx * scans[m].npy * scans[m].nz;
    }
    const ppfm_scan *scan = &scans[0];
    const double nn = (scan->dz > 0) ? A / scan->dz : -1.0;
    const long long n = std::llround(nn);
    if (h_df && (n < 1 || std::fabs(nn - (double)n) > 1e-6 || scan->nz <= n)) return PPFM_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t ndf = h_df ? (size_t)nsys * scan->npx * scan->npy * (size_t)(scan->nz - n) : 0;
    const size_t na = (size_t)(natoms > 0 ? natoms : 1);
    // zero-copy outputs?
    float *m_pos = (float *)mapped_alias(h_pos_fz);
    uint16_t *m_it = (uint16_t *)mapped_alias(h_iters);
    float *m_df = (float *)mapped_alias(h_df);
    const bool zc = h_pos_fz && m_pos && (!h_iters || m_it) && (!h_df || m_df);
    float *d_xyzq = nullptr, *d_ff = nullptr, *d_pos = nullptr, *d_df = nullptr, *d_fz = nullptr;
    float *d_lj = nullptr, *d_el = nullptr;
    int32_t *d_type = nullptr;
    uint16_t *d_it = nullptr;
    ppfm_stats *d_stats = nullptr;
    int rc = PPFM_OK;
    auto fail = [&](cudaError_t e, const char *w) { set_cuda_error(e, w); rc = (e == cudaErrorMemoryAllocation) ? PPFM_ENOMEM : PPFM_ECUDA; };
    cudaError_t e;
#define TRY(x) if (rc == PPFM_OK && (e = (x)) != cudaSuccess) fail(e, #x)
    TRY(scratch_alloc((void **)&d_xyzq, na * 16, st));
    TRY(scratch_alloc((void **)&d_type, na * 4, st));
    TRY(scratch_alloc((void **)&d_ff, npts * 16, st));
    if (nQ > 0) {
        TRY(scratch_alloc((void **)&d_lj, npts * 16, st));
        TRY(scratch_alloc((void **)&d_el, npts * 16, st));
    }
    TRY(scratch_alloc((void **)&d_stats, sizeof(ppfm_stats), st));
    if (zc) {
        if (h_df) TRY(scratch_alloc((void **)&d_fz, nps * 4, st));
        if (h_iters) TRY(scratch_alloc((void **)&d_it, nps * 2, st));
    } else {
        TRY(scratch_alloc((void **)&d_pos, nps * 16, st));
        TRY(scratch_alloc((void **)&d_it, nps * 2, st));
        if (h_df) TRY(scratch_alloc((void **)&d_df, ndf * 4, st));
    }
    if (natoms > 0) {
        TRY(cudaMemcpyAsync(d_xyzq, h_xyzq, (size_t)natoms * 16, cudaMemcpyHostToDevice, st));
        TRY(cudaMemcpyAsync(d_type, h_type, (size_t)natoms * 4, cudaMemcpyHostToDevice, st));
    }
    TRY(cudaMemsetAsync(d_stats, 0, sizeof(ppfm_stats), st));
    if (rc == PPFM_OK) {
        if (nQ > 0)          // S19: F_LJ and unit-charge F_el once, combined per Q
            rc = ppfm_forcefield_split(natoms, d_xyzq, d_type, ntypes, h_R, h_e, lattices, probes, grids, r_min, d_lj,
                                       d_el, cuda_stream);
        else
            rc = (nsys == 1) ? ppfm_forcefield(natoms, d_xyzq, d_type, ntypes, h_R, h_e, lattices, probes, grids, r_min,
                                               d_ff, cuda_stream)
                             : ppfm_forcefield_batch(nsys, h_atom_offset, d_xyzq, d_type, ntypes, h_R, h_e, lattices,
                                                     probes, grids, r_min, d_ff, cuda_stream);
    }
    for (int run = 0; run < nrun; run++) {
        if (rc == PPFM_OK && nQ > 0) rc = ppfm_combine(d_lj, d_el, h_Q[run], (int64_t)npts, d_ff, cuda_stream);
        const size_t op = (size_t)run * nps, od = (size_t)run * ndf;      // this run's slice of the host outputs
        if (zc) {
            if (rc == PPFM_OK)
                rc = relax_scan_fz(nsys, d_ff, grids, tips, fire, scans, m_pos + 4 * op, h_iters ? d_it : nullptr,
                                   d_stats, d_fz, cuda_stream);
            if (h_iters) TRY(cudaMemcpyAsync(h_iters + op, d_it, nps * 2, cudaMemcpyDeviceToHost, st));
            if (rc == PPFM_OK && h_df)
                rc = df_from_fz(nsys, d_fz, scan->npx, scan->npy, scan->nz, scan->dz, A, k0_Nm, f0_Hz, m_df + od,
                                cuda_stream);
        } else {
            if (rc == PPFM_OK)
                rc = relax_scan_fz(nsys, d_ff, grids, tips, fire, scans, d_pos, d_it, d_stats, nullptr, cuda_stream);
            if (rc == PPFM_OK && h_df)
                rc = ppfm_df_batch(nsys, d_pos, scan->npx, scan->npy, scan->nz, scan->dz, A, k0_Nm, f0_Hz, d_df,
                                   cuda_stream);
            if (h_pos_fz) TRY(cudaMemcpyAsync(h_pos_fz + 4 * op, d_pos, nps * 16, cudaMemcpyDeviceToHost, st));
            if (h_iters) TRY(cudaMemcpyAsync(h_iters + op, d_it, nps * 2, cudaMemcpyDeviceToHost, st));
            if (h_df) TRY(cudaMemcpyAsync(h_df + od, d_df, ndf * 4, cudaMemcpyDeviceToHost, st));
        }
    }
    if (h_stats) TRY(cudaMemcpyAsync(h_stats, d_stats, sizeof(ppfm_stats), cudaMemcpyDeviceToHost, st));
#undef TRY
    void *bufs[] = {d_xyzq, d_type, d_ff, d_pos, d_it, d_stats, d_df, d_fz, d_lj, d_el};
    for (void *b : bufs)
        if (b) cudaFreeAsync(b, st);
    e = cudaStreamSynchronize(st);
    if (rc == PPFM_OK && e != cudaSuccess) fail(e, "cudaStreamSynchronize");
    return rc;
}

extern "C" int ppfm_scan_host(int32_t natoms, const float *h_xyzq, const int32_t *h_type, int32_t ntypes,
                              const double *h_R, const double *h_e, const ppfm_lattice *lattice,
                              const ppfm_probe *probe, const ppfm_grid *grid, double r_min, const ppfm_tip *tip,
                              const ppfm_fire *fire, const ppfm_scan *scan, double A, double k0_Nm, double f0_Hz,
                              float *h_pos_fz, uint16_t *h_iters, float *h_df, ppfm_stats *h_stats,
                              void *cuda_stream) {
    if (natoms < 0) return PPFM_EINVAL;
    const int32_t off[2] = {0, natoms};
    return scan_host_impl(1, off, h_xyzq, h_type, ntypes, h_R, h_e, lattice, probe, grid, r_min, tip, fire, scan, A,
                          k0_Nm, f0_Hz, h_pos_fz, h_iters, h_df, h_stats, cuda_stream);
}

extern "C" int ppfm_scan_host_batch(int32_t nsys, const int32_t *h_atom_offset, const float *h_xyzq,
                                    const int32_t *h_type, int32_t ntypes, const double *h_R, const double *h_e,
                                    const ppfm_lattice *lattices, const ppfm_probe *probes, const ppfm_grid *grids,
                                    double r_min, const ppfm_tip *tips, const ppfm_fire *fire, const ppfm_scan *scans,
                                    double A, double k0_Nm, double f0_Hz, float *h_pos_fz, uint16_t *h_iters,
                                    float *h_df, ppfm_stats *h_stats, void *cuda_stream) {
    return scan_host_impl(nsys, h_atom_offset, h_xyzq, h_type, ntypes, h_R, h_e, lattices, probes, grids, r_min, tips,
                          fire, scans, A, k0_Nm, f0_Hz, h_pos_fz, h_iters, h_df, h_stats, cuda_stream);
}

extern "C" int ppfm_probe_fma(double *h_lane_instr_per_s, void *cuda_stream) {
    if (!h_lane_instr_per_s) return PPFM_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0;
    PPFM_CUDA(cudaGetDevice(&dev));
    PPFM_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    float *d_out = nullptr;
    PPFM_CUDA(cudaMallocAsync((void **)&d_out, 4, st));
    cudaEvent_t e0, e1;
    PPFM_CUDA(cudaEventCreate(&e0));
    PPFM_CUDA(cudaEventCreate(&e1));
    const int iters = 4000, blocks = sms * 8;
    double best = 0.0;
    for (int rep = 0; rep < 4; rep++) {
        PPFM_CUDA(cudaEventRecord(e0, st));
        probe_fma_kernel<<<blocks, 256, 0, st>>>(d_out, iters, 0.999f, 0.001f);
        PPFM_LAUNCH_CHECK();
        PPFM_CUDA(cudaEventRecord(e1, st));
        PPFM_CUDA(cudaEventSynchronize(e1));
        float ms = 0.f;
        PPFM_CUDA(cudaEventElapsedTime(&ms, e0, e1));
        const double lane_instr = (double)blocks * 256.0 * (double)iters * 8.0 * 16.0;
        const double rate = lane_instr / (ms * 1e-3);
        if (rep > 0 && rate > best) best = rate;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    PPFM_CUDA(cudaFreeAsync(d_out, st));
    PPFM_CUDA(cudaStreamSynchronize(st));
    *h_lane_instr_per_s = best;
    return PPFM_OK;
}

extern "C" int ppfm_probe_gather(int64_t n_float4, int32_t bypass_l1, double *h_gbs, void *cuda_stream) {
    if (!h_gbs || n_float4 < 64 * 64 * 8) return PPFM_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0;
    PPFM_CUDA(cudaGetDevice(&dev));
    PPFM_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    // volume nx = ny = 256, nz from the requested size (plane = 1 MiB)
    const int nx = 256, ny = 256;
    long long nzl = n_float4 / ((long long)nx * ny);
    if (nzl < 2) nzl = 2;
    if (nzl > 8192) nzl = 8192;
    const int nz = (int)nzl;
    const long long n = (long long)nx * ny * nz;
    float4 *d_g = nullptr;
    float *d_out = nullptr;
    PPFM_CUDA(cudaMallocAsync((void **)&d_g, (size_t)n * 16, st));
    PPFM_CUDA(cudaMallocAsync((void **)&d_out, 4, st));
    probe_fill_kernel<<<sms * 8, 256, 0, st>>>(d_g, n);
    PPFM_LAUNCH_CHECK();
    cudaEvent_t e0, e1;
    PPFM_CUDA(cudaEventCreate(&e0));
    PPFM_CUDA(cudaEventCreate(&e1));
    const int steps = 2000, blocks = sms * 16;
    double best = 0.0;
    for (int rep = 0; rep < 4; rep++) {
        PPFM_CUDA(cudaEventRecord(e0, st));
        if (bypass_l1)
            probe_gather_kernel<true><<<blocks, 128, 0, st>>>(d_g, nx, ny, nz, steps, d_out);
        else
            probe_gather_kernel<false><<<blocks, 128, 0, st>>>(d_g, nx, ny, nz, steps, d_out);
        PPFM_LAUNCH_CHECK();
        PPFM_CUDA(cudaEventRecord(e1, st));
        PPFM_CUDA(cudaEventSynchronize(e1));
        float ms = 0.f;
        PPFM_CUDA(cudaEventElapsedTime(&ms, e0, e1));
        const double bytes = (double)blocks * 128.0 * (double)steps * 128.0;
        const double gbs = bytes / (ms * 1e-3) * 1e-9;
        if (rep > 0 && gbs > best) best = gbs;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    PPFM_CUDA(cudaFreeAsync(d_g, st));
    PPFM_CUDA(cudaFreeAsync(d_out, st));
    PPFM_CUDA(cudaStreamSynchronize(st));
    *h_gbs = best;
    return PPFM_OK;
}

extern "C" int ppfm_scan_host_sweep(int32_t nQ, const double *h_Q, int32_t natoms, const float *h_xyzq,
                                    const int32_t *h_type, int32_t ntypes, const double *h_R, const double *h_e,
                                    const ppfm_lattice *lattice, const ppfm_probe *probe, const ppfm_grid *grid,
                                    double r_min, const ppfm_tip *tip, const ppfm_fire *fire, const ppfm_scan *scan,
                                    double A, double k0_Nm, double f0_Hz, float *h_pos_fz, uint16_t *h_iters,
                                    float *h_df, ppfm_stats *h_stats, void *cuda_stream) {
    if (natoms < 0 || nQ < 1) return PPFM_EINVAL;
    const int32_t off[2] = {0, natoms};
    return scan_host_impl(1, off, h_xyzq, h_type, ntypes, h_R, h_e, lattice, probe, grid, r_min, tip, fire, scan, A,
                          k0_Nm, f0_Hz, h_pos_fz, h_iters, h_df, h_stats, cuda_stream, nQ, h_Q);
}
