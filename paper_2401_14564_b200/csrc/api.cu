// api.cu — the rest of the C ABI: status text, defaults, scratch pool, the one-call host-buffer simulation
// and the launch counter / per-kernel timers of include/ppfm_bench.h.
#include "common.cuh"

#include <mutex>
#include <vector>

namespace ppfm {

std::atomic<long long> g_launches{0};
std::atomic<int> g_timing_on{0};
static thread_local char g_cuda_msg[256] = "no CUDA error recorded";

void set_cuda_error(cudaError_t e, const char *where) {
    snprintf(g_cuda_msg, sizeof(g_cuda_msg), "CUDA error %d (%s) in %s", (int)e, cudaGetErrorString(e), where);
    cudaGetLastError();      // clear the thread's sticky-less last-error state: one failed call must not make the
                             // next successful launch report a stale error through PPFM_LAUNCH_CHECK
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

}  // namespace ppfm

using namespace ppfm;

extern "C" int ppfm_version(void) { return PPFM_VERSION; }

extern "C" const char *ppfm_strerror(int code) {
    switch (code) {
        case PPFM_OK: return "ok";
        case PPFM_EINVAL: return "invalid argument";
        case PPFM_ECUDA: return g_cuda_msg;
        case PPFM_ENOMEM: return "device scratch allocation failed";
        case PPFM_ELIMIT: return "input exceeds the fixed scratch of a no-allocation entry point (natoms > PPFM_NOALLOC_MAX_ATOMS)";
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

extern "C" int ppfm_checks_read(uint64_t *h_counts) {
#ifdef PPFM_CHECKS
    if (!h_counts) return PPFM_EINVAL;
    unsigned long long c[PPFM_CHK_KINDS] = {};
    ff_checks_read(c);
    relax_checks_read(c);
    df_checks_read(c);
    for (int k = 0; k < PPFM_CHK_KINDS; k++) h_counts[k] = (uint64_t)c[k];
    return PPFM_OK;
#else
    (void)h_counts;
    return PPFM_EINVAL;      // not a checked build
#endif
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
    if (h_df && (n < 1 || n > PPFM_DF_MAX_N || std::fabs(nn - (double)n) > 1e-6 || scan->nz <= n)) return PPFM_EINVAL;
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
    // Q sweep (S19): the nQ combined grids are kept side by side and the nQ scans run as ONE batch launch (a single
    // 200 x 200 scan cannot fill the GPU: 1250 warps on 592 sub-partitions; three at once can), as long as the grids fit
    // the budget below; otherwise one scan after the other on one combined grid.
    const size_t sweep_budget = (size_t)8 << 30;
    const bool sweep_batched = nQ > 1 && (size_t)nQ * npts * 16 <= sweep_budget;
    const size_t nff = sweep_batched ? (size_t)nQ : 1;
    TRY(scratch_alloc((void **)&d_ff, nff * npts * 16, st));
    if (nQ > 0) {
        TRY(scratch_alloc((void **)&d_lj, npts * 16, st));
        TRY(scratch_alloc((void **)&d_el, npts * 16, st));
    }
    TRY(scratch_alloc((void **)&d_stats, sizeof(ppfm_stats), st));
    if (zc) {
        if (h_df) TRY(scratch_alloc((void **)&d_fz, nff * nps * 4, st));
        if (h_iters) TRY(scratch_alloc((void **)&d_it, nff * nps * 2, st));
    } else {
        TRY(scratch_alloc((void **)&d_pos, nff * nps * 16, st));
        TRY(scratch_alloc((void **)&d_it, nff * nps * 2, st));
        if (h_df) TRY(scratch_alloc((void **)&d_df, nff * ndf * 4, st));
    }
    if (natoms > 0) {
        TRY(cudaMemcpyAsync(d_xyzq, h_xyzq, (size_t)natoms * 16, cudaMemcpyHostToDevice, st));
        TRY(cudaMemcpyAsync(d_type, h_type, (size_t)natoms * 4, cudaMemcpyHostToDevice, st));
    }
    TRY(cudaMemsetAsync(d_stats, 0, sizeof(ppfm_stats), st));
    if (rc == PPFM_OK) {
        if (nQ > 0)          // S19: F_LJ and unit-charge F_el once, combined per Q
            rc = ppfm_forcefield_split(natoms, d_xyzq, d_type, ntypes, h_R, h_e, lattices, probes, grids, r_min, d_lj,
                                       d_el, nullptr, cuda_stream);
        else
            rc = (nsys == 1) ? ppfm_forcefield(natoms, d_xyzq, d_type, ntypes, h_R, h_e, lattices, probes, grids, r_min,
                                               d_ff, nullptr, cuda_stream)
                             : ppfm_forcefield_batch(nsys, h_atom_offset, d_xyzq, d_type, ntypes, h_R, h_e, lattices,
                                                     probes, grids, r_min, d_ff, nullptr, cuda_stream);
    }
    // one pass of (relaxation, df, copies) over `nb` systems laid out consecutively (grids at d_ff) that together make
    // `sets` result sets of nps pixel-steps / ndf df samples, written at the host offsets op / od
    auto scan_pass = [&](int nb, const ppfm_grid *g, const ppfm_tip *t, const ppfm_scan *sc, size_t sets, size_t op, size_t od) {
        const size_t tot_ps = sets * nps, tot_df = sets * ndf;
        if (zc) {
            if (rc == PPFM_OK)
                rc = relax_scan_fz(nb, d_ff, g, t, fire, sc, m_pos + 4 * op, h_iters ? d_it : nullptr, d_stats, d_fz,
                                   cuda_stream);
            if (h_iters) TRY(cudaMemcpyAsync(h_iters + op, d_it, tot_ps * 2, cudaMemcpyDeviceToHost, st));
            if (rc == PPFM_OK && h_df)
                rc = df_from_fz(nb, d_fz, scan->npx, scan->npy, scan->nz, scan->dz, A, k0_Nm, f0_Hz, m_df + od,
                                cuda_stream);
        } else {
            if (rc == PPFM_OK)
                rc = relax_scan_fz(nb, d_ff, g, t, fire, sc, d_pos, d_it, d_stats, nullptr, cuda_stream);
            if (rc == PPFM_OK && h_df)
                rc = ppfm_df_batch(nb, d_pos, scan->npx, scan->npy, scan->nz, scan->dz, A, k0_Nm, f0_Hz, d_df,
                                   cuda_stream);
            if (h_pos_fz) TRY(cudaMemcpyAsync(h_pos_fz + 4 * op, d_pos, tot_ps * 16, cudaMemcpyDeviceToHost, st));
            if (h_iters) TRY(cudaMemcpyAsync(h_iters + op, d_it, tot_ps * 2, cudaMemcpyDeviceToHost, st));
            if (h_df) TRY(cudaMemcpyAsync(h_df + od, d_df, tot_df * 4, cudaMemcpyDeviceToHost, st));
        }
    };
    if (sweep_batched) {
        std::vector<ppfm_grid> gs((size_t)nQ, grids[0]);
        std::vector<ppfm_tip> ts((size_t)nQ, tips[0]);
        std::vector<ppfm_scan> ss((size_t)nQ, scans[0]);
        for (int run = 0; run < nQ; run++)
            if (rc == PPFM_OK)
                rc = ppfm_combine(d_lj, d_el, h_Q[run], (int64_t)npts, d_ff + (size_t)run * npts * 4, cuda_stream);
        scan_pass(nQ, gs.data(), ts.data(), ss.data(), (size_t)nQ, 0, 0);   // nsys == 1: nQ systems = nQ result sets
    } else {
        for (int run = 0; run < nrun; run++) {
            if (rc == PPFM_OK && nQ > 0) rc = ppfm_combine(d_lj, d_el, h_Q[run], (int64_t)npts, d_ff, cuda_stream);
            scan_pass(nsys, grids, tips, scans, 1, (size_t)run * nps, (size_t)run * ndf);   // this run's slice of the outputs
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
