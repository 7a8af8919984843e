/*
 * ppfm_bench.h — measurement interface of libppfm, kept apart from the product ABI (include/ppfm.h).
 *
 * Two parts:
 *   (a) launch counting and per-kernel device timing, exported by libppfm.so itself (they bracket its launches);
 *   (b) two micro-benchmarks that define roofline denominators on the box, exported by a separate small library,
 *       libppfm_probes.so (paper_2401_14564_b200/csrc_probes/probes.cu), which the product never loads.
 * Used by bench.py and the tests only.
 */
#ifndef PPFM_BENCH_H
#define PPFM_BENCH_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* ---- (a) exported by libppfm.so ------------------------------------------------------------------------------ */
/* Number of kernels this library has launched on this process so far (for bench.py's gpu_launches). */
int64_t ppfm_launch_count(void);

/* Per-kernel device timing for the roofline legs of bench.py: while enabled, every launch of the kernels below is
 * bracketed by CUDA events recorded on the launching stream directly around the launch (no host work in between).
 * ppfm_timing_enable(on) clears the accumulators; ppfm_timing_read waits for the recorded events of `kernel_id`
 * (it synchronises on them, not on the stream) and returns the summed milliseconds and the number of launches.
 * Off by default; process-wide. */
typedef enum {
    PPFM_K_FF_PREP = 0, /* a1 atom-record packing            */
    PPFM_K_FF = 1,      /* a2 force-field grid               */
    PPFM_K_COMBINE = 2, /* a3 F_LJ + Q F_el                  */
    PPFM_K_RELAX = 3,   /* a4+a5 relaxation scan             */
    PPFM_K_DF = 4,      /* a6 frequency shift                */
    PPFM_K_STIFFNESS = 5, /* N2 stiffness map               */
    PPFM_K_FFT_EL = 6,  /* N3 Eq.7 electrostatics: own kernels + cuFFT, one timed region */
    PPFM_K_RELAX_TRICUBIC = 7, /* N4 relaxation with tri-cubic interpolation of the potential */
    PPFM_K_FF_ENERGY = 8, /* N4 energy-only force-field pass (ppfm_forcefield_energy) */
    PPFM_K_COUNT = 9
} ppfm_kernel_id;
int ppfm_timing_enable(int on);
int ppfm_timing_read(int kernel_id, double *h_ms_total, int64_t *h_launches);

/* Checked build only (libppfm_chk.so = the same sources compiled with -DPPFM_CHECKS; stands in for compute-sanitizer,
 * which is closed on the GPU pool this library is developed on).  The kernels then test every global store and gather
 * index against its buffer's extent and compare each stage of ff_kernel's shared-memory atom ring with the global
 * records when the stage is acquired and again when it is released.  ppfm_checks_read synchronises the device, writes
 * the counts since the last call to h_counts[8] and clears them:
 *   [0] ring stage wrong at acquire (read before the copy landed)   [1] ring stage changed before release (overwritten
 *   in use)   [2] force-field store out of range   [3] relaxation gather out of range   [4] relaxation store out of
 *   range   [5] df load out of range   [6] df store out of range   [7] checks executed.
 * The product build (libppfm.so) returns PPFM_EINVAL. */
int ppfm_checks_read(uint64_t *h_counts);

/* ---- (b) exported by libppfm_probes.so ------------------------------------------------------------------------
 * ppfm_probe_fma:    FFMA-only kernel; returns lane-instructions per second in *h_lane_instr_per_s.
 * ppfm_probe_gather: the relaxation's 8-corner float4 gather (a warp = 8 x 4 neighbouring cells) over an L2-resident
 *                    volume of `n_float4` entries with no dependent math; `bypass_l1` != 0 selects ld.global.cg (every
 *                    request goes to L2: "achievable L2 bandwidth"), 0 selects ld.global.nc through L1, where most
 *                    of the 8 overlapping corners of neighbouring lanes hit (an L1-assisted figure); returns GB/s.
 * Both synchronise the stream (they time with CUDA events) and return 0 or a negative status.
 */
int ppfm_probe_fma(double *h_lane_instr_per_s, void *cuda_stream);
int ppfm_probe_gather(int64_t n_float4, int32_t bypass_l1, double *h_gbs, void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* PPFM_BENCH_H */
