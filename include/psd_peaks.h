/*
 * psd_peaks.h -- C ABI of libpsd_peaks: micro-benchmarks for the roofline denominators that
 * MEASURED_PEAKS.json does not hold (it has HBM copy bandwidth and bf16 GEMM only).
 *
 * The deposit path (include/psd.h) is branchy scalar fp64 geometry plus
 * fp64 atomics, so its rooflines are the FP64 pipe, the shared-memory fp64 atomic rate and the L2
 * fp64 reduction rate (BASELINE.json north_star: "the slower of clip FLOPs at FP pipe peak, bytes
 * at HBM peak, and atomics at L2 atomic rate").  Each call launches a saturating kernel on
 * `device` (stream `cuda_stream`, NULL = default), times `reps` launches with CUDA events after
 * one warm-up launch, and writes the BEST rate to *out.  Returns 0 on success, 1 on a bad
 * argument, 4 on a CUDA error.  Nothing here is on the deposit path.
 */
#ifndef PSD_PEAKS_H
#define PSD_PEAKS_H

#if defined(__GNUC__)
#define PSD_PEAKS_API __attribute__((visibility("default")))
#else
#define PSD_PEAKS_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

/* dependent-chain-free DFMA stream, all SMs: *out = FLOP/s (2 per FMA). */
PSD_PEAKS_API int psd_peak_fp64_fma(int device, void* cuda_stream, int reps, double* out);
/* same with FFMA: *out = FLOP/s. */
PSD_PEAKS_API int psd_peak_fp32_fma(int device, void* cuda_stream, int reps, double* out);
/* atomicAdd(double) on shared memory, every lane of a warp a different cell of the CTA's 8^3
 * tile (the accumulate pattern of the tile deposit): *out = atomics/s over the chip. */
PSD_PEAKS_API int psd_peak_shared_atomic_f64(int device, void* cuda_stream, int reps, double* out);
/* red.global.add.f64 (atomicAdd without use of the result):
 *   pattern 0: the flush pattern -- each CTA adds an 8x8x8 tile into a 256^3 grid, 8 consecutive
 *              doubles per row;  pattern 1: every lane a different 128-byte line of a 1 GiB
 *              buffer (worst case, one sector per atomic).   *out = atomics/s. */
PSD_PEAKS_API int psd_peak_global_red_f64(int device, void* cuda_stream, int pattern, int reps, double* out);

#ifdef __cplusplus
}
#endif
#endif /* PSD_PEAKS_H */
