/* qsl_peaks.h - roofline denominators measured on the device (bench utilities; NOT part of libqsl).
 *
 * SURVEY.md 8(d) "Which roofline binds": MEASURED_PEAKS.json carries only the HBM copy bandwidth and the bf16 GEMM rate,
 * so the two peaks that bound the field-line tracer are measured by two micro-kernels of their own, built into
 * libqsl_peaks.so (paper_1609_00724_b200/peaks/peaks.cu).  The library shares no code with libqsl.so and nothing of the
 * method is in it; bench.py is its only caller.
 *
 * Both calls time themselves with CUDA events (2 warm-up launches, best of `reps`) on `stream` (a cudaStream_t passed as
 * void*) and synchronise it.  Results are written to HOST memory.  Return 0 or one of the codes below.                 */
#ifndef QSL_PEAKS_H
#define QSL_PEAKS_H
#ifdef __cplusplus
extern "C" {
#endif

#define QSL_PEAKS_EINVAL (-1)
#define QSL_PEAKS_ENOMEM (-2)
#define QSL_PEAKS_ECUDA  (-3)

/* fma_per_s (host): fused multiply-adds per second of the plain FP pipe, fp64 != 0 -> DFMA, else FFMA, from 8
 * independent register-only chains per thread, 8 blocks of 256 threads per SM.                                        */
int qsl_peak_fma(int fp64, int reps, double *fma_per_s, void *stream);
/* samples_per_s (host): divergent pseudo-random gathers per second of one 16-byte (float4) or 32-byte (double4) sample
 * per lane over a zero-filled device buffer of footprint_bytes (>= 4096, rounded down to a power of two; allocated and
 * freed by the call), i.e. the tracer's load shape with an L1-, L2- or HBM-resident field.                             */
int qsl_peak_gather(int bytes_per_sample, long long footprint_bytes, int reps, double *samples_per_s, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* QSL_PEAKS_H */
