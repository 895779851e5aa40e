/*
 * pwfs_peak.h -- C ABI of libpwfs_peak.so: a measurement aid that ships beside libpwfs.so,
 * not inside it.  bench.py loads it to measure the FP32 roofline denominator on the box
 * it runs on; the sensor library and its users never need it.
 */
#ifndef PWFS_PEAK_H
#define PWFS_PEAK_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* The FP32 arithmetic peak of `device`
 * as a stream of independent FFMA (packed = 0) or packed FFMA2 (packed = 1)
 * instructions on every SM (64 resident warps each, 8 independent accumulator
 * pairs per thread), best of five launches of ~10^12 flop, timed with CUDA events.
 * *tflops counts an FMA as 2 flop.  This is the measured counterpart of the
 * derived "148 SMs x 128 lanes x 2 x f_SM" roofline denominator that SURVEY.md
 * 8(d) asks for.  Synchronous; uses the legacy default stream. */
int pwfs_peak_fp32(int32_t device, int32_t packed, double *tflops, double *elapsed_ms);
/* Returns 0, or a negative pwfs_status value of pwfs.h (PWFS_EINVAL -1, PWFS_ENOMEM -2, PWFS_ECUDA -3). */

#ifdef __cplusplus
}
#endif
#endif /* PWFS_PEAK_H */
