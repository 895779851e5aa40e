/*
 * pwfs_sh.h -- C ABI of the Shack-Hartmann sensor (SURVEY.md 8(f) row f4,
 * second part): wavefront -> lenslet spots on the detector -> centre-of-gravity
 * slopes, on one B200.  Part of libpwfs.so (sm_100a, hand-written CUDA).
 *
 * Where this is defined.  PASSATA simulates "Shack-Hartmann" sensors
 * and "Pyramid and Shack Hartmann propagation (from wavefront to
 * detector plane)" is one of its GPU routines (sec. 6).  The
 * paper prints no SH parameter set or formula; readings F4e-F4i:
 *   F4e  n_sub x n_sub square subapertures of b = N / n_sub pupil pixels each.
 *   F4f  spot = |DFT2(zero-pad_P(A exp(i c phi) on the b x b pixels) *
 *        exp(-i pi (x + y) / P))|^2 / P^2, fftshifted: the flat-wavefront spot
 *        sits on the geometric centre of the P x P array; total = sum |g|^2.
 *   F4g  detector: central (n_px bin)^2 FFT pixels summed in bin x bin blocks;
 *        frame = mosaic [n_sub n_px][n_sub n_px], subaperture (j, i) at rows
 *        [j n_px, (j+1) n_px), columns [i n_px, (i+1) n_px).
 *   F4h  valid subaperture: sum A^2 over it >= thresh * b^2 * max A^2.
 *   F4i  slopes: centre of gravity in detector pixels from the window centre,
 *        Sx = sum (px - (n_px-1)/2) I / sum I, output [Sx(valid, row-major) ...,
 *        Sy ...]; +x tilt gives Sx > 0.
 *
 * Conventions as in pwfs.h (row-major [y][x], status codes, ownership,
 * asynchronous run call on `cuda_stream`, no host<->device copy, no
 * allocation in the run call).
 */
#ifndef PWFS_SH_H
#define PWFS_SH_H

#include <stdint.h>

#include "pwfs.h"

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pwfs_sh pwfs_sh_t; /* opaque */

typedef struct {
    int32_t n_pupil;        /* N >= 1                                                            */
    int32_t n_subap;        /* n_sub: must divide N; b = N / n_sub in [1, 16]                    */
    const float *pupil_amp; /* HOST ptr, N*N floats row-major; amplitude A >= 0, not all 0; copied */
    int32_t fft_px;         /* P: even, b <= P <= 64 (spot sampling lambda / (d P / b))          */
    int32_t n_px;           /* detector pixels across one subaperture window (>= 1)              */
    int32_t bin;            /* FFT pixels per detector pixel (>= 1); n_px * bin <= P, same parity */
    float illum_thresh;     /* F4h; <= 0 selects 0.5                                              */
    float phase_scale;      /* c: lambda_phase / lambda_sensor (1 = phase already at the sensor's) */
    int32_t device;         /* CUDA device ordinal                                               */
} pwfs_sh_params;

/* Validates p (PWFS_EINVAL; PWFS_EUNSUPPORTED for b > 16 or P > 64), builds the
 * twiddle table and the valid mask on the host, uploads.  n_valid == 0 is
 * PWFS_EINVAL.  On failure *out = NULL. */
int pwfs_sh_create(const pwfs_sh_params *p, pwfs_sh_t **out);

/* Detector size n_sub * n_px and number of valid subapertures (either may be NULL). */
int pwfs_sh_info(const pwfs_sh_t *h, int32_t *det_size, int32_t *n_valid);

/* Copy the n_sub*n_sub valid mask (row-major, 1 = valid) to HOST memory. */
int pwfs_sh_valid_mask(const pwfs_sh_t *h, uint8_t *host_mask);

/* d_phase: DEVICE float [B][N][N] radians.  d_frames: DEVICE float [B][D][D],
 * D = n_sub * n_px (F4g).  d_slopes: DEVICE float [B][2 n_valid] (F4i), may be
 * NULL.  B = 0 is a no-op. */
int pwfs_sh_run(pwfs_sh_t *h, const float *d_phase, int32_t B, float *d_frames, float *d_slopes,
                void *cuda_stream);

/* Release everything the handle owns.  NULL-safe. */
void pwfs_sh_destroy(pwfs_sh_t *h);

#ifdef __cplusplus
}
#endif
#endif /* PWFS_SH_H */
