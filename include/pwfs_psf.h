/*
 * pwfs_psf.h -- C ABI of the PSF camera (first part):
 * instantaneous and long-exposure point-spread function and Strehl ratio of a
 * batch of residual wavefronts, on one B200.  Part of libpwfs.so (sm_100a,
 * hand-written CUDA, the same register-resident FP32 FFT butterflies as the
 * pyramid path; no cuFFT).
 *
 * Where this is defined.  "generating a PSF at a given wavelength based on an
 * input wavefront" (sec. 2); Table 1 `camera` (L184-191):
 * wavelengthInNm, nd "padding coefficient for PSF computation", start_time;
 * `psf = factory.get_psf(params.camera)` (L247-248); `psf.out_sr` is what the
 * example stores (L270-271); "PSF generation from residual wavefront" is a GPU
 * routine (L344, sec. 6).  Readings F4a-F4d:
 *   F4a  G = A exp(i c phi), c = phase_scale (lambda_phase / lambda_camera),
 *        zero-padded to M x M; nd = M / N need not be an integer.
 *   F4b  PSF = |DFT2(G)|^2 / (M^2 sum A^2)  (forward, sign -; sum PSF = 1),
 *        zero frequency at pixel [M/2][M/2].
 *   F4c  Strehl ratio of a frame = |sum A exp(i c phi)|^2 / (sum A)^2.
 *   F4d  long exposure = mean of the PSFs of all frames accumulated since the
 *        last reset.
 *
 * Conventions as in pwfs.h (row-major [y][x], status codes, ownership,
 * asynchronous run calls on `cuda_stream`).
 */
#ifndef PWFS_PSF_H
#define PWFS_PSF_H

#include <stdint.h>

#include "pwfs.h"

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pwfs_psf pwfs_psf_t; /* opaque */

typedef struct {
    int32_t n_pupil;        /* N >= 2                                                        */
    int32_t m_grid;         /* M = nd * N: PSF grid.  M >= 2N (nd >= 2, Nyquist) and
                               pwfs_supported_grid(M), else PWFS_EINVAL / PWFS_EUNSUPPORTED  */
    const float *pupil_amp; /* HOST ptr, N*N floats row-major; amplitude A >= 0, not all 0; copied */
    float phase_scale;      /* c of F4a (1 = phase already at the imaging wavelength)        */
    int32_t device;         /* CUDA device ordinal                                           */
} pwfs_psf_params;

/* Validates p, builds the twiddle table in double on the host, uploads,
 * allocates the M x M accumulator (zeroed).  On failure *out = NULL. */
int pwfs_psf_create(const pwfs_psf_params *p, pwfs_psf_t **out);

/* Add the B frames d_phase (DEVICE float [B][N][N], radians) to the long
 * exposure.  d_sr: DEVICE float [B] Strehl ratio of each frame (F4c), may be
 * NULL.  Scratch (the half-transformed batch, 8 B * M * ceil32(N) per frame
 * of a chunk) is allocated on first use and reused; otherwise asynchronous,
 * no host<->device copy.  B = 0 is a no-op. */
int pwfs_psf_accumulate(pwfs_psf_t *h, const float *d_phase, int32_t B, float *d_sr, void *cuda_stream);

/* Write the long-exposure PSF (F4d, F4b normalisation) to d_psf: DEVICE float
 * [M][M].  frames_out (HOST, may be NULL) receives the number of frames
 * accumulated.  With no frames accumulated the PSF is all zeros. */
int pwfs_psf_read(pwfs_psf_t *h, float *d_psf, int64_t *frames_out, void *cuda_stream);

/* Zero the accumulator and the frame count (asynchronous on the stream). */
int pwfs_psf_reset(pwfs_psf_t *h, void *cuda_stream);

/* Release everything the handle owns.  NULL-safe. */
void pwfs_psf_destroy(pwfs_psf_t *h);

#ifdef __cplusplus
}
#endif
#endif /* PWFS_PSF_H */
