/*
 * pwfs_chain.h -- C ABI of the steps downstream of the pyramid (SURVEY.md 8(f)
 * row f2): CCD detector, pyramid slope computer with a reference vector, modal
 * reconstructor.  Part of libpwfs.so (sm_100a, hand-written CUDA); every array
 * the run calls touch is DEVICE memory, so pwfs_atmo_propagate -> pwfs_run ->
 * pwfs_ccd_run -> pwfs_slopec_run -> pwfs_rec_run is one chain of kernels on
 * one stream with no host round trip (sec. 6).
 *
 * Where this is defined.  The paper names objects, wiring and parameters only:
 *   CCD: "a CCD processing object might integrate its input data for several
 *     simulation steps, and produce output data (pixel frames) at a lower rate"
 *     (PAPER.md:L21, L31); Table 1 `detector` (L153-174): size, dt, bandw,
 *     photon_noise, readout_noise, readout_level [e-/pix/frame], quantum_eff;
 *     ccd.in_i = pyr.out_i (L318).
 *   slope computer: Table 1 `slopec` (L137-143): pupdata_tag (pupil
 *     subaperture indices), sn_tag (slope reference vector);
 *     sc.in_pixels = ccd.out_pixels (L261).
 *   reconstructor: Table 1 `modalrec` (L212-215) recmat_tag;
 *     rec.in_slopes = sc.out_slopes (L262); rec.out_modes (L265).
 * The readings F2a..F2g taken for everything the paper leaves open are listed
 * in DESIGN.md ("f2") and restated at each call below.
 *
 * Conventions as in pwfs.h: row-major [y][x]; 0 or a negative pwfs_status is
 * returned; nothing throws; a handle owns its device copies; the caller owns
 * every buffer it passes; run calls are asynchronous on `cuda_stream`, perform
 * no host<->device copy and no allocation.  Handles are not thread-safe.
 */
#ifndef PWFS_CHAIN_H
#define PWFS_CHAIN_H

#include <stdint.h>

#include "pwfs.h"

#ifdef __cplusplus
extern "C" {
#endif

/* ------------------------------------------------------------------ CCD --- */
typedef struct pwfs_ccd pwfs_ccd_t; /* opaque */

typedef struct {
    int32_t det_size;      /* D >= 1: frames are D x D (pwfs_info's det_size)                     */
    int32_t n_inst;        /* sensor instances per simulation step (>= 1); input frame
                              b = step * n_inst + inst (F2a; the order pwfs_atmo / pwfs_run use) */
    int32_t n_int;         /* simulation steps summed into one detector frame,
                              dt_ccd / dt_loop >= 1 (F2a)                                         */
    double gain;           /* photons per unit of input intensity per step (>= 0; F2b)           */
    double quantum_eff;    /* quantum efficiency * transmission, in [0, 1] (F2b)                 */
    int32_t photon_noise;  /* != 0: k ~ Poisson(lam) (F2c); 0: k = lam                            */
    int32_t readout_noise; /* != 0: + readout_level * N(0,1) (F2d)                                */
    double readout_level;  /* e-/pixel/frame rms (>= 0)                                          */
    uint64_t seed;         /* Philox4x32-10 key (F2e)                                            */
    int32_t device;        /* CUDA device ordinal                                                */
} pwfs_ccd_params;

/* Validates p.  PWFS_EINVAL: NULL, sizes < 1, negative or non-finite gain /
 * quantum_eff / readout_level, quantum_eff > 1. */
int pwfs_ccd_create(const pwfs_ccd_params *p, pwfs_ccd_t **out);

/* d_frames: DEVICE float [n_steps * n_inst][D][D] intensity (pwfs_run's frames).
 * d_pixels: DEVICE float [n_steps / n_int * n_inst][D][D] in electrons.
 * n_steps must be a multiple of n_int (else PWFS_EINVAL); 0 is a no-op.
 * Per output pixel (F2a-F2e, all in double precision on the device):
 *   lam = quantum_eff * gain * sum over the n_int steps of the instance;
 *   Philox4x32-10 with key = seed (lo, hi) and counter = (pixel index y*D + x,
 *   output frame index lo, hi, 0), output frame index = first_out_frame + p,
 *   gives r0..r3, u_i = (r_i + 1/2) / 2^32;
 *   photon noise: lam < 128: smallest k with u0 <= CDF_Poisson(lam)(k)
 *   (sequential search); lam >= 128: k = max(0, floor(lam + sqrt(lam) z + 1/2)),
 *   z = sqrt(-2 ln u0) cos(2 pi u1); lam <= 0: k = 0;
 *   read noise: + readout_level * sqrt(-2 ln u2) cos(2 pi u3).
 * Pixels are not clipped or digitised.  The same (seed, first_out_frame) gives
 * the same pixels on every call. */
int pwfs_ccd_run(pwfs_ccd_t *h, const float *d_frames, int32_t n_steps, int64_t first_out_frame,
                 float *d_pixels, void *cuda_stream);

void pwfs_ccd_destroy(pwfs_ccd_t *h); /* NULL-safe */

/* ------------------------------------------------------- slope computer --- */
typedef struct pwfs_slopec pwfs_slopec_t; /* opaque */

/* n_sub: subapertures across one pupil image (frames are 2n_sub x 2n_sub).
 * h_valid: HOST uint8 [n_sub][n_sub], != 0 = valid (pwfs_valid_mask's output:
 * the "pupdata" of PAPER.md:L139-140); at least one must be valid.
 * slope_norm: 0 = divide by the mean valid-subaperture flux of the frame,
 * 1 = by the subaperture's own flux (pwfs_params.slope_norm).
 * h_sn: HOST float [2 * n_valid] slope reference vector in
 * the output order below, or NULL for none.  Both arrays are copied. */
int pwfs_slopec_create(int32_t n_sub, const uint8_t *h_valid, int32_t slope_norm, const float *h_sn,
                       int32_t device, pwfs_slopec_t **out);

/* Replace (or, with NULL, clear) the slope reference vector.  Synchronous copy. */
int pwfs_slopec_set_reference(pwfs_slopec_t *h, const float *h_sn);

int pwfs_slopec_n_slopes(const pwfs_slopec_t *h, int32_t *n_slopes); /* 2 * n_valid */

/* d_pixels: DEVICE float [B][2n_sub][2n_sub].  d_slopes: DEVICE float
 * [B][2 n_valid] = [Sx(valid subaps, row-major) ..., Sy ...] - sn, with Sx, Sy
 * exactly as pwfs_run defines them (tiles a,b,c,d = (qx,qy) = (0,0),(1,0),(0,1),
 * (1,1); Sx = ((a+c)-(b+d))/norm, Sy = ((a+b)-(c+d))/norm) (F2f).  A zero
 * normalisation (possible on noisy frames) gives inf/nan, not an error. */
int pwfs_slopec_run(pwfs_slopec_t *h, const float *d_pixels, int32_t B, float *d_slopes, void *cuda_stream);

void pwfs_slopec_destroy(pwfs_slopec_t *h); /* NULL-safe */

/* -------------------------------------------------- modal reconstructor --- */
typedef struct pwfs_rec pwfs_rec_t; /* opaque */

/* h_recmat: HOST float [n_modes][n_slopes] row-major, copied to the device
 * (rows padded to a multiple of 4 floats).  n_modes, n_slopes >= 1. */
int pwfs_rec_create(int32_t n_modes, int32_t n_slopes, const float *h_recmat, int32_t device,
                    pwfs_rec_t **out);

/* d_slopes: DEVICE float [B][n_slopes]; d_modes: DEVICE float [B][n_modes],
 * modes[b][m] = sum_j recmat[m][j] * slopes[b][j] (F2g), FP32 accumulation in a
 * fixed order (deterministic).  B = 0 is a no-op.
 * WHICH ARITHMETIC RUNS DEPENDS ON THE BATCH SIZE: single frames and small
 * problems run FP32-FMA kernels (B = 1: a streaming GEMV); batches (B >= 24 and
 * n_modes * n_slopes >= 65536) run on the tensor cores: recmat (inside the
 * kernel) and the slopes (by a small kernel) are each split into two TF32 planes
 * and three tcgen05 products are accumulated in FP32, which keeps the FP32 bar
 * (error <= 7e-7 sum |R||s| from the split, plus FP32 accumulation) -- so a frame's
 * modes may differ in the last bits between a batched and a single-frame call.
 * Environment PWFS_REC_TC=0 at create keeps every call on the FP32 kernels.
 * The first batched call (or a larger batch later) sizes the slope planes and
 * split-K scratch: it synchronises the stream and allocates; call
 * pwfs_rec_reserve beforehand to keep pwfs_rec_run free of both.  While
 * `cuda_stream` is being captured into a CUDA graph a call that would have to
 * allocate returns PWFS_EINVAL instead. */
int pwfs_rec_run(pwfs_rec_t *h, const float *d_slopes, int32_t B, float *d_modes, void *cuda_stream);

/* Size the tensor-core path's scratch for every batch of 1..B frames (no-op for
 * batch sizes the FP32 kernels serve): the need is taken as the largest over the
 * batch sizes up to B, because a smaller batch is split further along K and can
 * write more partial sums than B itself.  Synchronous; allocates. */
int pwfs_rec_reserve(pwfs_rec_t *h, int32_t B);

void pwfs_rec_destroy(pwfs_rec_t *h); /* NULL-safe */

#ifdef __cplusplus
}
#endif
#endif /* PWFS_CHAIN_H */
