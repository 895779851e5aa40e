/*
 * pwfs_dm.h -- C ABI of the two objects that close the loop after the reconstructor:
 * the deformable mirror (influence-function multiply) and the integrator control.
 * Part of libpwfs.so (sm_100a, hand-written CUDA); every array the run calls touch is
 * DEVICE memory, so  pwfs_rec_run -> pwfs_int_step -> pwfs_dm_apply -> pwfs_run  is one
 * chain of kernels on one stream with no host round trip (sec. 6).
 *
 * Where this is defined.  The paper names objects, wiring and parameters only:
 *   DM: Table 1 `dm` (type 'zernike', nmodes 54, npixels 160, obsratio,
 *     height); dm = factory.get_dm(params.dm), dm.in_command = intc.out_comm (L246,
 *     L265-266); its output layer is added to the propagation's layer list
 *     (prop.add_layer_to_layer_list, dm.out_layer, L257).  "Influence function
 *     multiplication (from DM commands to applied wavefront)" is one of the four
 *     GPU-accelerated routine families (L343); for an EELT-like system "the influence
 *     functions matrix alone occupies between 4 and 5 GB" (L350).
 *   control: Table 1 `control` (L144-152): type 'INT', delay [frames], int_gain (a vector);
 *     intc.in_delta_comm = rec.out_modes (L265).
 * Readings D1, D2, C1, C2 (restated at each call).
 *
 * Conventions as in pwfs.h: row-major [y][x]; 0 or a negative pwfs_status is returned;
 * nothing throws; a handle owns its device copies; the caller owns every buffer it
 * passes; run calls are asynchronous on `cuda_stream`, copy nothing between host and
 * device and allocate nothing.  The device current on entry is current on return.
 */
#ifndef PWFS_DM_H
#define PWFS_DM_H

#include <stdint.h>

#include "pwfs.h"

#ifdef __cplusplus
extern "C" {
#endif

/* ------------------------------------------------------ deformable mirror --- */
typedef struct pwfs_dm pwfs_dm_t; /* opaque */

/* n_act actuators / modes, each with an influence function sampled on the same n_pix pupil
 * pixels: h_ifs HOST float [n_act][n_pix] row-major, h_pix HOST int32 [n_pix] = flat indices
 * y * n_pupil + x (distinct, in [0, n_pupil^2)).  Both are copied.  The matrix is kept on the
 * device as it is given (4 bytes per element: an EELT-class 4096 x 160 000 matrix is 2.6 GB).
 * PWFS_EINVAL: NULL, sizes < 1, an index out of range or repeated, a non-finite entry. */
int pwfs_dm_create(int32_t n_act, int32_t n_pupil, int32_t n_pix, const int32_t *h_pix, const float *h_ifs,
                   int32_t device, pwfs_dm_t **out);

/* D1, D2: for every frame b < B
 *     layer[b][y][x] = sum_m ifs[m][p] * cmd[b][m]   at the pixels p -> (y, x) the influence
 *                      functions are defined on, 0 elsewhere,
 *     phase[b]       = beta * phase[b] + alpha * layer[b]        (beta is 0 or 1).
 * d_cmd: DEVICE float [B][n_act].  d_phase: DEVICE float [B][n_pupil][n_pupil]; with beta = 0 it
 * is overwritten (pixels outside the influence functions become 0), with beta = 1 the scaled layer
 * is added in place -- the residual phase the sensor sees is atmosphere + alpha * DM layer, the sign
 * and the unit conversion being the caller's alpha.  FP32 FMA in a fixed order (deterministic):
 * the actuators are cut into `msplit` contiguous ranges, each range is summed per pixel in the
 * order m ascending, and the range sums are then added in range order.  msplit is fixed at create
 * (1 when n_act < 64; otherwise chosen from n_act, n_pix and the SM count of `device` so that the
 * kernel fills the machine), so results repeat bit for bit from call to call and do not depend on
 * B, but they can differ in the last bits between GPUs with different SM counts and are not the
 * plain m = 0, 1, ... sum once msplit > 1.  HBM-bound: the matrix is streamed once per group of up
 * to 8 frames.
 * PWFS_EINVAL for beta other than 0 or 1. */
int pwfs_dm_apply(pwfs_dm_t *h, const float *d_cmd, int32_t B, float *d_phase, float alpha, float beta,
                  void *cuda_stream);

void pwfs_dm_destroy(pwfs_dm_t *h); /* NULL-safe */

/* ------------------------------------------------------ integrator control --- */
typedef struct pwfs_int pwfs_int_t; /* opaque */

/* n_modes element-wise gains (HOST float, copied) and a delay of `delay` >= 0 whole frames.
 * The integrator state and its history live on the device and start at zero. */
int pwfs_int_create(int32_t n_modes, const float *h_gain, int32_t delay, int32_t device, pwfs_int_t **out);

/* C1, C2: one loop step.  state c_t = c_{t-1} + gain (.) delta_t; the command written to d_cmd
 * is c_{t-delay} (zero while t < delay), t counting the calls since create / reset.
 * d_delta, d_cmd: DEVICE float [n_modes].  The step counter lives on the device, so a call
 * captured in a CUDA graph advances correctly on every replay. */
int pwfs_int_step(pwfs_int_t *h, const float *d_delta, float *d_cmd, void *cuda_stream);

/* Back to t = 0 with a zero state (asynchronous on the stream). */
int pwfs_int_reset(pwfs_int_t *h, void *cuda_stream);

void pwfs_int_destroy(pwfs_int_t *h); /* NULL-safe */

#ifdef __cplusplus
}
#endif
#endif /* PWFS_DM_H */
