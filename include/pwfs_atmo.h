/*
 * pwfs_atmo.h -- C ABI of the upstream step of the pyramid-WFS path (SURVEY.md
 * 8(f) row f1): wavefront propagation through phase screens on the GPU, so the
 * phase batch pwfs_run() consumes is produced in device memory without a host
 * round trip.  Part of libpwfs.so (sm_100a, hand-written CUDA).
 *
 * Where this is defined.  "Wavefront propagation through phasescreens" is the
 * first GPU-accelerated routine the paper lists (sec. 6);
 * `prop = factory.get_atmo_propagation(atmo, source)`, layers
 * are added one by one (L254-257), `prop.pupil_list` feeds `pyr.in_ef` (L317);
 * the atmosphere is a stack of layers with heights, wind speed and direction
 * (Table 1) seen from sources at polar coordinates
 * (L175-183).  The paper gives no formula; the readings:
 *
 *   F1a frozen flow: layer l is a periodic G x G screen moving rigidly with
 *       velocity (vx_l, vy_l); at time t = step * dt pupil pixel (x, y) looks at
 *       screen coordinate X = x + (-vx_l t + h_l tan_x) / pitch (Y likewise),
 *       h_l = layer height, (tan_x, tan_y) = tangent of the source direction.
 *       Sources at infinity (no cone effect); pupil and screens share `pitch`.
 *   F1b bilinear interpolation of the four neighbours, indices modulo G.
 *   F1c layers are summed with unit weight, then multiplied by one scale
 *       factor per sensing wavelength (lambda_ref / lambda).
 *   F1d frame order: step-major, then source direction, then wavelength:
 *       b = (step * n_dirs + dir) * n_wl + wl.
 *
 * Conventions as in pwfs.h: arrays row-major [y][x]; 0 or a negative
 * pwfs_status is returned; nothing throws; the handle owns its device copies;
 * the caller owns every buffer it passes.  A handle is not thread-safe.
 */
#ifndef PWFS_ATMO_H
#define PWFS_ATMO_H

#include <stdint.h>

#include "pwfs.h"

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pwfs_atmo pwfs_atmo_t; /* opaque */

typedef struct {
    int32_t n_layers;       /* L >= 1                                                      */
    int32_t screen_px;      /* G : side of every (periodic) screen, G >= n_pupil           */
    const float *screens;   /* HOST ptr, L*G*G floats [l][y][x]: phase [rad] at the
                               reference wavelength; copied                                */
    double pitch;           /* metres per pixel (> 0), pupil and screens                   */
    const double *wind_vxy; /* HOST [L][2] layer velocity (vx, vy) in m/s                  */
    const double *heights;  /* HOST [L] layer height in m                                  */
    int32_t n_dirs;         /* S >= 1 source directions                                    */
    const double *dirs_tan; /* HOST [S][2] (tan_x, tan_y) of each direction                */
    int32_t n_wl;           /* W >= 1 sensing wavelengths                                  */
    const double *wl_scale; /* HOST [W] factor applied to the summed phase (lambda_ref/lambda) */
    int32_t n_pupil;        /* N >= 1 : output frames are N x N                            */
    int32_t device;         /* CUDA device ordinal                                         */
} pwfs_atmo_params;

/* Validates p, uploads the screens and the geometry.  On failure *out = NULL.
 * PWFS_EINVAL: NULL pointers, sizes out of range, non-finite numbers. */
int pwfs_atmo_create(const pwfs_atmo_params *p, pwfs_atmo_t **out);

/* Frames produced per simulation step (n_dirs * n_wl). */
int pwfs_atmo_frames_per_step(const pwfs_atmo_t *h, int32_t *frames);

/* Propagate `n_steps` consecutive steps starting at step index `first_step`
 * (time of step i is (first_step + i) * dt seconds, evaluated in double
 * precision on the device).  d_phase: DEVICE float [n_steps * n_dirs * n_wl][N][N]
 * in the order F1d -- exactly the layout pwfs_run() reads.  cuda_stream: a
 * cudaStream_t (NULL = default stream).  Asynchronous; performs no host<->device
 * copy and no allocation.  n_steps = 0 is a no-op. */
int pwfs_atmo_propagate(pwfs_atmo_t *h, int64_t first_step, int32_t n_steps, double dt,
                        float *d_phase, void *cuda_stream);

/* Release everything the handle owns.  NULL-safe. */
void pwfs_atmo_destroy(pwfs_atmo_t *h);

#ifdef __cplusplus
}
#endif
#endif /* PWFS_ATMO_H */
