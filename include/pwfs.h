/*
 * pwfs.h -- C ABI of libpwfs.so: the modulated pyramid wavefront-sensor forward
 * model on one NVIDIA B200 (sm_100a), hand-written CUDA, no cuFFT.
 *
 * What the library computes (one "frame" per input phase screen):
 *   for each of K points on the modulation circle build the pupil phasor
 *   A exp(i(phi + tilt_k)), zero-pad it into an M x M grid, 2-D DFT to the focal
 *   plane, multiply by the four-face pyramid phase mask, inverse 2-D DFT back
 *   to the pupil plane, accumulate |E|^2 over k; rebin the four pupil images to
 *   n_sub x n_sub subaperture pixels each (one 2n_sub x 2n_sub detector frame)
 *   and reduce them to normalised x/y slopes over the valid subapertures.
 *
 * Where this is defined.  The paper names the object and its wiring only:
 * "apply a transformation from focal plane to pupil plane emulating an optical
 * pyramid" (sec. 2); parameters pup_diam / pup_dist / mod_amp /
 * output_resolution / wavelengthInNm (Table 1);
 * pyr.in_ef -> pyr.out_i -> ccd.in_i, ccd.out_pixels ->
 * sc.in_pixels -> sc.out_slopes; GPU-resident data passed
 * by opaque handle (sec. 6); "Pyramid ... propagation (from
 * wavefront to detector plane)" is one of the GPU-accelerated routines
 * (PAPER.md:L342).  The arithmetic is BASELINE.json `north_star`, written out
 * as steps O0..O9 in SURVEY.md section 8(c) and restated with every reading of
 * a silent point in DESIGN.md.
 *
 * Conventions
 *   - 2-D arrays are row-major [y][x] (x fast).  Phase is in radians at the
 *     sensing wavelength.  1 lambda/D of tilt = 2 pi across the N pupil pixels.
 *   - Every function returns PWFS_OK (0) or a negative pwfs_status; nothing
 *     throws or aborts across this boundary and there is no global mutable state
 *     (one exception, stated there: the fixed scratch array of pwfs_run_noalloc).
 *   - A handle owns its device tables and scratch memory.  The caller owns
 *     pupil_amp (host memory, copied by pwfs_create) and the phase / frames /
 *     slopes buffers.  A handle is not thread-safe; distinct handles are.
 *   - Non-finite phase values propagate to the outputs (no checking on the hot
 *     path).
 *   - Environment, read once when a handle is created (none is needed for normal
 *     use, none changes a result beyond FP32 summation order): PWFS_SCRATCH_MB
 *     (scratch budget, default 32768), PWFS_SMALL=0/1 (never / always take the fused
 *     M = 128 kernel), PWFS_REC_TC=0 (pwfs_chain.h).  The measurement hooks that DO
 *     change results or schedules behind the caller's back -- PWFS_DEBUG_T_ALIAS=1
 *     (every frame aliases the intermediate of frame 0: a timing experiment with
 *     wrong output) and PWFS_REC_KSPLIT (forced K split of the tensor-core
 *     reconstructor) -- exist only in a build made with -DPWFS_TUNING
 *     (`python -m paper_1607_07624_b200.build --tuning` -> libpwfs_tuning.so);
 *     libpwfs.so does not contain them.  The Python binding loads the library named
 *     by PWFS_LIB_PATH, else the in-tree libpwfs.so.
 */
#ifndef PWFS_H
#define PWFS_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pwfs pwfs_t; /* opaque */

typedef enum {
    PWFS_OK = 0,
    PWFS_EINVAL = -1,       /* bad parameter, NULL pointer, geometry that leaves the grid, n_valid == 0 */
    PWFS_ENOMEM = -2,       /* host or device allocation failed */
    PWFS_ECUDA = -3,        /* a CUDA runtime call failed (see pwfs_last_cuda_error) */
    PWFS_EUNSUPPORTED = -4, /* valid request this build has no kernel for (e.g. M/32 not instantiated) */
    PWFS_ELIMIT = -5        /* pwfs_run_noalloc only: the batch does not fit the library's fixed scratch array */
} pwfs_status;

/* Parameters of one sensor (names follow PAPER.md Table 1 where
 * the paper has one: n_subap = pup_diam, mod_radius = mod_amp). */
typedef struct {
    int32_t n_pupil;        /* N >= 2 : pupil sampling, D spans exactly N px                  */
    int32_t m_grid;         /* M : FFT grid.  M >= 2N, M = 32*R with R in the built set: every
                               2/3/5-smooth R in 4..64, i.e. 24 grids from M = 128 to 2048
                               (pwfs_supported_grid)                                          */
    const float *pupil_amp; /* HOST ptr, N*N floats row-major [y][x]; amplitude A >= 0; copied */
    int32_t mask_shift_px;  /* s : pupil-image offset in px (mask phase 2 pi s (|u~|+|v~|)/M).
                               <= 0 selects the default M/4 (needs M % 4 == 0).
                               Needs N <= 2 s and s <= M/2 - N/2 (windows disjoint, in grid).
                               An INTEGER by design: the pupil images are read back through
                               windows of whole grid pixels (O7's origin M/2 +- s - N/2), and
                               DESIGN.md reading A8 fixes s to whole pixels; a half-pixel shift
                               would need an interpolating window and is not part of the model */
    float mod_radius;       /* r >= 0 in lambda/D                                             */
    int32_t mod_points;     /* K >= 1 points equally spaced on the circle (K=1, r=0: none)    */
    float mod_angle0;       /* theta_0 [rad] of point 0, counter-clockwise from +x            */
    int32_t n_subap;        /* n_sub in [1, N]: subapertures across one pupil image;
                               binning b = N / n_sub need not be an integer (area weights)    */
    float illum_thresh;     /* valid iff illumination >= thresh * full subaperture; <= 0 -> 0.5 */
    int32_t slope_norm;     /* 0: divide by the mean valid-subaperture flux (default);
                               1: divide by the subaperture's own flux                        */
    int32_t device;         /* CUDA device ordinal                                            */
} pwfs_params;

/* Build a sensor: validates p, computes all tables on the host in double
 * precision (tilt tables, mask, twiddles, rebin weights, valid mask), uploads
 * them.  Scratch memory is allocated lazily by the first pwfs_run and reused.
 * On failure *out is set to NULL.  Defined by: north_star "pwfs_create(pupil,
 * M, mask params, mod radius, K, binning)". */
int pwfs_create(const pwfs_params *p, pwfs_t **out);

/* Extensions of the sensor model, all optional.
 *   Tilt list: n_tilts > 0 replaces the modulation circle (mod_radius, mod_points,
 *   mod_angle0 are then ignored) by the points (tilt_x[k], tilt_y[k]) in lambda/D
 *   with non-negative weights tilt_w[k] (NULL = uniform; only ratios matter):
 *       I = sum_k w_k |E_k|^2 / sum_k w_k.
 *   This is how an extended / resolved reference source, or any non-circular
 *   modulation, is given ("resolved sources", L77 "Extended (non
 *   point-like) reference source studies").  The uniform circle list reproduces
 *   pwfs_create exactly.  The row pass is shared between points of equal tilt_x.
 *   Field stop: field_stop_px >= 0 multiplies the pyramid mask by the SQUARE stop
 *   |u~| <= h and |v~| <= h (h = field_stop_px in focal-plane bins, signed
 *   frequencies u~ in [-M/2, M/2); 1 lambda/D = M/N bins): the focal-plane
 *   field of view (Table 1 `pyramid`, "Requested
 *   field-of-view [arcsec]").  < 0, or >= M/2, means no stop.  A square stop keeps
 *   the mask separable; a stop selects the table-mask kernels.
 * All pointers are HOST memory, copied by the call. */
typedef struct {
    int32_t n_tilts;
    const float *tilt_x;
    const float *tilt_y;
    const float *tilt_w;
    float field_stop_px;
} pwfs_ext;

/* pwfs_create with the extensions above; x == NULL is pwfs_create. */
int pwfs_create_ex(const pwfs_params *p, const pwfs_ext *x, pwfs_t **out);

/* Detector size (2*n_sub) and number of valid subapertures.  Either pointer
 * may be NULL. */
int pwfs_info(const pwfs_t *h, int32_t *det_size, int32_t *n_valid);

/* Copy the n_sub*n_sub valid-subaperture mask (row-major [j][i], 1 = valid,
 * same mask for all four pupil images) to HOST memory. */
int pwfs_valid_mask(const pwfs_t *h, uint8_t *host_mask);

/* The hot path.  d_phase: DEVICE float [B][N][N] (radians).  d_frames: DEVICE
 * float [B][2n_sub][2n_sub], frame[qy*n_sub + j][qx*n_sub + i] = area-weighted
 * SUM of I = mean_k |E_k|^2 over subaperture (j,i) of the pupil image at
 * (M/2 + (2qx-1)s, M/2 + (2qy-1)s).  d_slopes: DEVICE float [B][2*n_valid] =
 * [Sx(valid subaps, row-major) ..., Sy(...)], Sx = ((a+c)-(b+d))/norm,
 * Sy = ((a+b)-(c+d))/norm with a,b,c,d the tiles (qx,qy) = (0,0),(1,0),(0,1),
 * (1,1); may be NULL.  cuda_stream: a cudaStream_t (NULL = default stream).
 * Asynchronous: work is enqueued on the stream and the call returns; buffers
 * must stay alive until the stream reaches that point.  B = 0 is a no-op.
 * Does not allocate once scratch has been sized for a batch this large
 * (pwfs_reserve, or an earlier call); when a larger batch arrives it frees and
 * re-allocates its scratch -- except while `cuda_stream` is being captured into a
 * CUDA graph, where it returns PWFS_EINVAL and enqueues nothing.  The CUDA device
 * that was current on entry is current again on return.
 * Defined by: north_star "pwfs_run(phase batch -> frames, slopes)". */
int pwfs_run(pwfs_t *h, const float *d_phase, int32_t B, float *d_frames, float *d_slopes,
             void *cuda_stream);

/* Size the handle's scratch memory (and, for batches that run in several chunks,
 * its internal side stream and events) for pwfs_run calls of up to B frames, so
 * that those calls neither allocate nor create anything.  Required before a
 * pwfs_run of a batch size the handle has not seen is captured into a CUDA graph:
 * cudaMalloc is not allowed during stream capture, and pwfs_run then returns
 * PWFS_EINVAL instead of allocating.  "Up to B" is meant literally: the scratch is
 * sized for the largest need over ALL batch sizes 1..B -- a smaller batch may take the
 * fused M = 128 kernel where B itself does not, or split its modulation loop further
 * and so need more column scratch per frame than B does.  Call it again after
 * pwfs_set_schedule (the knobs change the need).  Synchronous; may free and
 * re-allocate. */
int pwfs_reserve(pwfs_t *h, int32_t B);

/* Same computation with HOST buffers (h_slopes may be NULL): copies the phase
 * batch host->device, runs, copies frames and slopes device->host and returns
 * after they have arrived (synchronous).  Works chunk by chunk on three
 * internal streams, so with pinned host memory the copy-in of the next chunk
 * and the copy-out of the previous one run under the kernels of the current
 * chunk; pageable memory works but is slower. */
int pwfs_run_host(pwfs_t *h, const float *h_phase, int32_t B, float *h_frames, float *h_slopes);

/* pwfs_run for callers that are not allowed to allocate device memory.
 *
 * Who needs this.  Two kinds of user of this library cannot let a sensor call reach
 * cudaMalloc / cudaFree, which pwfs_run does whenever a batch is larger than any it has
 * seen (and pwfs_reserve does on request):
 *   - a real-time control thread (the adaptive-optics loop this sensor model stands in
 *     for runs at a fixed frame rate): cudaMalloc and cudaFree take a process-wide lock,
 *     may wait for ALL work on the device to drain, and have no upper bound on how long
 *     they take, so one call in the wrong step is a missed deadline;
 *   - a process in which something else has been given the device memory -- a pooling
 *     allocator that grabbed nearly all of HBM at start-up, a fixed per-client memory
 *     quota -- so that a cudaMalloc from inside this library would fail or steal from
 *     that budget behind its owner's back.
 * Such a caller creates the handle during start-up (pwfs_create uploads its tables, that
 * is the one allocation) and from then on calls this function only.
 *
 * What it does.  Exactly what pwfs_run does on the M = 128 grid for a small batch: the
 * whole path -- phasor, both transforms, mask, sum over the modulation points, rebin,
 * slopes -- in one kernel launch on `cuda_stream`.  Arguments, layouts, ownership and
 * asynchrony are those of pwfs_run; the caller passes the phase batch and the output
 * buffers (DEVICE memory; d_slopes may be NULL).  The results are the ones pwfs_run
 * gives when it takes its fused-kernel path (same kernel, same order of additions).
 * The kernel's working memory (one partial detector frame per frame and modulation
 * point, one counter per frame) does not come from the heap: it is a fixed array inside
 * libpwfs.so, PWFS_NOALLOC_SCRATCH_BYTES (4 MiB + 256 B) on every GPU that loads the
 * library, held until the process exits.  The call itself performs no cudaMalloc,
 * no cudaFree, and creates no stream or event.
 *
 * Limits.  Sensors the fused kernel serves: m_grid = 128, n_pupil <= 64, n_subap <= 32.
 * Others get PWFS_EUNSUPPORTED.  A batch must satisfy B <= PWFS_NOALLOC_MAX_FRAMES and
 * B * K * (2 n_subap)^2 <= PWFS_NOALLOC_MAX_PART_FLOATS (K = modulation points; the
 * 10-frame, K = 12, n_subap = 16 case of BASELINE.json's first config uses 12 % of it);
 * a larger one gets PWFS_ELIMIT and nothing is enqueued -- split it into several calls
 * on the same stream.
 *
 * First call.  The first call on a given GPU asks the CUDA runtime where the array
 * sits on that GPU (with the handle's device current) and remembers the answer; this may
 * make the runtime load the library's device code there.  Make that first call during
 * start-up, outside any stream capture; later calls on that GPU skip the step.
 *
 * Sharing.  There is ONE array per GPU, shared by every handle and every thread in the
 * process, and it keeps the contents the last call left.  Each call clears the counters
 * it needs in stream order before its kernel, and overwrites the partial frames before
 * reading them, so calls that execute one after another (same stream, or ordered by
 * events) need no clean-up in between.  Two calls that can EXECUTE at the same time on
 * one GPU -- different streams without an ordering, or two host threads -- race on the
 * array and produce garbage; serialise them, or use pwfs_run (whose scratch is per
 * handle) for all but one of them.
 *
 * Errors: PWFS_EINVAL (NULL handle or buffer, B < 0, debug handle), PWFS_EUNSUPPORTED,
 * PWFS_ELIMIT, PWFS_ECUDA.  B = 0 is a no-op.  The CUDA device that was current on entry
 * is current again on return.
 * Defined by: north_star "pwfs_run(phase batch -> frames, slopes)"; the per-step call of
 * a closed loop is PAPER.md:L33 ("triggers all processing objects once per simulation
 * step"). */
#define PWFS_NOALLOC_MAX_FRAMES 64
#define PWFS_NOALLOC_MAX_PART_FLOATS (1u << 20)
#define PWFS_NOALLOC_SCRATCH_BYTES (256u + 4u * PWFS_NOALLOC_MAX_PART_FLOATS)
int pwfs_run_noalloc(pwfs_t *h, const float *d_phase, int32_t B, float *d_frames, float *d_slopes,
                     void *cuda_stream);

/* Release everything the handle owns.  NULL-safe. */
void pwfs_destroy(pwfs_t *h);

/* Static description of a status code. */
const char *pwfs_strerror(int code);

/* cudaError_t (as int) of the last failing CUDA call on this handle, 0 if none. */
int pwfs_last_cuda_error(const pwfs_t *h);

/* Kernel class (see pwfs_get_timing) of the last launch the CUDA runtime refused on
 * this handle, -1 if none: pwfs_run checks cudaGetLastError after every launch. */
int pwfs_last_failed_kernel(const pwfs_t *h);

/* 1 if this build has kernels for an M-point grid, else 0. */
int pwfs_supported_grid(int32_t m_grid);

/* Scheduling knobs (0 keeps the built-in heuristic): frames processed per
 * kernel chunk, and the number of ways the K modulation points are split
 * across warps in the column pass.  Results do not depend on them beyond FP32
 * summation order.  Non-zero knobs also select the two-kernel path where the
 * fused small-grid kernel would otherwise run (M = 128, N <= 64, n_sub <= 32,
 * batches of up to ~16 SMs' worth of x-tilts; environment PWFS_SMALL=0 / 1
 * forces it off / on whenever the geometry allows). */
int pwfs_set_schedule(pwfs_t *h, int32_t frames_per_chunk, int32_t k_split);

/* Instrumentation.  Kernel classes: 0 = row pass (phasor + x-convolution),
 * 1 = column pass (y-convolution + |E|^2 accumulation + y-rebin),
 * 2 = x-rebin, 3 = slopes, 4 = the fused single-kernel path that serves small
 * batches on the M = 128 grid (all of the above in one launch).  pwfs_set_timing(h, 1) makes pwfs_run bracket every
 * kernel with CUDA events on the caller's stream; pwfs_get_timing then
 * synchronises those events and returns, for everything run since timing was
 * enabled (or last read), the summed device time per class in milliseconds and
 * the launch count per class.  launches[] is counted even when timing is off. */
#define PWFS_NUM_KERNEL_CLASSES 5
int pwfs_set_timing(pwfs_t *h, int32_t enable);
int pwfs_get_timing(pwfs_t *h, float ms[PWFS_NUM_KERNEL_CLASSES],
                    int64_t launches[PWFS_NUM_KERNEL_CLASSES]);

/* Internal geometry, for reports: n_cols = pupil-plane columns actually
 * computed (<= 2N), k_unique = distinct x-tilts among the K modulation points
 * (the row pass is shared between points with equal x-tilt), frames_per_chunk
 * and k_split as they would be used for a batch of B frames. */
int pwfs_geometry(const pwfs_t *h, int32_t B, int32_t *n_cols, int32_t *k_unique,
                  int32_t *frames_per_chunk, int32_t *k_split);

/* TEST-ONLY exports (SURVEY.md 8(b) "optional test-only export", pins P2 / P7 of 8(c)).
 * pwfs_debug_intensity runs the row pass and the column pass of the hot path -- the
 * same kernels pwfs_run launches -- one frame at a time and returns the FULL-resolution
 * intensity I = (1/K) sum_k |E_k|^2 before rebinning: DEVICE float [B][M][M], row-major
 * [y][x] in the placement of definition O2 (pupil at offset M/2 - N/2 on both axes,
 * i.e. directly comparable with the definition).  Only the columns that hold a pupil
 * image are computed (all of them when M = 2N); the others are returned as zero.
 * Synchronous; allocates and frees a temporary buffer; not for production use.
 * pwfs_debug_create is pwfs_create_ex with the mask shift given explicitly
 * (mask_shift_px >= 0; 0 is the identity mask) and WITHOUT the window constraints
 * N <= 2 s <= M - N, so that the identity case s = 0 (I = A^2 embedded at the pupil's
 * place) can be checked on the CUDA path; such a handle serves pwfs_debug_intensity
 * only (pwfs_run returns PWFS_EINVAL). */
int pwfs_debug_create(const pwfs_params *p, const pwfs_ext *x, int32_t mask_shift_px, pwfs_t **out);
int pwfs_debug_intensity(pwfs_t *h, const float *d_phase, int32_t B, float *d_intensity,
                         void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* PWFS_H */
