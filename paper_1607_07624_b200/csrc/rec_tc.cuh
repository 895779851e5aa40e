// rec_tc.cuh -- internal interface of the tensor-core batched reconstructor (rec_tc.cu), used by
// chain_api.cu's pwfs_rec_* calls.  Not part of the C ABI.
#pragma once
#include <cuda_runtime.h>

struct RecTc;   // opaque: TF32 planes of recmat, slope planes, split-K partials, TMA descriptors

// Describes d_R ([n_modes][ldk] FP32 on `device`, ldk % 4 == 0) to TMA; launches nothing and allocates nothing on the
// device.  Returns 0 or a PWFS_* error code; *out = nullptr on failure.
int rec_tc_create(RecTc **out, const float *d_R, int n_modes, int n_slopes, int ldk, int device, int num_sms);

// Sizes the slope planes / split-K partials for batches of up to B frames.  PWFS_EINVAL while `st` is being captured
// and buffers would have to grow.
int rec_tc_reserve(RecTc *h, int B, cudaStream_t st);

// modes[b][m] = sum_j recmat[m][j] slopes[b][j] for B frames, asynchronous on `st`.
// Grows its slope/partial scratch (rec_tc_reserve) when B exceeds what it has been sized for.
int rec_tc_run(RecTc *h, const float *d_slopes, int B, float *d_modes, cudaStream_t st);

void rec_tc_destroy(RecTc *h);
