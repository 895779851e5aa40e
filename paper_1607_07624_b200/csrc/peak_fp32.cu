// peak_fp32.cu -- the FP32 "plain ALU" roofline denominator, MEASURED: a dependent-chain-free stream of FFMA
// (scalar) or FFMA2 (packed FP32x2, the instruction the FFT butterflies are written in) on every SM, timed with
// CUDA events.  SURVEY.md 8(d) asks for this number next to the derived 148 x 128 x 2 x f_SM figure; bench.py
// reports both (roofline.peak_measured, roofline.frac_vs_measured).  Not part of the hot path and not part of
// libpwfs.so: built into its own small library, libpwfs_peak.so, which only bench.py loads.
#include "../../include/pwfs.h"        // status codes
#include "../../include/pwfs_peak.h"

#include <cuda_runtime.h>

#include <algorithm>

namespace {

constexpr int kChains = 8;        // independent accumulators per thread (float2 each: 16 lane-FMAs per round)
constexpr int kUnroll = 8;        // rounds per loop iteration
constexpr int kThreads = 256;

template <bool PACKED>
__global__ void __launch_bounds__(kThreads) fma_stream_kernel(float *out, int iters, float a, float b) {
    float2 x[kChains];
#pragma unroll
    for (int c = 0; c < kChains; ++c) x[c] = make_float2(1e-3f * (float)(threadIdx.x + c), 1e-3f * (float)(blockIdx.x + c));
    const float2 a2 = make_float2(a, a), b2 = make_float2(b, b);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < kUnroll; ++u)
#pragma unroll
            for (int c = 0; c < kChains; ++c) {
                if constexpr (PACKED) {
                    x[c] = __ffma2_rn(x[c], a2, b2);
                } else {
                    x[c].x = fmaf(x[c].x, a, b);
                    x[c].y = fmaf(x[c].y, a, b);
                }
            }
    }
    float s = 0.f;
#pragma unroll
    for (int c = 0; c < kChains; ++c) s += x[c].x + x[c].y;
    out[(size_t)blockIdx.x * kThreads + threadIdx.x] = s;
}

}  // namespace

extern "C" int pwfs_peak_fp32(int32_t device, int32_t packed, double *tflops, double *elapsed_ms) {
    if (!tflops) return PWFS_EINVAL;
    int prev = -1;
    cudaGetDevice(&prev);
    if (cudaSetDevice(device) != cudaSuccess) return PWFS_ECUDA;
    int rc = PWFS_OK;
    cudaDeviceProp prop;
    float *out = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) rc = PWFS_ECUDA;
    const int blocks = rc ? 0 : prop.multiProcessorCount * (2048 / kThreads);   // every SM full: 64 warps
    const int iters = 4096;
    if (!rc && cudaMalloc((void **)&out, (size_t)blocks * kThreads * sizeof(float)) != cudaSuccess) rc = PWFS_ENOMEM;
    if (!rc && (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess)) rc = PWFS_ECUDA;
    double best_ms = 1e300;
    for (int rep = 0; !rc && rep < 6; ++rep) {          // first repetition is the warm-up
        cudaEventRecord(e0, 0);
        if (packed) fma_stream_kernel<true><<<blocks, kThreads>>>(out, iters, 0.999f, 1e-4f);
        else fma_stream_kernel<false><<<blocks, kThreads>>>(out, iters, 0.999f, 1e-4f);
        cudaEventRecord(e1, 0);
        if (cudaEventSynchronize(e1) != cudaSuccess || cudaGetLastError() != cudaSuccess) { rc = PWFS_ECUDA; break; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0) best_ms = std::min(best_ms, (double)ms);
    }
    if (!rc) {
        const double flop = 2.0 * (double)blocks * kThreads * (double)iters * kUnroll * kChains * 2.0;
        *tflops = flop / (best_ms * 1e-3) / 1e12;
        if (elapsed_ms) *elapsed_ms = best_ms;
    }
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    if (out) cudaFree(out);
    if (prev >= 0 && prev != device) cudaSetDevice(prev);
    return rc;
}
