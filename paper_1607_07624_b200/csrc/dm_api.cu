// dm_api.cu -- deformable mirror (influence-function multiply) and integrator control: the C ABI of
// include/pwfs_dm.h and its kernels.
//
//   dm_kernel<FB>   phase[b][pix[p]] = beta phase + alpha sum_m ifs[m][p] cmd[b][m].  The matrix is
//                   [n_act][ldp] row-major, so the OUTPUT index p is the contiguous one: a thread owns 4
//                   consecutive pixels (one 128-bit load per actuator, streamed with evict-first) and FB
//                   frames, the commands of a block of actuators sit in shared memory (broadcast reads).
//                   Loads are issued 8 actuators ahead of their FMAs.  HBM-bound: 4 bytes per matrix
//                   element per group of FB <= 8 frames; a closed loop (B = sensor instances per step)
//                   streams the matrix once per step.  The actuator range is split over gridDim.z so that
//                   a few thousand pixel columns still fill the machine; the partial sums meet in
//   dm_fold_kernel  phase = beta phase + alpha (part[0] + part[1] + ...), fixed order: deterministic.
//   int_kernel      one CTA: c += gain * delta; ring[t % (d+1)] = c; out = ring[(t - d) % (d+1)] or 0.
#include "../../include/pwfs_dm.h"

#include <cuda_runtime.h>

#include "device_guard.cuh"

#include <algorithm>
#include <cmath>
#include <new>
#include <vector>

namespace {

constexpr int kDmThreads = 128;
constexpr int kDmChunk = 256;     // actuators whose commands are staged in shared memory at a time
constexpr int kDmAhead = 8;       // independent 128-bit loads in flight per thread

// grid (ceil(ldp / 4 / kDmThreads), ceil(B / FB), msplit).  msplit == 1: writes the phase itself; else the partial
// sums part[z][b][p] of actuators [z n_act / msplit, (z + 1) n_act / msplit), folded by dm_fold_kernel.
template <int FB>
__global__ void __launch_bounds__(kDmThreads)
dm_kernel(const float *__restrict__ ifs, int n_act, int ldp, const int *__restrict__ pix, int n_pix, int npx2,
          const float *__restrict__ cmd, int B, float *__restrict__ phase, float alpha, int accumulate,
          float *__restrict__ part) {
    __shared__ float s_cmd[FB][kDmChunk];
    const int p4 = (blockIdx.x * kDmThreads + threadIdx.x) * 4;
    const int b0 = blockIdx.y * FB;
    const bool live = p4 < ldp;
    const float4 *col = reinterpret_cast<const float4 *>(ifs + (live ? p4 : 0));
    const int ld4 = ldp >> 2;
    float acc[FB][4];
#pragma unroll
    for (int f = 0; f < FB; ++f)
#pragma unroll
        for (int q = 0; q < 4; ++q) acc[f][q] = 0.f;
    const int m_lo = (int)(((long long)blockIdx.z * n_act) / gridDim.z), m_hi = (int)(((long long)(blockIdx.z + 1) * n_act) / gridDim.z);
    for (int m0 = m_lo; m0 < m_hi; m0 += kDmChunk) {
        const int mc = min(kDmChunk, m_hi - m0);
        __syncthreads();                                   // the previous chunk's commands are no longer read
        for (int i = threadIdx.x; i < FB * kDmChunk; i += kDmThreads) {
            const int f = i / kDmChunk, mm = i - f * kDmChunk;
            s_cmd[f][mm] = (mm < mc && b0 + f < B) ? __ldg(cmd + (size_t)(b0 + f) * n_act + m0 + mm) : 0.f;
        }
        __syncthreads();
        if (live) {
            for (int mm = 0; mm < mc; mm += kDmAhead) {
                float4 v[kDmAhead];
#pragma unroll
                for (int u = 0; u < kDmAhead; ++u)
                    v[u] = mm + u < mc ? __ldcs(col + (size_t)(m0 + mm + u) * ld4) : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
                for (int u = 0; u < kDmAhead; ++u)
#pragma unroll
                    for (int f = 0; f < FB; ++f) {
                        const float c = s_cmd[f][mm + u];           // zero beyond mc / B
                        acc[f][0] = fmaf(v[u].x, c, acc[f][0]);
                        acc[f][1] = fmaf(v[u].y, c, acc[f][1]);
                        acc[f][2] = fmaf(v[u].z, c, acc[f][2]);
                        acc[f][3] = fmaf(v[u].w, c, acc[f][3]);
                    }
            }
        }
    }
    if (!live) return;
    if (gridDim.z > 1) {                                   // partial sums, folded in a fixed order afterwards
#pragma unroll
        for (int f = 0; f < FB; ++f)
            if (b0 + f < B)
                *reinterpret_cast<float4 *>(part + ((size_t)blockIdx.z * B + b0 + f) * ldp + p4) =
                    make_float4(acc[f][0], acc[f][1], acc[f][2], acc[f][3]);
        return;
    }
    int idx[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) idx[q] = p4 + q < n_pix ? __ldg(pix + p4 + q) : -1;
#pragma unroll
    for (int f = 0; f < FB; ++f) {
        if (b0 + f >= B) break;
        float *out = phase + (size_t)(b0 + f) * npx2;
#pragma unroll
        for (int q = 0; q < 4; ++q)
            if (idx[q] >= 0) out[idx[q]] = accumulate ? fmaf(alpha, acc[f][q], out[idx[q]]) : alpha * acc[f][q];
    }
}

// grid (ceil(n_pix / 256), B)
__global__ void __launch_bounds__(256)
dm_fold_kernel(const float *__restrict__ part, int msplit, int ldp, const int *__restrict__ pix, int n_pix, int npx2, int B,
               float *__restrict__ phase, float alpha, int accumulate) {
    const int p = blockIdx.x * blockDim.x + threadIdx.x, b = blockIdx.y;
    if (p >= n_pix) return;
    float s = 0.f;
    for (int z = 0; z < msplit; ++z) s += __ldg(part + ((size_t)z * B + b) * ldp + p);
    float *out = phase + (size_t)b * npx2 + __ldg(pix + p);
    *out = accumulate ? fmaf(alpha, s, *out) : alpha * s;
}

// one CTA of 256 threads; t lives on the device (graph replays advance it)
__global__ void __launch_bounds__(256)
int_kernel(int n, int delay, const float *__restrict__ gain, float *__restrict__ state, float *__restrict__ ring,
           unsigned long long *__restrict__ t_ptr, const float *__restrict__ delta, float *__restrict__ cmd) {
    const unsigned long long t = *t_ptr;
    const int depth = delay + 1;
    const int wr = (int)(t % (unsigned long long)depth);
    const int rd = (int)((t + 1ull) % (unsigned long long)depth);      // slot written at step t - delay (depth = delay + 1)
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
        const float c = fmaf(__ldg(gain + i), __ldg(delta + i), state[i]);
        state[i] = c;
        ring[(size_t)wr * n + i] = c;
        cmd[i] = (t >= (unsigned long long)delay) ? ring[(size_t)rd * n + i] : 0.f;   // rd == wr when delay == 0
    }
    __syncthreads();
    if (threadIdx.x == 0) *t_ptr = t + 1ull;
}

int cuda_rc(cudaError_t e) { return e == cudaErrorMemoryAllocation ? PWFS_ENOMEM : PWFS_ECUDA; }

}  // namespace

constexpr int kDmMaxFrames = 8;   // frames per register tile (and per partial-sum buffer)

struct pwfs_dm {
    int device = 0, n_act = 0, n_pupil = 0, n_pix = 0, ldp = 0;
    int msplit = 1;                 // actuator-range split (fixed at create: results do not depend on the batch)
    float *d_ifs = nullptr;
    int *d_pix = nullptr;
    float *d_part = nullptr;        // [msplit][kDmMaxFrames][ldp]
};

struct pwfs_int {
    int device = 0, n = 0, delay = 0;
    float *d_gain = nullptr, *d_state = nullptr, *d_ring = nullptr;
    unsigned long long *d_t = nullptr;
};

extern "C" {

int pwfs_dm_create(int32_t n_act, int32_t n_pupil, int32_t n_pix, const int32_t *h_pix, const float *h_ifs,
                   int32_t device, pwfs_dm_t **out) {
    if (out) *out = nullptr;
    if (!out || !h_pix || !h_ifs || n_act < 1 || n_pupil < 1 || n_pix < 1) return PWFS_EINVAL;
    const long long npx2 = (long long)n_pupil * n_pupil;
    if (n_pix > npx2) return PWFS_EINVAL;
    std::vector<unsigned char> seen((size_t)npx2, 0);
    for (int p = 0; p < n_pix; ++p) {
        if (h_pix[p] < 0 || h_pix[p] >= npx2 || seen[h_pix[p]]) return PWFS_EINVAL;
        seen[h_pix[p]] = 1;
    }
    for (size_t i = 0; i < (size_t)n_act * n_pix; ++i)
        if (!std::isfinite(h_ifs[i])) return PWFS_EINVAL;
    pwfs_dm *h = new (std::nothrow) pwfs_dm();
    if (!h) return PWFS_ENOMEM;
    h->device = device; h->n_act = n_act; h->n_pupil = n_pupil; h->n_pix = n_pix; h->ldp = (n_pix + 3) / 4 * 4;
    pwk::DeviceGuard dg(device);
    cudaError_t e = dg.err;
    const size_t bytes = (size_t)n_act * h->ldp * sizeof(float);
    if (e == cudaSuccess) e = cudaMalloc((void **)&h->d_ifs, bytes);
    if (e == cudaSuccess && h->ldp != n_pix) e = cudaMemset(h->d_ifs, 0, bytes);
    if (e == cudaSuccess)
        e = cudaMemcpy2D(h->d_ifs, (size_t)h->ldp * sizeof(float), h_ifs, (size_t)n_pix * sizeof(float),
                         (size_t)n_pix * sizeof(float), (size_t)n_act, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMalloc((void **)&h->d_pix, (size_t)n_pix * sizeof(int));
    if (e == cudaSuccess) e = cudaMemcpy(h->d_pix, h_pix, (size_t)n_pix * sizeof(int), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
        // enough CTAs for ~12 per SM (128 threads, 32 registers: the loads in flight are what hides HBM latency), at
        // least 32 actuators per part
        int sms = 148;
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
        const int gx = (h->ldp / 4 + kDmThreads - 1) / kDmThreads;
        h->msplit = std::max(1, std::min(std::min(n_act / 32, 64), (12 * sms + gx - 1) / gx));
        if (h->msplit > 1) e = cudaMalloc((void **)&h->d_part, (size_t)h->msplit * kDmMaxFrames * h->ldp * sizeof(float));
    }
    if (e != cudaSuccess) { const int rc = cuda_rc(e); pwfs_dm_destroy(h); return rc; }
    *out = h;
    return PWFS_OK;
}

int pwfs_dm_apply(pwfs_dm_t *h, const float *d_cmd, int32_t B, float *d_phase, float alpha, float beta,
                  void *cuda_stream) {
    if (!h || B < 0 || !(beta == 0.f || beta == 1.f) || !std::isfinite(alpha)) return PWFS_EINVAL;
    if (B == 0) return PWFS_OK;
    if (!d_cmd || !d_phase) return PWFS_EINVAL;
    pwk::DeviceGuard dg(h->device);
    if (dg.err != cudaSuccess) return PWFS_ECUDA;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int npx2 = h->n_pupil * h->n_pupil, acc = beta == 1.f ? 1 : 0;
    if (!acc && cudaMemsetAsync(d_phase, 0, (size_t)B * npx2 * sizeof(float), st) != cudaSuccess) return PWFS_ECUDA;
    const unsigned gx = (unsigned)((h->ldp / 4 + kDmThreads - 1) / kDmThreads);
    // frames per register tile: the whole batch when it is small (the matrix is then streamed once)
    int FB = 1;
    while (FB < B && FB < kDmMaxFrames) FB *= 2;
    const int ms = h->msplit;
    const int step = ms > 1 ? kDmMaxFrames : 65535 * FB;               // partial buffer holds 8 frames; grid.y limit
    for (int b0 = 0; b0 < B; b0 += step) {
        const int Bc = std::min(B - b0, step);
        const dim3 grid(gx, (unsigned)((Bc + FB - 1) / FB), (unsigned)ms);
        const float *c = d_cmd + (size_t)b0 * h->n_act;
        float *ph = d_phase + (size_t)b0 * npx2;
        switch (FB) {
            case 1: dm_kernel<1><<<grid, kDmThreads, 0, st>>>(h->d_ifs, h->n_act, h->ldp, h->d_pix, h->n_pix, npx2, c, Bc, ph, alpha, acc, h->d_part); break;
            case 2: dm_kernel<2><<<grid, kDmThreads, 0, st>>>(h->d_ifs, h->n_act, h->ldp, h->d_pix, h->n_pix, npx2, c, Bc, ph, alpha, acc, h->d_part); break;
            case 4: dm_kernel<4><<<grid, kDmThreads, 0, st>>>(h->d_ifs, h->n_act, h->ldp, h->d_pix, h->n_pix, npx2, c, Bc, ph, alpha, acc, h->d_part); break;
            default: dm_kernel<8><<<grid, kDmThreads, 0, st>>>(h->d_ifs, h->n_act, h->ldp, h->d_pix, h->n_pix, npx2, c, Bc, ph, alpha, acc, h->d_part); break;
        }
        if (ms > 1)
            dm_fold_kernel<<<dim3((unsigned)((h->n_pix + 255) / 256), (unsigned)Bc), 256, 0, st>>>(
                h->d_part, ms, h->ldp, h->d_pix, h->n_pix, npx2, Bc, ph, alpha, acc);
    }
    return cudaGetLastError() == cudaSuccess ? PWFS_OK : PWFS_ECUDA;
}

void pwfs_dm_destroy(pwfs_dm_t *h) {
    if (!h) return;
    pwk::DeviceGuard dg(h->device);
    if (h->d_ifs) cudaFree(h->d_ifs);
    if (h->d_pix) cudaFree(h->d_pix);
    if (h->d_part) cudaFree(h->d_part);
    delete h;
}

int pwfs_int_create(int32_t n_modes, const float *h_gain, int32_t delay, int32_t device, pwfs_int_t **out) {
    if (out) *out = nullptr;
    if (!out || !h_gain || n_modes < 1 || delay < 0 || delay > 4096) return PWFS_EINVAL;
    for (int i = 0; i < n_modes; ++i)
        if (!std::isfinite(h_gain[i])) return PWFS_EINVAL;
    pwfs_int *h = new (std::nothrow) pwfs_int();
    if (!h) return PWFS_ENOMEM;
    h->device = device; h->n = n_modes; h->delay = delay;
    pwk::DeviceGuard dg(device);
    cudaError_t e = dg.err;
    const size_t nb = (size_t)n_modes * sizeof(float);
    if (e == cudaSuccess) e = cudaMalloc((void **)&h->d_gain, nb);
    if (e == cudaSuccess) e = cudaMemcpy(h->d_gain, h_gain, nb, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMalloc((void **)&h->d_state, nb);
    if (e == cudaSuccess) e = cudaMalloc((void **)&h->d_ring, nb * (size_t)(delay + 1));
    if (e == cudaSuccess) e = cudaMalloc((void **)&h->d_t, sizeof(unsigned long long));
    if (e == cudaSuccess) e = cudaMemset(h->d_state, 0, nb);
    if (e == cudaSuccess) e = cudaMemset(h->d_ring, 0, nb * (size_t)(delay + 1));
    if (e == cudaSuccess) e = cudaMemset(h->d_t, 0, sizeof(unsigned long long));
    if (e != cudaSuccess) { const int rc = cuda_rc(e); pwfs_int_destroy(h); return rc; }
    *out = h;
    return PWFS_OK;
}

int pwfs_int_step(pwfs_int_t *h, const float *d_delta, float *d_cmd, void *cuda_stream) {
    if (!h || !d_delta || !d_cmd) return PWFS_EINVAL;
    pwk::DeviceGuard dg(h->device);
    if (dg.err != cudaSuccess) return PWFS_ECUDA;
    int_kernel<<<1, 256, 0, (cudaStream_t)cuda_stream>>>(h->n, h->delay, h->d_gain, h->d_state, h->d_ring, h->d_t, d_delta, d_cmd);
    return cudaGetLastError() == cudaSuccess ? PWFS_OK : PWFS_ECUDA;
}

int pwfs_int_reset(pwfs_int_t *h, void *cuda_stream) {
    if (!h) return PWFS_EINVAL;
    pwk::DeviceGuard dg(h->device);
    if (dg.err != cudaSuccess) return PWFS_ECUDA;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t nb = (size_t)h->n * sizeof(float);
    cudaError_t e = cudaMemsetAsync(h->d_state, 0, nb, st);
    if (e == cudaSuccess) e = cudaMemsetAsync(h->d_ring, 0, nb * (size_t)(h->delay + 1), st);
    if (e == cudaSuccess) e = cudaMemsetAsync(h->d_t, 0, sizeof(unsigned long long), st);
    return e == cudaSuccess ? PWFS_OK : PWFS_ECUDA;
}

void pwfs_int_destroy(pwfs_int_t *h) {
    if (!h) return;
    pwk::DeviceGuard dg(h->device);
    if (h->d_gain) cudaFree(h->d_gain);
    if (h->d_state) cudaFree(h->d_state);
    if (h->d_ring) cudaFree(h->d_ring);
    if (h->d_t) cudaFree(h->d_t);
    delete h;
}

}  // extern "C"
