// atmo_api.cu -- f1: propagation through phase screens, C ABI of
// include/pwfs_atmo.h and its one kernel.  HBM/L2-bound: per output frame it writes
// N*N floats per wavelength and reads L (N+1)^2 screen samples, which stay resident in L2
// (a few screens of 4 MB each against 126 MB).
#include "../../include/pwfs_atmo.h"

#include <cuda_runtime.h>

#include "device_guard.cuh"

#include <cmath>
#include <new>
#include <vector>

namespace {

constexpr int kTX = 4, kTY = 4;          // outputs per thread
constexpr int kBX = 32, kBY = 8;         // threads per CTA  ->  CTA tile 128 x 32 outputs
constexpr int kMaxLayers = 16;

struct AtmoDev {
    int L, G, S, W, N;
    double inv_pitch;
    const float *screens;    // [L][G][G]
    const double *layer;     // [L][3]  vx, vy, height
    const double *dirs;      // [S][2]  tan_x, tan_y
    const float *wl;         // [W]
};

// grid (ceil(N/128), ceil(N/32), n_steps*S); block (32, 8).  F1a-F1d of pwfs_atmo.h.
// All pixels of a frame share the fractional offsets of a layer, so the bilinear sample is a
// separable 2-tap filter: a thread loads a 5 x 5 patch and produces 4 x 4 outputs.
__global__ void __launch_bounds__(kBX *kBY)
atmo_propagate_kernel(AtmoDev a, long long first_step, double dt, float *__restrict__ out) {
    __shared__ int s_ix[kMaxLayers], s_iy[kMaxLayers];
    __shared__ float s_fx[kMaxLayers], s_fy[kMaxLayers];
    const int fr = blockIdx.z, step = fr / a.S, d = fr % a.S;
    const int tid = threadIdx.y * kBX + threadIdx.x;
    if (tid < a.L) {
        // F1a in double: the shift can be thousands of pixels and its fraction matters
        const double t = (double)(first_step + step) * dt;
        const double sx = (-a.layer[3 * tid + 0] * t + a.layer[3 * tid + 2] * a.dirs[2 * d + 0]) * a.inv_pitch;
        const double sy = (-a.layer[3 * tid + 1] * t + a.layer[3 * tid + 2] * a.dirs[2 * d + 1]) * a.inv_pitch;
        const double flx = floor(sx), fly = floor(sy);
        s_fx[tid] = (float)(sx - flx);
        s_fy[tid] = (float)(sy - fly);
        const double G = (double)a.G;
        s_ix[tid] = (int)(flx - floor(flx / G) * G);     // floor(sx) mod G, in [0, G)
        s_iy[tid] = (int)(fly - floor(fly / G) * G);
    }
    __syncthreads();
    const int x0 = (blockIdx.x * kBX + threadIdx.x) * kTX;
    const int y0 = (blockIdx.y * kBY + threadIdx.y) * kTY;
    if (x0 >= a.N || y0 >= a.N) return;
    float acc[kTY][kTX];
#pragma unroll
    for (int j = 0; j < kTY; ++j)
#pragma unroll
        for (int i = 0; i < kTX; ++i) acc[j][i] = 0.f;
    const int G = a.G;
    for (int l = 0; l < a.L; ++l) {
        const float *scr = a.screens + (size_t)l * G * G;
        const float fx = s_fx[l], fy = s_fy[l];
        int c[kTX + 1], r[kTY + 1];
        c[0] = (s_ix[l] + x0) % G;
        r[0] = (s_iy[l] + y0) % G;
#pragma unroll
        for (int i = 1; i <= kTX; ++i) c[i] = (c[i - 1] + 1 == G) ? 0 : c[i - 1] + 1;
#pragma unroll
        for (int j = 1; j <= kTY; ++j) r[j] = (r[j - 1] + 1 == G) ? 0 : r[j - 1] + 1;
        float h[kTY + 1][kTX];     // F1b along x
#pragma unroll
        for (int j = 0; j <= kTY; ++j) {
            const float *row = scr + (size_t)r[j] * G;
            float v[kTX + 1];
#pragma unroll
            for (int i = 0; i <= kTX; ++i) v[i] = __ldg(row + c[i]);
#pragma unroll
            for (int i = 0; i < kTX; ++i) h[j][i] = fmaf(fx, v[i + 1] - v[i], v[i]);
        }
#pragma unroll
        for (int j = 0; j < kTY; ++j)   // F1b along y, F1c layer sum
#pragma unroll
            for (int i = 0; i < kTX; ++i) acc[j][i] += fmaf(fy, h[j + 1][i] - h[j][i], h[j][i]);
    }
    const size_t NN = (size_t)a.N * a.N;
    const bool vec = (a.N % 4 == 0);
    for (int w = 0; w < a.W; ++w) {     // F1c wavelength scale, F1d order
        const float sc = __ldg(a.wl + w);
        float *dst = out + ((size_t)fr * a.W + w) * NN;
#pragma unroll
        for (int j = 0; j < kTY; ++j) {
            const int y = y0 + j;
            if (y >= a.N) break;
            float *p = dst + (size_t)y * a.N + x0;
            if (vec) {
                *reinterpret_cast<float4 *>(p) = make_float4(acc[j][0] * sc, acc[j][1] * sc, acc[j][2] * sc, acc[j][3] * sc);
            } else {
#pragma unroll
                for (int i = 0; i < kTX; ++i)
                    if (x0 + i < a.N) p[i] = acc[j][i] * sc;
            }
        }
    }
}

}  // namespace

struct pwfs_atmo {
    int device = 0;
    AtmoDev dev{};
    std::vector<void *> allocs;
    int last_cuda = 0;
};

namespace {
template <typename T>
int put(pwfs_atmo *h, const T *src, size_t n, const T **dst) {
    void *d = nullptr;
    cudaError_t e = cudaMalloc(&d, n * sizeof(T));
    if (e != cudaSuccess) { h->last_cuda = (int)e; return e == cudaErrorMemoryAllocation ? PWFS_ENOMEM : PWFS_ECUDA; }
    h->allocs.push_back(d);
    e = cudaMemcpy(d, src, n * sizeof(T), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) { h->last_cuda = (int)e; return PWFS_ECUDA; }
    *dst = (const T *)d;
    return PWFS_OK;
}
}  // namespace

extern "C" {

int pwfs_atmo_create(const pwfs_atmo_params *p, pwfs_atmo_t **out) {
    if (out) *out = nullptr;
    if (!p || !out || !p->screens || !p->wind_vxy || !p->heights || !p->dirs_tan || !p->wl_scale) return PWFS_EINVAL;
    if (p->n_layers < 1 || p->n_layers > kMaxLayers || p->n_dirs < 1 || p->n_wl < 1) return PWFS_EINVAL;
    if (p->n_pupil < 1 || p->screen_px < p->n_pupil || p->screen_px < 2) return PWFS_EINVAL;
    if (!(p->pitch > 0.0) || !std::isfinite(p->pitch)) return PWFS_EINVAL;
    std::vector<double> layer((size_t)3 * p->n_layers);
    for (int l = 0; l < p->n_layers; ++l) {
        layer[3 * l + 0] = p->wind_vxy[2 * l + 0];
        layer[3 * l + 1] = p->wind_vxy[2 * l + 1];
        layer[3 * l + 2] = p->heights[l];
        for (int c = 0; c < 3; ++c)
            if (!std::isfinite(layer[3 * l + c])) return PWFS_EINVAL;
    }
    for (int i = 0; i < 2 * p->n_dirs; ++i)
        if (!std::isfinite(p->dirs_tan[i])) return PWFS_EINVAL;
    std::vector<float> wl(p->n_wl);
    for (int w = 0; w < p->n_wl; ++w) {
        if (!std::isfinite(p->wl_scale[w])) return PWFS_EINVAL;
        wl[w] = (float)p->wl_scale[w];
    }
    pwfs_atmo *h = new (std::nothrow) pwfs_atmo();
    if (!h) return PWFS_ENOMEM;
    h->device = p->device;
    int rc = PWFS_OK;
    pwk::DeviceGuard dg(p->device);
    cudaError_t e = dg.err;
    if (e != cudaSuccess) { h->last_cuda = (int)e; rc = PWFS_ECUDA; }
    AtmoDev &a = h->dev;
    a.L = p->n_layers; a.G = p->screen_px; a.S = p->n_dirs; a.W = p->n_wl; a.N = p->n_pupil;
    a.inv_pitch = 1.0 / p->pitch;
    if (!rc) rc = put(h, p->screens, (size_t)a.L * a.G * a.G, &a.screens);
    if (!rc) rc = put(h, layer.data(), layer.size(), &a.layer);
    if (!rc) rc = put(h, p->dirs_tan, (size_t)2 * a.S, &a.dirs);
    if (!rc) rc = put(h, wl.data(), wl.size(), &a.wl);
    if (rc) { pwfs_atmo_destroy(h); return rc; }
    *out = h;
    return PWFS_OK;
}

int pwfs_atmo_frames_per_step(const pwfs_atmo_t *h, int32_t *frames) {
    if (!h || !frames) return PWFS_EINVAL;
    *frames = h->dev.S * h->dev.W;
    return PWFS_OK;
}

int pwfs_atmo_propagate(pwfs_atmo_t *h, int64_t first_step, int32_t n_steps, double dt, float *d_phase,
                        void *cuda_stream) {
    if (!h || n_steps < 0 || !std::isfinite(dt)) return PWFS_EINVAL;
    if (n_steps == 0) return PWFS_OK;
    if (!d_phase) return PWFS_EINVAL;
    pwk::DeviceGuard dg(h->device);
    cudaError_t e = dg.err;
    if (e != cudaSuccess) { h->last_cuda = (int)e; return PWFS_ECUDA; }
    const AtmoDev &a = h->dev;
    const int per_launch = 65535 / a.S;                  // grid.z limit
    if (per_launch < 1) return PWFS_EINVAL;
    const size_t step_elems = (size_t)a.S * a.W * a.N * a.N;
    for (int s0 = 0; s0 < n_steps; s0 += per_launch) {
        const int ns = n_steps - s0 < per_launch ? n_steps - s0 : per_launch;
        dim3 grid((a.N + kBX * kTX - 1) / (kBX * kTX), (a.N + kBY * kTY - 1) / (kBY * kTY), ns * a.S);
        atmo_propagate_kernel<<<grid, dim3(kBX, kBY), 0, (cudaStream_t)cuda_stream>>>(
            a, (long long)first_step + s0, dt, d_phase + (size_t)s0 * step_elems);
    }
    e = cudaGetLastError();
    if (e != cudaSuccess) { h->last_cuda = (int)e; return PWFS_ECUDA; }
    return PWFS_OK;
}

void pwfs_atmo_destroy(pwfs_atmo_t *h) {
    if (!h) return;
    pwk::DeviceGuard dg(h->device);
    for (void *d : h->allocs) cudaFree(d);
    delete h;
}

}  // extern "C"
