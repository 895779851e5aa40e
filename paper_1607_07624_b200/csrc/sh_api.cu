// sh_api.cu -- f4, Shack-Hartmann: C ABI of include/pwfs_sh.h and its kernel.
//
// One warp = one subaperture of one frame, everything in shared memory:
//   1. phasor of the b x b pupil pixels (range-reduced MUFU sincos),
//   2. DFT along x to the Pc = n_px * bin kept columns only (b inputs each: direct sums against
//      a 2P-entry twiddle table that carries the half-pixel centring),
//   3. DFT along y to the Pc kept rows, |.|^2 / P^2,
//   4. bin x bin sums -> the subaperture's detector window, centre of gravity -> slopes.
// b <= 16 and P <= 64, so a transform is at most 16 terms: direct sums beat any FFT staging, and
// the whole subaperture costs b Pc (b + Pc) complex FMAs.  HBM sees the phase once and the frame
// once; the kernel is bound by those bytes for small P and by FP32 FMAs for large P.
#include "../../include/pwfs_sh.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstring>
#include <new>
#include <vector>

namespace {

constexpr int kShWarps = 4;
constexpr int kMaxB = 16, kMaxP = 64;
constexpr float kInv2PiHiS = 0.15915493667125702f;
constexpr float kInv2PiLoS = 6.4206382e-09f;

struct ShDev {
    int N, n_sub, b, P, n_px, bin, Pc;
    float scale, invP2;
    const float *amp;        // [N][N]
    const float2 *tw;        // [2P] exp(-2 pi i m / (2P))
    const int *vslot;        // [n_sub^2] slope slot of a valid subaperture, -1 otherwise
    int n_valid;
};

__host__ __device__ inline size_t sh_warp_floats(int b, int Pc) {
    return (size_t)2 * b * b + (size_t)2 * b * Pc + (size_t)Pc * Pc;
}

__device__ __forceinline__ float2 cfma(float2 a, float2 w, float2 acc) {   // acc + a * w
    acc.x = fmaf(a.x, w.x, acc.x); acc.x = fmaf(-a.y, w.y, acc.x);
    acc.y = fmaf(a.x, w.y, acc.y); acc.y = fmaf(a.y, w.x, acc.y);
    return acc;
}

// grid (ceil(n_sub^2 / kShWarps), F); block 32 * kShWarps; dynamic smem: tw[2P] + per-warp buffers.
__global__ void __launch_bounds__(32 * kShWarps)
sh_kernel(ShDev t, const float *__restrict__ phase, float *__restrict__ frames, float *__restrict__ slopes) {
    extern __shared__ float2 sh_smem[];
    float2 *s_tw = sh_smem;
    const int lane = threadIdx.x & 31, wl = threadIdx.x >> 5;
    const int b = t.b, P = t.P, Pc = t.Pc, P2 = 2 * t.P;
    float *wbase = reinterpret_cast<float *>(sh_smem + P2) + (size_t)wl * sh_warp_floats(b, Pc);
    float2 *g = reinterpret_cast<float2 *>(wbase);                 // [b][b]
    float2 *H = g + b * b;                                         // [b][Pc]
    float *spot = reinterpret_cast<float *>(H + b * Pc);           // [Pc][Pc]
    for (int i = threadIdx.x; i < P2; i += blockDim.x) s_tw[i] = __ldg(t.tw + i);
    __syncthreads();
    const int sub = blockIdx.x * kShWarps + wl, f = blockIdx.y;
    if (sub >= t.n_sub * t.n_sub) return;
    const int sj = sub / t.n_sub, si = sub - sj * t.n_sub;

    // 1. phasor (F4f)
    const float *ph0 = phase + ((size_t)f * t.N + (size_t)sj * b) * t.N + (size_t)si * b;
    const float *am0 = t.amp + ((size_t)sj * b) * t.N + (size_t)si * b;
    for (int e = lane; e < b * b; e += 32) {
        const int y = e / b, x = e - y * b;
        const float ph = __ldg(ph0 + (size_t)y * t.N + x) * t.scale;
        const float am = __ldg(am0 + (size_t)y * t.N + x);
        const float q = rintf(ph * kInv2PiHiS);
        float tr = fmaf(ph, kInv2PiHiS, -q);
        tr = fmaf(ph, kInv2PiLoS, tr);
        float sn, cs;
        __sincosf(tr * 6.283185307179586f, &sn, &cs);
        g[e] = make_float2(am * cs, am * sn);
    }
    __syncwarp();
    // 2. along x: H[y][uc] = sum_x g[y][x] exp(-2 pi i (u~ + 1/2) x / P), u~ = uc - Pc/2 (fftshifted crop)
    for (int e = lane; e < b * Pc; e += 32) {
        const int y = e / Pc, uc = e - y * Pc;
        int step = (2 * (uc - Pc / 2) + 1) % P2;
        if (step < 0) step += P2;
        float2 acc = make_float2(0.f, 0.f);
        int m = 0;
        for (int x = 0; x < b; ++x) {
            acc = cfma(g[y * b + x], s_tw[m], acc);
            m += step;
            if (m >= P2) m -= P2;
        }
        H[e] = acc;
    }
    __syncwarp();
    // 3. along y, |.|^2 / P^2
    for (int e = lane; e < Pc * Pc; e += 32) {
        const int vc = e / Pc, uc = e - vc * Pc;
        int step = (2 * (vc - Pc / 2) + 1) % P2;
        if (step < 0) step += P2;
        float2 acc = make_float2(0.f, 0.f);
        int m = 0;
        for (int y = 0; y < b; ++y) {
            acc = cfma(H[y * Pc + uc], s_tw[m], acc);
            m += step;
            if (m >= P2) m -= P2;
        }
        spot[e] = fmaf(acc.x, acc.x, acc.y * acc.y) * t.invP2;
    }
    __syncwarp();
    // 4. detector window (F4g) and centre of gravity (F4i)
    const int n_px = t.n_px, bin = t.bin, D = t.n_sub * n_px;
    float *win = frames + ((size_t)f * D + (size_t)sj * n_px) * D + (size_t)si * n_px;
    const float c0 = 0.5f * (float)(n_px - 1);
    float tot = 0.f, mx = 0.f, my = 0.f;
    for (int e = lane; e < n_px * n_px; e += 32) {
        const int py = e / n_px, px = e - py * n_px;
        float s = 0.f;
        for (int yy = 0; yy < bin; ++yy)
            for (int xx = 0; xx < bin; ++xx) s += spot[(py * bin + yy) * Pc + px * bin + xx];
        win[(size_t)py * D + px] = s;
        tot += s;
        mx = fmaf((float)px - c0, s, mx);
        my = fmaf((float)py - c0, s, my);
    }
    if (slopes) {
        const int slot = __ldg(t.vslot + sub);
        if (slot >= 0) {                                           // warp-uniform
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                tot += __shfl_xor_sync(0xffffffffu, tot, o);
                mx += __shfl_xor_sync(0xffffffffu, mx, o);
                my += __shfl_xor_sync(0xffffffffu, my, o);
            }
            if (lane == 0) {
                float *out = slopes + (size_t)f * 2 * t.n_valid;
                out[slot] = mx / tot;
                out[t.n_valid + slot] = my / tot;
            }
        }
    }
}

int cuda_rc(cudaError_t e) { return e == cudaErrorMemoryAllocation ? PWFS_ENOMEM : PWFS_ECUDA; }

}  // namespace

struct pwfs_sh {
    int device = 0;
    ShDev dev{};
    size_t smem = 0;
    std::vector<uint8_t> valid;
    float *d_amp = nullptr;
    float2 *d_tw = nullptr;
    int *d_vslot = nullptr;
};

extern "C" {

int pwfs_sh_create(const pwfs_sh_params *p, pwfs_sh_t **out) {
    if (out) *out = nullptr;
    if (!p || !out || !p->pupil_amp) return PWFS_EINVAL;
    const int N = p->n_pupil, ns = p->n_subap, P = p->fft_px;
    if (N < 1 || ns < 1 || N % ns != 0 || !std::isfinite(p->phase_scale)) return PWFS_EINVAL;
    const int b = N / ns;
    if (P < 2 || P % 2 || P < b || p->n_px < 1 || p->bin < 1) return PWFS_EINVAL;
    const long long Pc = (long long)p->n_px * p->bin;
    if (Pc > P || (P - Pc) % 2) return PWFS_EINVAL;
    if (b > kMaxB || P > kMaxP) return PWFS_EUNSUPPORTED;
    const double thresh = p->illum_thresh > 0.f ? (double)p->illum_thresh : 0.5;
    double amax2 = 0.0;
    for (size_t i = 0; i < (size_t)N * N; ++i) {
        const double a = p->pupil_amp[i];
        if (!(a >= 0.0) || !std::isfinite(a)) return PWFS_EINVAL;
        amax2 = std::max(amax2, a * a);
    }
    if (!(amax2 > 0.0)) return PWFS_EINVAL;
    // F4h
    std::vector<uint8_t> valid((size_t)ns * ns, 0);
    std::vector<int> vslot((size_t)ns * ns, -1);
    int nv = 0;
    for (int j = 0; j < ns; ++j)
        for (int i = 0; i < ns; ++i) {
            double lit = 0.0;
            for (int y = 0; y < b; ++y)
                for (int x = 0; x < b; ++x) {
                    const double a = p->pupil_amp[(size_t)(j * b + y) * N + i * b + x];
                    lit += a * a;
                }
            if (lit >= thresh * b * b * amax2) { valid[(size_t)j * ns + i] = 1; vslot[(size_t)j * ns + i] = nv++; }
        }
    if (nv == 0) return PWFS_EINVAL;
    std::vector<float2> tw((size_t)2 * P);
    for (int m = 0; m < 2 * P; ++m) {
        const double a = -3.14159265358979323846264338327950288 * (double)m / (double)P;
        tw[m] = make_float2((float)std::cos(a), (float)std::sin(a));
    }
    pwfs_sh *h = new (std::nothrow) pwfs_sh();
    if (!h) return PWFS_ENOMEM;
    h->device = p->device;
    h->valid = valid;
    h->smem = (size_t)2 * P * sizeof(float2) + kShWarps * sh_warp_floats(b, (int)Pc) * sizeof(float);
    cudaError_t e = cudaSetDevice(p->device);
    if (e == cudaSuccess) e = cudaMalloc((void **)&h->d_amp, (size_t)N * N * sizeof(float));
    if (e == cudaSuccess) e = cudaMemcpy(h->d_amp, p->pupil_amp, (size_t)N * N * sizeof(float), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMalloc((void **)&h->d_tw, tw.size() * sizeof(float2));
    if (e == cudaSuccess) e = cudaMemcpy(h->d_tw, tw.data(), tw.size() * sizeof(float2), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMalloc((void **)&h->d_vslot, vslot.size() * sizeof(int));
    if (e == cudaSuccess) e = cudaMemcpy(h->d_vslot, vslot.data(), vslot.size() * sizeof(int), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(sh_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->smem);
    if (e != cudaSuccess) { int rc = cuda_rc(e); pwfs_sh_destroy(h); return rc; }
    ShDev &d = h->dev;
    d.N = N; d.n_sub = ns; d.b = b; d.P = P; d.n_px = p->n_px; d.bin = p->bin; d.Pc = (int)Pc;
    d.scale = p->phase_scale; d.invP2 = (float)(1.0 / ((double)P * P));
    d.amp = h->d_amp; d.tw = h->d_tw; d.vslot = h->d_vslot; d.n_valid = nv;
    *out = h;
    return PWFS_OK;
}

int pwfs_sh_info(const pwfs_sh_t *h, int32_t *det_size, int32_t *n_valid) {
    if (!h) return PWFS_EINVAL;
    if (det_size) *det_size = h->dev.n_sub * h->dev.n_px;
    if (n_valid) *n_valid = h->dev.n_valid;
    return PWFS_OK;
}

int pwfs_sh_valid_mask(const pwfs_sh_t *h, uint8_t *host_mask) {
    if (!h || !host_mask) return PWFS_EINVAL;
    std::memcpy(host_mask, h->valid.data(), h->valid.size());
    return PWFS_OK;
}

int pwfs_sh_run(pwfs_sh_t *h, const float *d_phase, int32_t B, float *d_frames, float *d_slopes, void *cuda_stream) {
    if (!h || B < 0) return PWFS_EINVAL;
    if (B == 0) return PWFS_OK;
    if (!d_phase || !d_frames) return PWFS_EINVAL;
    if (cudaSetDevice(h->device) != cudaSuccess) return PWFS_ECUDA;
    const ShDev &d = h->dev;
    const int subs = d.n_sub * d.n_sub, D = d.n_sub * d.n_px;
    const size_t NN = (size_t)d.N * d.N, DD = (size_t)D * D;
    for (int f0 = 0; f0 < B; f0 += 65535) {
        const int Fc = B - f0 < 65535 ? B - f0 : 65535;
        sh_kernel<<<dim3((subs + kShWarps - 1) / kShWarps, Fc), 32 * kShWarps, h->smem, (cudaStream_t)cuda_stream>>>(
            d, d_phase + (size_t)f0 * NN, d_frames + (size_t)f0 * DD,
            d_slopes ? d_slopes + (size_t)f0 * 2 * d.n_valid : nullptr);
    }
    return cudaGetLastError() == cudaSuccess ? PWFS_OK : PWFS_ECUDA;
}

void pwfs_sh_destroy(pwfs_sh_t *h) {
    if (!h) return;
    cudaSetDevice(h->device);
    if (h->d_amp) cudaFree(h->d_amp);
    if (h->d_tw) cudaFree(h->d_tw);
    if (h->d_vslot) cudaFree(h->d_vslot);
    delete h;
}

}  // extern "C"
