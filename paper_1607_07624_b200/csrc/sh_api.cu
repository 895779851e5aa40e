// sh_api.cu -- f4, Shack-Hartmann: C ABI of include/pwfs_sh.h and its kernel.
//
// Both DFTs of a subaperture are b-term direct sums against one table W[t][c] =
// exp(-2 pi i (c - Pc/2 + 1/2) t / P), t < b, c < Pc = n_px * bin (the kept, fftshifted columns with the
// half-pixel centring folded in): H = g W along x, spot = |W^T H|^2 along y.  b <= 16 and P <= 64, so
// direct sums beat any FFT staging; the whole subaperture costs b Pc (b + Pc) complex FMAs.
//
// sh_kernel<B, NC>: LPS = 2^k lanes own one subaperture, each lane NC adjacent columns c, so a warp
// works on 32 / LPS neighbouring subapertures of one lenslet row (coalesced phase rows in, coalesced
// detector rows out).
//   1. phasor of the b x b pupil pixels (range-reduced MUFU sincos) -> shared memory, stored as
//      (re, re, im, im) so that one LDS.128 feeds two FFMA2;
//   2. along x: the lane keeps its NC columns of W in registers and accumulates H[y][c] for all y
//      in registers: one g load per 2 NC FFMA2;
//   3. along y: for each kept row v the b table entries W[y][v] are warp-uniform loads, again one per
//      2 NC FFMA2; |.|^2 / P^2 falls out in the lane that owns the column;
//   4. bin x bin sums (rows in the lane, columns through a per-warp row buffer), detector window
//      written from registers, centre of gravity reduced over the LPS lanes by shuffles.
// A complex sum  sum a w  is kept as two packed accumulators P = sum re(a) w, Q = sum im(a) w and
// folded once at the end (P.x - Q.y, P.y + Q.x): two FFMA2 per complex FMA, no operand shuffling.
// HBM sees the phase once and the frame once.
#include "../../include/pwfs_sh.h"

#include <cuda_runtime.h>

#include "device_guard.cuh"

#include <algorithm>
#include <cmath>
#include <cstring>
#include <new>
#include <vector>

namespace {

constexpr int kShWarps = 4;
constexpr int kMaxB = 16, kMaxP = 64;
constexpr size_t kShSmemBudget = 160 * 1024;
constexpr float kInv2PiHiS = 0.15915493667125702f;
constexpr float kInv2PiLoS = 6.4206382e-09f;

struct ShDev {
    int N, n_sub, b, P, n_px, bin, Pc;
    int lg_lps;              // log2 of the lanes that share one subaperture
    int gpitch;              // float4 per subaperture in the phasor buffer (b*b padded to 1 mod 8)
    int gpr;                 // warp tasks per lenslet row = ceil(n_sub / (32 >> lg_lps))
    int vec;                 // 1: detector rows may be stored NC-wide (alignment holds)
    float scale, invP2;
    const float *amp;        // [N][N]
    const float4 *wtab;      // [b][Pc] (re, re, im, im) of W[t][c]
    const int2 *pix;         // [b * b * SPW] pixel map of a warp task (see sh_kernel, step 1)
    const int *vslot;        // [n_sub^2] slope slot of a valid subaperture, -1 otherwise
    int n_valid;
};

__device__ __forceinline__ float2 lo2(float4 v) { return make_float2(v.x, v.y); }
__device__ __forceinline__ float2 hi2(float4 v) { return make_float2(v.z, v.w); }

// One detector row of one subaperture from the lane's NC adjacent FFT columns when BIN divides NC:
// NO = NC / BIN detector pixels starting at col * NO, stored NO-wide when `vec` says the alignment holds.
template <int NC, int BIN>
__device__ __forceinline__ void emit_row(float (&racc)[NC], float *row, int col, int n_px, bool live, int vec,
                                         float c0, float fy, float &tot, float &mx, float &my) {
    if constexpr (NC % BIN == 0) {
        constexpr int NO = NC / BIN;
        float v[NO];
#pragma unroll
        for (int k = 0; k < NO; ++k) {
            float a = 0.f;
#pragma unroll
            for (int x = 0; x < BIN; ++x) a += racc[k * BIN + x];
            v[k] = col * NO + k < n_px ? a : 0.f;
        }
#pragma unroll
        for (int j = 0; j < NC; ++j) racc[j] = 0.f;
        if (live) {
            if (NO == 4 && vec && col * NO + NO <= n_px) {
                *reinterpret_cast<float4 *>(row + col * NO) = make_float4(v[0], v[1], v[2], v[3]);
            } else if (NO == 2 && vec && col * NO + NO <= n_px) {
                *reinterpret_cast<float2 *>(row + col * NO) = make_float2(v[0], v[1]);
            } else {
#pragma unroll
                for (int k = 0; k < NO; ++k) if (col * NO + k < n_px) row[col * NO + k] = v[k];
            }
        }
#pragma unroll
        for (int k = 0; k < NO; ++k) {
            tot += v[k];
            mx = fmaf((float)(col * NO + k) - c0, v[k], mx);
            my = fmaf(fy, v[k], my);
        }
    }
}

// grid (ceil(n_sub * gpr / kShWarps), F); block 32 * kShWarps;
// dynamic smem: W[B][Pc] float4, then per warp the phasor buffer [SPW][gpitch] float4 and a row buffer [32 NC] float.
template <int B, int NC>
__global__ void __launch_bounds__(32 * kShWarps, (B * NC <= 24) ? 4 : 2)
sh_kernel(ShDev t, const float *__restrict__ phase, float *__restrict__ frames, float *__restrict__ slopes) {
    extern __shared__ float4 sh_smem[];
    const int lane = threadIdx.x & 31, wl = threadIdx.x >> 5;
    const int Pc = t.Pc, lgL = t.lg_lps, lgS = 5 - lgL, LPS = 1 << lgL, SPW = 1 << lgS;
    float4 *s_w = sh_smem;                                                    // [B][Pc]
    float4 *g = s_w + B * Pc + (size_t)wl * ((size_t)SPW * t.gpitch + 8 * NC); // [SPW][gpitch]
    float *rowbuf = reinterpret_cast<float *>(g + (size_t)SPW * t.gpitch);    // [32 NC]
    for (int i = threadIdx.x; i < B * Pc; i += blockDim.x) s_w[i] = __ldg(t.wtab + i);
    __syncthreads();
    const int task = blockIdx.x * kShWarps + wl, f = blockIdx.y;
    if (task >= t.n_sub * t.gpr) return;                                      // warp-uniform
    const int sj = task / t.gpr, si0 = (task - sj * t.gpr) << lgS;
    const int s = lane >> lgL, col = lane & (LPS - 1), si = si0 + s;

    // 1. phasor (F4f): rows of SPW * B contiguous pupil pixels
    {
        const int rowlen = B << lgS;
        const float *ph0 = phase + ((size_t)f * t.N + (size_t)sj * B) * t.N + (size_t)si0 * B;
        const float *am0 = t.amp + ((size_t)sj * B) * t.N + (size_t)si0 * B;
        const int xmax = t.N - si0 * B;                                       // pixels left in this pupil row
        constexpr int U = 4;                                                  // loads of U rounds in flight
        const int rawlen = B * rowlen;
        for (int e0 = lane; e0 < rawlen; e0 += 32 * U) {
            float ph[U], am[U];
            int dst[U];
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int e = e0 + 32 * u;
                // pixel e of the task: .x = y * N + sx (offset in the pupil), .y = sx << 16 | slot in the phasor buffer
                const int2 m = e < rawlen ? __ldg(t.pix + e) : make_int2(0, 0x7fff0000);
                const bool in = (m.y >> 16) < xmax;
                dst[u] = e < rawlen ? (m.y & 0xffff) : -1;
                ph[u] = in ? __ldg(ph0 + m.x) : 0.f;
                am[u] = in ? __ldg(am0 + m.x) : 0.f;
            }
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const float p = ph[u] * t.scale;
                const float q = rintf(p * kInv2PiHiS);
                float tr = fmaf(p, kInv2PiHiS, -q);
                tr = fmaf(p, kInv2PiLoS, tr);
                float sn, cs;
                __sincosf(tr * 6.283185307179586f, &sn, &cs);
                const float re = am[u] * cs, im = am[u] * sn;
                if (dst[u] >= 0) g[dst[u]] = make_float4(re, re, im, im);
            }
        }
    }
    // the lane's NC columns of W
    float2 Wl[NC][B];
#pragma unroll
    for (int j = 0; j < NC; ++j) {
        const int uc = min(col * NC + j, Pc - 1);
#pragma unroll
        for (int x = 0; x < B; ++x) { const float4 w = s_w[x * Pc + uc]; Wl[j][x] = make_float2(w.x, w.z); }
    }
    __syncwarp();
    // 2. along x: H[y][c] = sum_x g[y][x] W[x][c]
    float2 H[NC][B];
    {
        const float4 *gs = g + s * t.gpitch;
#pragma unroll
        for (int y = 0; y < B; ++y) {
            float2 Pa[NC], Qa[NC];
#pragma unroll
            for (int j = 0; j < NC; ++j) Pa[j] = Qa[j] = make_float2(0.f, 0.f);
#pragma unroll
            for (int x = 0; x < B; ++x) {
                const float4 a = gs[y * B + x];
#pragma unroll
                for (int j = 0; j < NC; ++j) {
                    Pa[j] = __ffma2_rn(lo2(a), Wl[j][x], Pa[j]);
                    Qa[j] = __ffma2_rn(hi2(a), Wl[j][x], Qa[j]);
                }
            }
#pragma unroll
            for (int j = 0; j < NC; ++j) H[j][y] = make_float2(Pa[j].x - Qa[j].y, Pa[j].y + Qa[j].x);
        }
    }
    // 3./4. along y, |.|^2 / P^2, detector window (F4g), centre of gravity (F4i)
    const int n_px = t.n_px, bin = t.bin, D = t.n_sub * n_px;
    const bool live = si < t.n_sub;
    float *win = frames + ((size_t)f * D + (size_t)sj * n_px) * D + (size_t)min(si, t.n_sub - 1) * n_px;
    const float c0 = 0.5f * (float)(n_px - 1);
    float tot = 0.f, mx = 0.f, my = 0.f;
    float racc[NC];
#pragma unroll
    for (int j = 0; j < NC; ++j) racc[j] = 0.f;
    int cnt = 0, py = 0;
    for (int vc = 0; vc < Pc; ++vc) {
        float2 Pa[NC], Qa[NC];
#pragma unroll
        for (int j = 0; j < NC; ++j) Pa[j] = Qa[j] = make_float2(0.f, 0.f);
#pragma unroll
        for (int y = 0; y < B; ++y) {
            const float4 w = s_w[y * Pc + vc];
#pragma unroll
            for (int j = 0; j < NC; ++j) {
                Pa[j] = __ffma2_rn(lo2(w), H[j][y], Pa[j]);
                Qa[j] = __ffma2_rn(hi2(w), H[j][y], Qa[j]);
            }
        }
#pragma unroll
        for (int j = 0; j < NC; ++j) {
            const float er = Pa[j].x - Qa[j].y, ei = Pa[j].y + Qa[j].x;
            racc[j] += fmaf(er, er, ei * ei) * t.invP2;
        }
        if (++cnt < bin) continue;
        cnt = 0;
        const float fy = (float)py - c0;
        if (bin == 1) {                                                       // detector pixel = FFT pixel
            emit_row<NC, 1>(racc, win + (size_t)py * D, col, n_px, live, t.vec, c0, fy, tot, mx, my);
        } else if (bin == 2 && NC % 2 == 0) {                                 // column pairs live in one lane
            emit_row<NC, 2>(racc, win + (size_t)py * D, col, n_px, live, t.vec, c0, fy, tot, mx, my);
        } else if (bin == 4 && NC == 4) {
            emit_row<NC, 4>(racc, win + (size_t)py * D, col, n_px, live, t.vec, c0, fy, tot, mx, my);
        } else {                                                              // columns through the row buffer
            float *rb = rowbuf + s * (LPS * NC);
#pragma unroll
            for (int j = 0; j < NC; ++j) { rb[col * NC + j] = racc[j]; racc[j] = 0.f; }
            __syncwarp();
            for (int px = col; px < n_px; px += LPS) {
                float v = 0.f;
                for (int xx = 0; xx < bin; ++xx) v += rb[px * bin + xx];
                if (live) win[(size_t)py * D + px] = v;
                tot += v;
                mx = fmaf((float)px - c0, v, mx);
                my = fmaf(fy, v, my);
            }
            __syncwarp();
        }
        ++py;
    }
    if (slopes) {
        for (int o = LPS >> 1; o > 0; o >>= 1) {
            tot += __shfl_xor_sync(0xffffffffu, tot, o);
            mx += __shfl_xor_sync(0xffffffffu, mx, o);
            my += __shfl_xor_sync(0xffffffffu, my, o);
        }
        if (live && col == 0) {
            const int slot = __ldg(t.vslot + sj * t.n_sub + si);
            if (slot >= 0) {
                float *out = slopes + (size_t)f * 2 * t.n_valid;
                out[slot] = mx / tot;
                out[t.n_valid + slot] = my / tot;
            }
        }
    }
}

using ShKernel = void (*)(ShDev, const float *, float *, float *);

template <int B>
ShKernel sh_pick_nc(int nc) {
    if constexpr (B <= 8) { if (nc == 4) return sh_kernel<B, 4>; }
    return nc >= 2 ? sh_kernel<B, 2> : sh_kernel<B, 1>;
}

ShKernel sh_pick(int b, int nc) {
    switch (b) {
#define SH_CASE(B_) case B_: return sh_pick_nc<B_>(nc);
        SH_CASE(1) SH_CASE(2) SH_CASE(3) SH_CASE(4) SH_CASE(5) SH_CASE(6) SH_CASE(7) SH_CASE(8)
        SH_CASE(9) SH_CASE(10) SH_CASE(11) SH_CASE(12) SH_CASE(13) SH_CASE(14) SH_CASE(15) SH_CASE(16)
#undef SH_CASE
    }
    return nullptr;
}

int cuda_rc(cudaError_t e) { return e == cudaErrorMemoryAllocation ? PWFS_ENOMEM : PWFS_ECUDA; }

}  // namespace

struct pwfs_sh {
    int device = 0;
    ShDev dev{};
    ShKernel kernel = nullptr;
    int nc = 1;
    size_t smem = 0;
    std::vector<uint8_t> valid;
    float *d_amp = nullptr;
    float4 *d_wtab = nullptr;
    int2 *d_pix = nullptr;
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
    // W[t][c] = exp(-2 pi i (2 (c - Pc/2) + 1) t / (2P)), argument reduced in integers
    std::vector<float4> wtab((size_t)b * Pc);
    for (int tt = 0; tt < b; ++tt)
        for (int c = 0; c < (int)Pc; ++c) {
            long long m = ((2LL * (c - Pc / 2) + 1) * tt) % (2LL * P);
            if (m < 0) m += 2LL * P;
            const double a = -3.14159265358979323846264338327950288 * (double)m / (double)P;
            const float wr = (float)std::cos(a), wi = (float)std::sin(a);
            wtab[(size_t)tt * Pc + c] = make_float4(wr, wr, wi, wi);
        }
    // columns per lane, lanes per subaperture (a power of two), subapertures per warp
    const int nc = (b <= 8 && Pc >= 16) ? 4 : (Pc >= 4 ? 2 : 1);
    int lg = 0;
    while ((nc << lg) < Pc) ++lg;                                  // Pc <= 64 = 2 * 32 -> lg <= 5
    const int gpitch = ((b * b + 6) / 8) * 8 + 1;                  // = 1 mod 8: subapertures land on distinct banks
    auto smem_of = [&](int l) {
        return ((size_t)b * Pc + (size_t)kShWarps * ((size_t)(32 >> l) * gpitch + 8 * nc)) * sizeof(float4);
    };
    while (lg < 5 && smem_of(lg) > kShSmemBudget) ++lg;            // large b with a tiny window: fewer subapertures per warp
    pwfs_sh *h = new (std::nothrow) pwfs_sh();
    if (!h) return PWFS_ENOMEM;
    h->device = p->device;
    h->valid = valid;
    h->nc = nc;
    h->kernel = sh_pick(b, nc);
    h->smem = smem_of(lg);
    pwk::DeviceGuard dg(p->device);
    cudaError_t e = dg.err;
    if (e == cudaSuccess) e = cudaMalloc((void **)&h->d_amp, (size_t)N * N * sizeof(float));
    if (e == cudaSuccess) e = cudaMemcpy(h->d_amp, p->pupil_amp, (size_t)N * N * sizeof(float), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMalloc((void **)&h->d_wtab, wtab.size() * sizeof(float4));
    if (e == cudaSuccess) e = cudaMemcpy(h->d_wtab, wtab.data(), wtab.size() * sizeof(float4), cudaMemcpyHostToDevice);
    // pixel map of a warp task: element e = y * (SPW b) + sx of its SPW b x b pixels -> pupil offset and buffer slot
    const int spw = 32 >> lg, rowlen = b * spw;
    std::vector<int2> pix((size_t)b * rowlen);
    for (int y = 0; y < b; ++y)
        for (int sx = 0; sx < rowlen; ++sx) {
            const int ss = sx / b, x = sx - ss * b;
            pix[(size_t)y * rowlen + sx] = make_int2(y * N + sx, (sx << 16) | (ss * gpitch + y * b + x));
        }
    if (e == cudaSuccess) e = cudaMalloc((void **)&h->d_pix, pix.size() * sizeof(int2));
    if (e == cudaSuccess) e = cudaMemcpy(h->d_pix, pix.data(), pix.size() * sizeof(int2), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMalloc((void **)&h->d_vslot, vslot.size() * sizeof(int));
    if (e == cudaSuccess) e = cudaMemcpy(h->d_vslot, vslot.data(), vslot.size() * sizeof(int), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaFuncSetAttribute((const void *)h->kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->smem);
    if (e != cudaSuccess) { int rc = cuda_rc(e); pwfs_sh_destroy(h); return rc; }
    ShDev &d = h->dev;
    d.N = N; d.n_sub = ns; d.b = b; d.P = P; d.n_px = p->n_px; d.bin = p->bin; d.Pc = (int)Pc;
    d.lg_lps = lg; d.gpitch = gpitch; d.gpr = (ns + (32 >> lg) - 1) / (32 >> lg);
    d.vec = (nc % p->bin == 0 && p->n_px % (nc / p->bin) == 0) ? 1 : 0;   // NO-wide stores stay aligned
    d.scale = p->phase_scale; d.invP2 = (float)(1.0 / ((double)P * P));
    d.amp = h->d_amp; d.wtab = h->d_wtab; d.pix = h->d_pix; d.vslot = h->d_vslot; d.n_valid = nv;
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
    pwk::DeviceGuard dg(h->device);
    if (dg.err != cudaSuccess) return PWFS_ECUDA;
    ShDev d = h->dev;
    const int tasks = d.n_sub * d.gpr, D = d.n_sub * d.n_px;
    const size_t NN = (size_t)d.N * d.N, DD = (size_t)D * D;
    if ((uintptr_t)d_frames % 16 != 0) d.vec = 0;                  // NC-wide stores need the caller's buffer aligned
    for (int f0 = 0; f0 < B; f0 += 65535) {
        const int Fc = B - f0 < 65535 ? B - f0 : 65535;
        h->kernel<<<dim3((tasks + kShWarps - 1) / kShWarps, Fc), 32 * kShWarps, h->smem, (cudaStream_t)cuda_stream>>>(
            d, d_phase + (size_t)f0 * NN, d_frames + (size_t)f0 * DD,
            d_slopes ? d_slopes + (size_t)f0 * 2 * d.n_valid : nullptr);
    }
    return cudaGetLastError() == cudaSuccess ? PWFS_OK : PWFS_ECUDA;
}

void pwfs_sh_destroy(pwfs_sh_t *h) {
    if (!h) return;
    pwk::DeviceGuard dg(h->device);
    if (h->d_amp) cudaFree(h->d_amp);
    if (h->d_wtab) cudaFree(h->d_wtab);
    if (h->d_pix) cudaFree(h->d_pix);
    if (h->d_vslot) cudaFree(h->d_vslot);
    delete h;
}

}  // extern "C"
