// chain_api.cu -- f2: CCD detector, slope computer with reference vector,
// modal reconstructor; the C ABI of include/pwfs_chain.h and its kernels.
//
//   ccd_kernel      one thread per detector pixel: integrate n_int steps, quantum efficiency,
//                   Philox4x32-10 -> Poisson / normal photon noise, read noise.  All decisions
//                   in double (B200 keeps full-rate FP64 units; the detector is <= 184^2 px).
//                   HBM-bound: 4 n_int bytes in, 4 bytes out per pixel.
//   slopec_kernel   one cluster of 8 CTAs per frame: normalisation sum over valid subapertures through
//                   distributed shared memory, slopes - sn.
//   rec_kernel      modes = slopes x recmat^T.  One warp = MR rows of recmat x FB frames, lanes
//                   stride over the slope index with 128-bit loads, FP32 FMA, shuffle reduction.
//                   B = 1 is a GEMV streaming recmat once from HBM; larger batches re-use each
//                   recmat line for FB frames out of registers.
#include "../../include/pwfs_chain.h"
#include "rec_tc.cuh"

#include <cooperative_groups.h>
#include <cuda_runtime.h>

#include "device_guard.cuh"

#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

namespace {

// ------------------------------------------------------------------ Philox ---
// Philox4x32-10 (Salmon et al., SC'11): counter (c0..c3), key (k0, k1) -> 4 words.
struct U4 { unsigned x, y, z, w; };

__device__ __forceinline__ U4 philox4x32_10(U4 c, unsigned k0, unsigned k1) {
    constexpr unsigned M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const unsigned hi0 = __umulhi(M0, c.x), lo0 = M0 * c.x;
        const unsigned hi1 = __umulhi(M1, c.z), lo1 = M1 * c.z;
        c = U4{hi1 ^ c.y ^ k0, lo1, hi0 ^ c.w ^ k1, lo0};
        k0 += W0;
        k1 += W1;
    }
    return c;
}

__device__ __forceinline__ double u01(unsigned r) { return ((double)r + 0.5) * (1.0 / 4294967296.0); }

// z = sqrt(-2 ln ua) cos(2 pi ub), written without contraction so that the value is the
// same expression tree as the definition (F2e)
__device__ __forceinline__ double box_muller(double ua, double ub) {
    const double rad = sqrt(__dmul_rn(-2.0, log(ua)));
    const double ang = __dmul_rn(6.283185307179586476925286766559, ub);
    return __dmul_rn(rad, cos(ang));
}

// The read-noise deviate only has to reach the pixel within a float ulp (it is added to the count and rounded to
// float): cos(2 pi ub) is taken as cospi(2 ub) -- no multiply by a rounded 2 pi, no Payne-Hanek range reduction.
__device__ __forceinline__ double box_muller_readout(double ua, double ub) {
    const double rad = sqrt(__dmul_rn(-2.0, log(ua)));
    return __dmul_rn(rad, cospi(__dadd_rn(ub, ub)));
}

struct CcdDev {
    int D, n_inst, n_int;
    double qe_gain, ron;
    int photon, readout;
    unsigned k0, k1;
    const double *rcp;     // [kPoissonMaxN + 1] rcp[n] = RN(1 / n), correctly rounded on the host (rcp[0] unused)
};

constexpr int kPoissonMaxN = 4096;

// RN(a / n) for 0 < a < 2^10 and an integer 1 <= n <= 4096 held as the double nd, with y = RN(1 / n) from the table:
// two Newton steps on the quotient and Markstein's final correction -- q1 is within one ulp of a / n (its error before
// rounding is O(2^-104)), the residual r1 = a - n q1 is exact in one FMA, and RN(q1 + r1 y) is then the correctly
// rounded quotient (Markstein 1990).  Five FP64 pipe operations instead of the ~25 of the generic __ddiv_rn (which
// also handles subnormals, infinities and exponent extremes that cannot occur here); the photon counts stay
// bit-identical to the oracle's IEEE division (tests/test_gpu_chain.py compares millions of pixels exactly).
__device__ __forceinline__ double div_small_int(double a, double nd, double y) {
    const double q0 = __dmul_rn(a, y);
    const double r0 = __fma_rn(-nd, q0, a);
    const double q1 = __fma_rn(r0, y, q0);
    const double r1 = __fma_rn(-nd, q1, a);
    return __fma_rn(r1, y, q1);
}

constexpr double kPoissonSwitch = 128.0;   // F2c

__global__ void __launch_bounds__(256)
ccd_kernel(CcdDev c, const float *__restrict__ frames, long long n_out, long long first_out,
           float *__restrict__ pix) {
    const long long DD = (long long)c.D * c.D;
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= n_out * DD) return;
    const long long p = idx / DD;
    const int px = (int)(idx - p * DD);
    const long long ostep = p / c.n_inst;
    const int inst = (int)(p - ostep * c.n_inst);
    // F2a: sum the n_int steps of this instance, in step order
    double acc = 0.0;
    const float *src = frames + ((size_t)(ostep * c.n_int) * c.n_inst + inst) * DD + px;
    for (int j = 0; j < c.n_int; ++j) acc = __dadd_rn(acc, (double)__ldg(src + (size_t)j * c.n_inst * DD));
    const double lam = __dmul_rn(c.qe_gain, acc);                      // F2b
    double k = lam;
    if (c.photon | c.readout) {
        const unsigned long long fi = (unsigned long long)(first_out + p);
        const U4 r = philox4x32_10(U4{(unsigned)px, (unsigned)fi, (unsigned)(fi >> 32), 0u}, c.k0, c.k1);
        if (c.photon) {                                                // F2c
            if (!(lam > 0.0)) {
                k = 0.0;
            } else if (lam < kPoissonSwitch) {
                const double u = u01(r.x);
                double pr = exp(-lam), s = pr, nd = 0.0;
                int n = 0;
                while (u > s && n < kPoissonMaxN) {
                    ++n;
                    nd = __dadd_rn(nd, 1.0);
                    pr = __dmul_rn(pr, div_small_int(lam, nd, __ldg(c.rcp + n)));
                    s = __dadd_rn(s, pr);
                }
                k = nd;
            } else {
                const double z = box_muller(u01(r.x), u01(r.y));
                k = fmax(0.0, floor(__dadd_rn(__dadd_rn(lam, __dmul_rn(sqrt(lam), z)), 0.5)));
            }
        }
        if (c.readout) k = __dadd_rn(k, __dmul_rn(c.ron, box_muller_readout(u01(r.z), u01(r.w))));   // F2d
    }
    pix[idx] = (float)k;
}

// ------------------------------------------------------------- slope computer ---
struct SlopecDev {
    int n_sub, n_valid, norm;
    const int *vidx;      // [n_valid] j * n_sub + i, row-major
    const float *sn;      // [2 n_valid] or nullptr
};

// One thread-block CLUSTER of kSlopecCluster CTAs per frame (grid (kSlopecCluster, B)): each CTA takes a contiguous
// share of the valid subapertures, the partial normalisation sums meet through distributed shared memory and every CTA
// adds them in rank order (same value in all of them, deterministic), then writes the slopes of its share.  One
// launch, no second pass through global memory, and a single frame (closed loop) is spread over 8 SMs.
constexpr int kSlopecCluster = 8;

__global__ void __cluster_dims__(kSlopecCluster, 1, 1) __launch_bounds__(256)
slopec_kernel(SlopecDev t, const float *__restrict__ pixels, float *__restrict__ slopes) {
    namespace cg = cooperative_groups;
    cg::cluster_group cluster = cg::this_cluster();
    __shared__ float red[8];
    __shared__ float s_part;
    const int ns = t.n_sub, D = 2 * ns, nv = t.n_valid;
    const int rank = (int)cluster.block_rank(), share = (nv + kSlopecCluster - 1) / kSlopecCluster;
    const int i_lo = rank * share, i_hi = min(nv, i_lo + share);
    const float *fr = pixels + (size_t)blockIdx.y * D * D;
    float part = 0.f;
    for (int i = i_lo + threadIdx.x; i < i_hi; i += blockDim.x) {
        const int id = __ldg(t.vidx + i), jj = id / ns, ii = id - jj * ns;
        part += (fr[jj * D + ii] + fr[jj * D + ns + ii]) + (fr[(ns + jj) * D + ii] + fr[(ns + jj) * D + ns + ii]);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = part;
    __syncthreads();
    if (threadIdx.x == 0) {
        float v = 0.f;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) v += red[w];
        s_part = v;
    }
    cluster.sync();                                                    // every CTA's partial is in its shared memory
    float nbar = 0.f;
    for (int r = 0; r < kSlopecCluster; ++r) nbar += *cluster.map_shared_rank(&s_part, r);
    nbar /= (float)nv;
    cluster.sync();                                                    // nobody leaves while its partial may still be read
    float *out = slopes + (size_t)blockIdx.y * 2 * nv;
    for (int i = i_lo + threadIdx.x; i < i_hi; i += blockDim.x) {
        const int id = __ldg(t.vidx + i), jj = id / ns, ii = id - jj * ns;
        const float a = fr[jj * D + ii], b = fr[jj * D + ns + ii];
        const float c = fr[(ns + jj) * D + ii], d = fr[(ns + jj) * D + ns + ii];
        const float den = t.norm == 1 ? ((a + b) + (c + d)) : nbar;
        float sx = ((a + c) - (b + d)) / den, sy = ((a + b) - (c + d)) / den;
        if (t.sn) { sx -= __ldg(t.sn + i); sy -= __ldg(t.sn + nv + i); }     // F2f
        out[i] = sx;
        out[nv + i] = sy;
    }
}

// --------------------------------------------------------------- reconstructor ---
constexpr int kRecWarps = 8;

// grid (ceil(n_modes / (kRecWarps * MR)), ceil(B / FB)); block 32 * kRecWarps.
// R: [n_modes][ldk] (ldk % 4 == 0, zero padded).  S: [B][ns].  VEC: S rows are 16-byte aligned.
template <int MR, int FB, bool VEC>
__global__ void __launch_bounds__(32 * kRecWarps)
rec_kernel(const float *__restrict__ R, int n_modes, int ldk, const float *__restrict__ S, int ns, int B,
           float *__restrict__ out) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int m0 = (blockIdx.x * kRecWarps + warp) * MR;
    const int b0 = blockIdx.y * FB;
    if (m0 >= n_modes) return;
    const float4 *rrow[MR];
#pragma unroll
    for (int r = 0; r < MR; ++r) rrow[r] = reinterpret_cast<const float4 *>(R + (size_t)min(m0 + r, n_modes - 1) * ldk);
    const float *srow[FB];
#pragma unroll
    for (int f = 0; f < FB; ++f) srow[f] = S + (size_t)min(b0 + f, B - 1) * ns;
    float acc[MR][FB];
#pragma unroll
    for (int r = 0; r < MR; ++r)
#pragma unroll
        for (int f = 0; f < FB; ++f) acc[r][f] = 0.f;
    const int n4 = ldk >> 2;
    for (int k4 = lane; k4 < n4; k4 += 32) {
        float4 rv[MR];
#pragma unroll
        for (int r = 0; r < MR; ++r) rv[r] = __ldg(rrow[r] + k4);
#pragma unroll
        for (int f = 0; f < FB; ++f) {
            float4 sv;
            if (VEC) {
                sv = __ldg(reinterpret_cast<const float4 *>(srow[f]) + k4);
            } else {
                const int k = 4 * k4;
                sv.x = k + 0 < ns ? __ldg(srow[f] + k + 0) : 0.f;
                sv.y = k + 1 < ns ? __ldg(srow[f] + k + 1) : 0.f;
                sv.z = k + 2 < ns ? __ldg(srow[f] + k + 2) : 0.f;
                sv.w = k + 3 < ns ? __ldg(srow[f] + k + 3) : 0.f;
            }
#pragma unroll
            for (int r = 0; r < MR; ++r) {
                acc[r][f] = fmaf(rv[r].x, sv.x, acc[r][f]);
                acc[r][f] = fmaf(rv[r].y, sv.y, acc[r][f]);
                acc[r][f] = fmaf(rv[r].z, sv.z, acc[r][f]);
                acc[r][f] = fmaf(rv[r].w, sv.w, acc[r][f]);
            }
        }
    }
#pragma unroll
    for (int r = 0; r < MR; ++r)
#pragma unroll
        for (int f = 0; f < FB; ++f) {
            float v = acc[r][f];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
            if (lane == 0 && m0 + r < n_modes && b0 + f < B) out[(size_t)(b0 + f) * n_modes + m0 + r] = v;
        }
}

// ---- single frame (closed loop): a pure stream of recmat, 4 bytes per element, HBM-bound -------------------------
// One CTA of 16 warps = one row of recmat at a time, each warp a contiguous sixteenth of the row; every thread keeps
// ITS slope values in registers for the whole launch (thread t always meets slope indices 4 (t + 512 i) .. + 3), so per
// row a thread issues NK independent 128-bit loads and 4 NK FMAs.  The loads of the CTA's NEXT row are issued before the
// current row is reduced, so the memory system always has one to two rows (up to 96 KB) per SM in flight and the
// per-row barrier costs nothing.  One CTA per SM, rows round-robin: thousands of rows leave no ragged last wave.
// Warp partials meet in shared memory and are added in warp order: deterministic.
constexpr int kGemvThreads = 512;

template <int NK>
__global__ void __launch_bounds__(kGemvThreads, 1)
rec_gemv_kernel(const float *__restrict__ R, int n_modes, int ldk, const float *__restrict__ S, int ns,
                float *__restrict__ out) {
    __shared__ float red[2][kGemvThreads / 32];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int n4 = ldk >> 2;
    float4 sv[NK];
#pragma unroll
    for (int i = 0; i < NK; ++i) {
        const int k = 4 * (tid + kGemvThreads * i);
        sv[i].x = k + 0 < ns ? __ldg(S + k + 0) : 0.f;
        sv[i].y = k + 1 < ns ? __ldg(S + k + 1) : 0.f;
        sv[i].z = k + 2 < ns ? __ldg(S + k + 2) : 0.f;
        sv[i].w = k + 3 < ns ? __ldg(S + k + 3) : 0.f;
    }
    float4 rv[NK], rn[NK];
    auto fetch = [&](float4 (&dst)[NK], int m) {
        const float4 *row = reinterpret_cast<const float4 *>(R + (size_t)m * ldk);
#pragma unroll
        for (int i = 0; i < NK; ++i) {
            const int k4 = tid + kGemvThreads * i;
            dst[i] = k4 < n4 ? __ldcs(row + k4) : make_float4(0.f, 0.f, 0.f, 0.f);      // streamed once: evict first
        }
    };
    int par = 0;
    if ((int)blockIdx.x < n_modes) fetch(rv, blockIdx.x);
    for (int m = blockIdx.x; m < n_modes; m += gridDim.x, par ^= 1) {
        const int m_next = m + gridDim.x;
        if (m_next < n_modes) fetch(rn, m_next);
        float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f;
#pragma unroll
        for (int i = 0; i < NK; ++i) {
            a0 = fmaf(rv[i].x, sv[i].x, a0);
            a1 = fmaf(rv[i].y, sv[i].y, a1);
            a2 = fmaf(rv[i].z, sv[i].z, a2);
            a3 = fmaf(rv[i].w, sv[i].w, a3);
        }
        float v = (a0 + a1) + (a2 + a3);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) red[par][warp] = v;
        __syncthreads();                         // red[par] complete; red[par ^ 1] is free again after the next barrier
        if (tid == 0) {
            float t = 0.f;
#pragma unroll
            for (int w = 0; w < kGemvThreads / 32; ++w) t += red[par][w];
            out[m] = t;
        }
#pragma unroll
        for (int i = 0; i < NK; ++i) rv[i] = rn[i];
    }
}

constexpr int kRecTcMinBatch = 24;              // below this the FP32 kernel's register tiles win
constexpr long long kRecTcMinElems = 1 << 16;   // recmat elements

template <int MR, int FB>
void launch_rec(bool vec, dim3 grid, cudaStream_t st, const float *R, int n_modes, int ldk, const float *S, int ns,
                int B, float *out) {
    if (vec) rec_kernel<MR, FB, true><<<grid, 32 * kRecWarps, 0, st>>>(R, n_modes, ldk, S, ns, B, out);
    else     rec_kernel<MR, FB, false><<<grid, 32 * kRecWarps, 0, st>>>(R, n_modes, ldk, S, ns, B, out);
}

template <int MR>
void launch_rec_fb(int FB, bool vec, cudaStream_t st, const float *R, int n_modes, int ldk, const float *S, int ns,
                   int B, float *out) {
    dim3 grid((n_modes + kRecWarps * MR - 1) / (kRecWarps * MR), (B + FB - 1) / FB);
    switch (FB) {
        case 1:  launch_rec<MR, 1>(vec, grid, st, R, n_modes, ldk, S, ns, B, out); break;
        case 2:  launch_rec<MR, 2>(vec, grid, st, R, n_modes, ldk, S, ns, B, out); break;
        case 4:  launch_rec<MR, 4>(vec, grid, st, R, n_modes, ldk, S, ns, B, out); break;
        case 8:  launch_rec<MR, 8>(vec, grid, st, R, n_modes, ldk, S, ns, B, out); break;
        default: launch_rec<MR, 16>(vec, grid, st, R, n_modes, ldk, S, ns, B, out); break;
    }
}

int cuda_rc(cudaError_t e) { return e == cudaErrorMemoryAllocation ? PWFS_ENOMEM : PWFS_ECUDA; }

}  // namespace

struct pwfs_ccd {
    int device = 0;
    CcdDev dev{};
    double *d_rcp = nullptr;
};

struct pwfs_slopec {
    int device = 0;
    SlopecDev dev{};
    int *d_vidx = nullptr;
    float *d_sn = nullptr;
};

struct pwfs_rec {
    int device = 0;
    int n_modes = 0, n_slopes = 0, ldk = 0;
    float *d_R = nullptr;
    int num_sms = 148;
    RecTc *tc = nullptr;       // tensor-core path for batches, built on the first batched call
    bool tc_off = false;       // PWFS_REC_TC=0, or the driver lacks cuTensorMapEncodeTiled
};

extern "C" {

// ------------------------------------------------------------------ CCD ---
int pwfs_ccd_create(const pwfs_ccd_params *p, pwfs_ccd_t **out) {
    if (out) *out = nullptr;
    if (!p || !out) return PWFS_EINVAL;
    if (p->det_size < 1 || p->n_inst < 1 || p->n_int < 1) return PWFS_EINVAL;
    if (!std::isfinite(p->gain) || p->gain < 0.0) return PWFS_EINVAL;
    if (!std::isfinite(p->quantum_eff) || p->quantum_eff < 0.0 || p->quantum_eff > 1.0) return PWFS_EINVAL;
    if (!std::isfinite(p->readout_level) || p->readout_level < 0.0) return PWFS_EINVAL;
    int count = 0;
    if (cudaGetDeviceCount(&count) != cudaSuccess || p->device < 0 || p->device >= count) return PWFS_ECUDA;
    pwfs_ccd *h = new (std::nothrow) pwfs_ccd();
    if (!h) return PWFS_ENOMEM;
    h->device = p->device;
    CcdDev &c = h->dev;
    c.D = p->det_size; c.n_inst = p->n_inst; c.n_int = p->n_int;
    c.qe_gain = p->quantum_eff * p->gain;
    c.ron = p->readout_level;
    c.photon = p->photon_noise != 0; c.readout = p->readout_noise != 0;
    c.k0 = (unsigned)(p->seed & 0xFFFFFFFFull); c.k1 = (unsigned)(p->seed >> 32);
    {
        std::vector<double> rcp(kPoissonMaxN + 1, 0.0);
        for (int n = 1; n <= kPoissonMaxN; ++n) rcp[n] = 1.0 / (double)n;       // IEEE division: correctly rounded
        pwk::DeviceGuard dg(p->device);
        cudaError_t e = dg.err;
        if (e == cudaSuccess) e = cudaMalloc((void **)&h->d_rcp, rcp.size() * sizeof(double));
        if (e == cudaSuccess) e = cudaMemcpy(h->d_rcp, rcp.data(), rcp.size() * sizeof(double), cudaMemcpyHostToDevice);
        if (e != cudaSuccess) { const int rc = cuda_rc(e); pwfs_ccd_destroy(h); return rc; }
        c.rcp = h->d_rcp;
    }
    *out = h;
    return PWFS_OK;
}

int pwfs_ccd_run(pwfs_ccd_t *h, const float *d_frames, int32_t n_steps, int64_t first_out_frame, float *d_pixels,
                 void *cuda_stream) {
    if (!h || n_steps < 0 || n_steps % h->dev.n_int != 0) return PWFS_EINVAL;
    if (n_steps == 0) return PWFS_OK;
    if (!d_frames || !d_pixels) return PWFS_EINVAL;
    pwk::DeviceGuard dg(h->device);
    if (dg.err != cudaSuccess) return PWFS_ECUDA;
    const long long n_out = (long long)(n_steps / h->dev.n_int) * h->dev.n_inst;
    const long long total = n_out * h->dev.D * h->dev.D;
    const long long blocks = (total + 255) / 256;
    if (blocks > 0x7fffffffLL) return PWFS_EINVAL;
    ccd_kernel<<<(unsigned)blocks, 256, 0, (cudaStream_t)cuda_stream>>>(h->dev, d_frames, n_out,
                                                                        (long long)first_out_frame, d_pixels);
    return cudaGetLastError() == cudaSuccess ? PWFS_OK : PWFS_ECUDA;
}

void pwfs_ccd_destroy(pwfs_ccd_t *h) {
    if (!h) return;
    if (h->d_rcp) {
        pwk::DeviceGuard dg(h->device);
        cudaFree(h->d_rcp);
    }
    delete h;
}

// ------------------------------------------------------- slope computer ---
int pwfs_slopec_create(int32_t n_sub, const uint8_t *h_valid, int32_t slope_norm, const float *h_sn, int32_t device,
                       pwfs_slopec_t **out) {
    if (out) *out = nullptr;
    if (!out || !h_valid || n_sub < 1 || n_sub > 16384 || (slope_norm != 0 && slope_norm != 1)) return PWFS_EINVAL;
    std::vector<int> vidx;
    for (int i = 0; i < n_sub * n_sub; ++i)
        if (h_valid[i]) vidx.push_back(i);
    if (vidx.empty()) return PWFS_EINVAL;
    pwfs_slopec *h = new (std::nothrow) pwfs_slopec();
    if (!h) return PWFS_ENOMEM;
    h->device = device;
    pwk::DeviceGuard dg(device);
    cudaError_t e = dg.err;
    if (e == cudaSuccess) e = cudaMalloc((void **)&h->d_vidx, vidx.size() * sizeof(int));
    if (e == cudaSuccess) e = cudaMemcpy(h->d_vidx, vidx.data(), vidx.size() * sizeof(int), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMalloc((void **)&h->d_sn, 2 * vidx.size() * sizeof(float));
    if (e != cudaSuccess) { int rc = cuda_rc(e); pwfs_slopec_destroy(h); return rc; }
    h->dev.n_sub = n_sub; h->dev.n_valid = (int)vidx.size(); h->dev.norm = slope_norm;
    h->dev.vidx = h->d_vidx; h->dev.sn = nullptr;
    int rc = pwfs_slopec_set_reference(h, h_sn);
    if (rc) { pwfs_slopec_destroy(h); return rc; }
    *out = h;
    return PWFS_OK;
}

int pwfs_slopec_set_reference(pwfs_slopec_t *h, const float *h_sn) {
    if (!h) return PWFS_EINVAL;
    if (!h_sn) { h->dev.sn = nullptr; return PWFS_OK; }
    pwk::DeviceGuard dg(h->device);
    if (dg.err != cudaSuccess) return PWFS_ECUDA;
    if (cudaMemcpy(h->d_sn, h_sn, (size_t)2 * h->dev.n_valid * sizeof(float), cudaMemcpyHostToDevice) != cudaSuccess)
        return PWFS_ECUDA;
    h->dev.sn = h->d_sn;
    return PWFS_OK;
}

int pwfs_slopec_n_slopes(const pwfs_slopec_t *h, int32_t *n_slopes) {
    if (!h || !n_slopes) return PWFS_EINVAL;
    *n_slopes = 2 * h->dev.n_valid;
    return PWFS_OK;
}

int pwfs_slopec_run(pwfs_slopec_t *h, const float *d_pixels, int32_t B, float *d_slopes, void *cuda_stream) {
    if (!h || B < 0) return PWFS_EINVAL;
    if (B == 0) return PWFS_OK;
    if (!d_pixels || !d_slopes) return PWFS_EINVAL;
    pwk::DeviceGuard dg(h->device);
    if (dg.err != cudaSuccess) return PWFS_ECUDA;
    for (int b0 = 0; b0 < B; b0 += 65535) {                      // grid.y limit
        const int Bc = B - b0 < 65535 ? B - b0 : 65535;
        slopec_kernel<<<dim3(kSlopecCluster, Bc), 256, 0, (cudaStream_t)cuda_stream>>>(
            h->dev, d_pixels + (size_t)b0 * 4 * h->dev.n_sub * h->dev.n_sub, d_slopes + (size_t)b0 * 2 * h->dev.n_valid);
    }
    return cudaGetLastError() == cudaSuccess ? PWFS_OK : PWFS_ECUDA;
}

void pwfs_slopec_destroy(pwfs_slopec_t *h) {
    if (!h) return;
    pwk::DeviceGuard dg(h->device);
    if (h->d_vidx) cudaFree(h->d_vidx);
    if (h->d_sn) cudaFree(h->d_sn);
    delete h;
}

// -------------------------------------------------- modal reconstructor ---
int pwfs_rec_create(int32_t n_modes, int32_t n_slopes, const float *h_recmat, int32_t device, pwfs_rec_t **out) {
    if (out) *out = nullptr;
    if (!out || !h_recmat || n_modes < 1 || n_slopes < 1) return PWFS_EINVAL;
    pwfs_rec *h = new (std::nothrow) pwfs_rec();
    if (!h) return PWFS_ENOMEM;
    h->device = device; h->n_modes = n_modes; h->n_slopes = n_slopes; h->ldk = (n_slopes + 3) / 4 * 4;
    const size_t bytes = (size_t)n_modes * h->ldk * sizeof(float);
    pwk::DeviceGuard dg(device);
    cudaError_t e = dg.err;
    if (e == cudaSuccess) e = cudaMalloc((void **)&h->d_R, bytes);
    if (e == cudaSuccess && h->ldk != n_slopes) e = cudaMemset(h->d_R, 0, bytes);
    if (e == cudaSuccess)
        e = cudaMemcpy2D(h->d_R, (size_t)h->ldk * sizeof(float), h_recmat, (size_t)n_slopes * sizeof(float),
                         (size_t)n_slopes * sizeof(float), (size_t)n_modes, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
        int sms = 0;
        if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device) == cudaSuccess && sms > 0) h->num_sms = sms;
    }
    if (e != cudaSuccess) { int rc = cuda_rc(e); pwfs_rec_destroy(h); return rc; }
    const char *env = std::getenv("PWFS_REC_TC");
    h->tc_off = env && env[0] == '0';
    *out = h;
    return PWFS_OK;
}

static int rec_uses_tc(pwfs_rec *h, int B) {
    return !h->tc_off && B >= kRecTcMinBatch && (long long)h->n_modes * h->n_slopes >= kRecTcMinElems;
}

static int rec_ensure_tc(pwfs_rec *h) {
    if (h->tc || h->tc_off) return PWFS_OK;
    const int rc = rec_tc_create(&h->tc, h->d_R, h->n_modes, h->n_slopes, h->ldk, h->device, h->num_sms);
    if (rc == PWFS_EUNSUPPORTED) { h->tc_off = true; return PWFS_OK; }
    return rc;
}

int pwfs_rec_reserve(pwfs_rec_t *h, int32_t B) {
    if (!h || B < 1) return PWFS_EINVAL;
    pwk::DeviceGuard dg(h->device);
    if (dg.err != cudaSuccess) return PWFS_ECUDA;
    if (!rec_uses_tc(h, B)) return PWFS_OK;                    // the FP32 kernels need no scratch
    if (int rc = rec_ensure_tc(h)) return rc;
    return h->tc ? rec_tc_reserve(h->tc, B, nullptr) : PWFS_OK;
}

int pwfs_rec_run(pwfs_rec_t *h, const float *d_slopes, int32_t B, float *d_modes, void *cuda_stream) {
    if (!h || B < 0) return PWFS_EINVAL;
    if (B == 0) return PWFS_OK;
    if (!d_slopes || !d_modes) return PWFS_EINVAL;
    pwk::DeviceGuard dg(h->device);
    if (dg.err != cudaSuccess) return PWFS_ECUDA;
    // batches: TF32x3 on the tensor cores (rec_tc.cu); single frames and small problems: FP32 FMA below
    if (rec_uses_tc(h, B)) {
        if (int rc = rec_ensure_tc(h)) return rc;
        if (h->tc) return rec_tc_run(h->tc, d_slopes, B, d_modes, (cudaStream_t)cuda_stream);
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (B == 1 && h->ldk <= 4 * kGemvThreads * 6 && h->n_modes >= 64) {   // closed loop: one frame, recmat streamed once
        const int nk = (h->ldk / 4 + kGemvThreads - 1) / kGemvThreads;
        const int grid = std::min(h->n_modes, h->num_sms);
        if (nk <= 2)      rec_gemv_kernel<2><<<grid, kGemvThreads, 0, st>>>(h->d_R, h->n_modes, h->ldk, d_slopes, h->n_slopes, d_modes);
        else if (nk <= 4) rec_gemv_kernel<4><<<grid, kGemvThreads, 0, st>>>(h->d_R, h->n_modes, h->ldk, d_slopes, h->n_slopes, d_modes);
        else              rec_gemv_kernel<6><<<grid, kGemvThreads, 0, st>>>(h->d_R, h->n_modes, h->ldk, d_slopes, h->n_slopes, d_modes);
        return cudaGetLastError() == cudaSuccess ? PWFS_OK : PWFS_ECUDA;
    }
    // frames per warp tile: the whole batch when it is small, else 16 or 8, whichever pads less
    int FB = 1;
    while (FB < B && FB < 16) FB *= 2;
    if (B > 16 && (B + 7) / 8 * 8 < (B + 15) / 16 * 16) FB = 8;
    const bool vec = (h->n_slopes % 4 == 0) && ((uintptr_t)d_slopes % 16 == 0);
    // four rows per warp once that still leaves >= 2 CTAs per SM
    const long long ctas4 = (long long)((h->n_modes + kRecWarps * 4 - 1) / (kRecWarps * 4)) * ((B + FB - 1) / FB);
    if (ctas4 >= 2LL * h->num_sms) launch_rec_fb<4>(FB, vec, st, h->d_R, h->n_modes, h->ldk, d_slopes, h->n_slopes, B, d_modes);
    else                           launch_rec_fb<1>(FB, vec, st, h->d_R, h->n_modes, h->ldk, d_slopes, h->n_slopes, B, d_modes);
    return cudaGetLastError() == cudaSuccess ? PWFS_OK : PWFS_ECUDA;
}

void pwfs_rec_destroy(pwfs_rec_t *h) {
    if (!h) return;
    pwk::DeviceGuard dg(h->device);
    if (h->d_R) cudaFree(h->d_R);
    rec_tc_destroy(h->tc);
    delete h;
}

}  // extern "C"
