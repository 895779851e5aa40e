// psf_api.cu -- f4, PSF camera: C ABI of include/pwfs_psf.h and its kernels.
//
// PSF = |DFT2(A exp(i c phi))|^2 on an M x M grid, M = 32 R1 >= 2N.  Same 1-D engine as the
// pyramid path (pwfs_kernels.cuh): one warp = one length-M transform, a zero-pad-pruned DFT of
// size R1 in registers, one exchange through padded shared memory, a DFT of size 32 -- but
// forward only, so the result stays in the "k1 + R1 k2" register order and is consumed there.
//
//   psf_row_kernel   N pupil rows per frame: phasor (phase rescaled to the imaging wavelength)
//                    -> DFT over x -> T[f][y / 8][u][y % 8] in natural frequency order (same blocked layout
//                    as the pyramid path's T).  The size-32 stage is done "transposed": a thread takes
//                    exchange row k1 of another warp's pupil row, so adjacent lanes hold adjacent rows y and
//                    the results go from registers straight to global memory (256 contiguous bytes per warp
//                    store, compile-time offsets) -- no staging copy.  A CTA keeps its rows for several
//                    frames, so the twiddle table is loaded once.
//   psf_col_kernel   one warp per NB columns u, looping over its share of the frames: DFT over
//                    y (only the N non-zero inputs are read, 64-byte runs), |.|^2 accumulated over the
//                    frames in registers; Strehl ratio from the (0,0) bin; one partial PSF per frame
//                    split, written column-major [u][v] so that a warp's stores are contiguous.
//   psf_fold_kernel  accumulator[v][u] += sum of the partial PSFs [u][v] (fixed order: deterministic),
//                    transposing 32 x 32 tiles through shared memory.
//   psf_read_kernel  long exposure = accumulator / (frames M^2 sum A^2).
// Work per frame: (N + M) transforms of length M; HBM: phase in, T out and back, nothing else.
#include "../../include/pwfs_psf.h"

#include <cuda_runtime.h>

#include "device_guard.cuh"

#include <algorithm>
#include <cmath>
#include <new>
#include <vector>

#include "pwfs_dft.cuh"

using namespace pwk;

namespace {

constexpr int kPitchP = 33;                         // float2 pitch of an exchange row (conflict-free 64-bit)
constexpr float kInv2PiHiP = 0.15915493667125702f;  // fl32(1/(2 pi))
constexpr float kInv2PiLoP = 6.4206382e-09f;        // 1/(2 pi) - hi

template <int R1_, int NB_, int WPB_>
struct PsfCfg {
    static constexpr int R1 = R1_, NB = NB_, WPB = WPB_;
    static constexpr int M = 32 * R1_;
    static constexpr int NZ = (R1_ + 1) / 2;         // M >= 2N: at most ceil(R1/2) non-zero inputs per lane
    static constexpr int ITEMS = NB_ * R1_;          // size-32 DFTs per warp batch
    static constexpr int ROUNDS = (ITEMS + 31) / 32; // lanes take them in rounds (R1 > 32: two)
    static constexpr bool PREFETCH = R1_ <= 32;      // column pass: next frame's inputs in registers while this one runs
    static_assert(ITEMS <= 32 || NB_ == 1, "more than one round only for a single transform per warp");
    // pad so that the row pass's copy-out (8 rows x 4 adjacent k2 per warp instruction) is conflict-free for NB = 1
    static constexpr int WARP_BUF = ITEMS * kPitchP + ((2 - (ITEMS * kPitchP) % 16) + 16) % 16;
    static constexpr int TAB = R1_ * kPitchP;
    static constexpr int RPC = NB_ * WPB_;           // rows per CTA, row pass

    static constexpr size_t smem = (size_t)(TAB + WPB_ * WARP_BUF) * sizeof(float2);
};

struct PsfDev {
    int N, M, NP;            // NP = N rounded up to 32
    float scale;             // phase_scale
    float inv_sumA_sq;       // 1 / (sum A)^2
    const float *amp;        // [N][N]
    const float2 *tw;        // [R1][32] exp(-2 pi i k1 n2 / M)
};

template <class C>
__device__ __forceinline__ void load_tw(float2 *s_tw, const PsfDev &t) {
    for (int i = threadIdx.x; i < C::R1 * 32; i += blockDim.x) s_tw[(i >> 5) * kPitchP + (i & 31)] = __ldg(t.tw + i);
}

constexpr int kRowFrames = 4;    // frames a row-pass CTA works through (amortises the twiddle-table load)

// grid (ceil(NP / RPC), ceil(F / kRowFrames)); block 32 * WPB.
template <class C>
__global__ void __launch_bounds__(32 * C::WPB)
psf_row_kernel(PsfDev t, const float *__restrict__ phase, float2 *__restrict__ T, int F) {
    static_assert(C::RPC % 8 == 0, "row pass: rows per CTA must be whole 8-row blocks of T");
    extern __shared__ float2 smem[];
    float2 *s_tw = smem, *s_buf = smem + C::TAB;
    const int lane = threadIdx.x & 31, wl = threadIdx.x >> 5;
    const int N = t.N, y0 = blockIdx.x * C::RPC;
    float2 *buf = s_buf + wl * C::WARP_BUF;
    load_tw<C>(s_tw, t);
    float am[C::NB][C::NZ];
#pragma unroll
    for (int b = 0; b < C::NB; ++b)
#pragma unroll
        for (int n1 = 0; n1 < C::NZ; ++n1) {
            const int y = y0 + wl * C::NB + b, x = 32 * n1 + lane;
            am[b][n1] = (y < N && x < N) ? __ldg(t.amp + (size_t)y * N + x) : 0.f;
        }
    const int f_end = min(F, (int)(blockIdx.y + 1) * kRowFrames);
    // the next frame's phase is fetched while this frame is transformed
    float ph[C::NB][C::NZ];
    auto fetch = [&](int f) {
#pragma unroll
        for (int b = 0; b < C::NB; ++b)
#pragma unroll
            for (int n1 = 0; n1 < C::NZ; ++n1) {
                const int y = y0 + wl * C::NB + b, x = 32 * n1 + lane;
                ph[b][n1] = (y < N && x < N) ? __ldg(phase + ((size_t)f * N + y) * N + x) : 0.f;
            }
    };
    if ((int)blockIdx.y * kRowFrames < f_end) fetch(blockIdx.y * kRowFrames);
    for (int f = blockIdx.y * kRowFrames; f < f_end; ++f) {
#pragma unroll
        for (int b = 0; b < C::NB; ++b) {
            float2 v[C::R1];
#pragma unroll
            for (int n1 = 0; n1 < C::NZ; ++n1) {
                const float p = ph[b][n1] * t.scale;
                // phase in turns, reduced with a two-term 1/(2 pi) (exact integer part, FMA keeps the low bits)
                const float q = rintf(p * kInv2PiHiP);
                float tr = fmaf(p, kInv2PiHiP, -q);
                tr = fmaf(p, kInv2PiLoP, tr);
                float sn, cs;
                __sincosf(tr * 6.283185307179586f, &sn, &cs);
                v[n1] = make_float2(am[b][n1] * cs, am[b][n1] * sn);
            }
            if (b == C::NB - 1 && f + 1 < f_end) fetch(f + 1);
            DftP<C::R1, -1, C::NZ>::run(v);
#pragma unroll
            for (int k1 = 0; k1 < C::R1; ++k1) buf[(b * C::R1 + k1) * kPitchP + lane] = v[k1];
        }
        __syncthreads();     // also: the twiddle table is complete (first pass)
        // Size-32 stage, done "transposed" like the last stage of the pyramid's row pass: thread item
        // i = r_lo + 8 (k1 + R1 r_hi) takes exchange row k1 of CTA row r = 8 r_hi + r_lo (another warp's buffer), so that
        // adjacent lanes hold adjacent rows y of one frequency.  X[u = k1 + R1 k2] goes from registers straight to
        // T[f][(y0 + r) / 8][u][r_lo]: 8 lanes x 4 adjacent k1 write 256 contiguous bytes, every store of a thread is a
        // compile-time offset (k2 * R1 * 8 float2) from one base.  No staging pass, no third barrier.
        float2 *Tf = T + (size_t)f * C::M * t.NP + (size_t)(y0 / 8) * (C::M * 8);
#pragma unroll
        for (int it = 0; it < C::ROUNDS; ++it) {
            const int i = threadIdx.x + it * 32 * C::WPB;
            const int q = i >> 3, r_hi = q / C::R1, k1 = q - r_hi * C::R1, r = 8 * r_hi + (i & 7);
            if (i < C::RPC * C::R1 && y0 + r < t.NP) {
                const float2 *row = s_buf + (r / C::NB) * C::WARP_BUF + ((r % C::NB) * C::R1 + k1) * kPitchP;
                const float2 *twr = s_tw + k1 * kPitchP;
                float2 u[32];
#pragma unroll
                for (int n2 = 0; n2 < 32; ++n2) u[n2] = cmul(row[n2], twr[n2]);
                Dft<32, -1>::run(u);
                float2 *dst = Tf + ((size_t)r_hi * C::M + k1) * 8 + (i & 7);
#pragma unroll
                for (int k2 = 0; k2 < 32; ++k2) dst[k2 * (C::R1 * 8)] = u[k2];
            }
        }
        __syncthreads();     // the next frame overwrites the buffers
    }
}

// grid (ceil(M / (NB * WPB)), fsplit); block 32 * WPB.  partial: [fsplit][M][M] (fftshifted).
template <class C>
__global__ void __launch_bounds__(32 * C::WPB)
psf_col_kernel(PsfDev t, const float2 *__restrict__ T, int F, int fsplit, float *__restrict__ partial,
               float *__restrict__ sr) {
    extern __shared__ float2 smem[];
    float2 *s_tw = smem, *s_buf = smem + C::TAB;
    const int lane = threadIdx.x & 31, wl = threadIdx.x >> 5;
    const int NP = t.NP, fs = blockIdx.y;
    const int u0 = (blockIdx.x * C::WPB + wl) * C::NB;
    float2 *buf = s_buf + wl * C::WARP_BUF;
    load_tw<C>(s_tw, t);
    __syncthreads();
    if (u0 >= C::M) return;
    const int f_lo = (int)(((long long)fs * F) / fsplit), f_hi = (int)(((long long)(fs + 1) * F) / fsplit);
    float acc[C::ROUNDS][32];
#pragma unroll
    for (int rd = 0; rd < C::ROUNDS; ++rd)
#pragma unroll
        for (int k2 = 0; k2 < 32; ++k2) acc[rd][k2] = 0.f;
    float2 pre[C::NB][C::NZ];
    // T[f][y / 8][u][y % 8]: lane reads y = 32 n1 + lane, i.e. block 4 n1 + lane / 8, row lane % 8 of column u = u0 + b
    auto fetch = [&](int f) {
        const float2 *src = T + (size_t)f * C::M * NP + (size_t)(lane >> 3) * (C::M * 8) + (size_t)u0 * 8 + (lane & 7);
#pragma unroll
        for (int b = 0; b < C::NB; ++b)
#pragma unroll
            for (int n1 = 0; n1 < C::NZ; ++n1)
                pre[b][n1] = (32 * n1 < NP && u0 + b < C::M) ? __ldg(src + b * 8 + (size_t)n1 * (32 * C::M)) : make_float2(0.f, 0.f);
    };
    if (C::PREFETCH && f_lo < f_hi) fetch(f_lo);
    for (int f = f_lo; f < f_hi; ++f) {
        if (!C::PREFETCH) fetch(f);
#pragma unroll
        for (int b = 0; b < C::NB; ++b) {
            float2 v[C::R1];
#pragma unroll
            for (int n1 = 0; n1 < C::NZ; ++n1) v[n1] = pre[b][n1];
            if (C::PREFETCH && b == C::NB - 1 && f + 1 < f_hi) fetch(f + 1);
            DftP<C::R1, -1, C::NZ>::run(v);
#pragma unroll
            for (int k1 = 0; k1 < C::R1; ++k1) buf[(b * C::R1 + k1) * kPitchP + lane] = v[k1];
        }
        __syncwarp();
#pragma unroll
        for (int rd = 0; rd < C::ROUNDS; ++rd) {
            const int w = rd * 32 + lane;
            if (w < C::ITEMS) {
                const int my_b = w / C::R1, my_k1 = w % C::R1;
                const float2 *row = buf + w * kPitchP;
                const float2 *twr = s_tw + my_k1 * kPitchP;
                float2 u[32];
#pragma unroll
                for (int n2 = 0; n2 < 32; ++n2) u[n2] = cmul(row[n2], twr[n2]);
                Dft<32, -1>::run(u);
#pragma unroll
                for (int k2 = 0; k2 < 32; ++k2) acc[rd][k2] = fmaf(u[k2].x, u[k2].x, fmaf(u[k2].y, u[k2].y, acc[rd][k2]));
                if (sr && my_k1 == 0 && u0 + my_b == 0)          // F4c: the (0, 0) bin (column c = 0 is u = 0)
                    sr[f] = fmaf(u[0].x, u[0].x, u[0].y * u[0].y) * t.inv_sumA_sq;
            }
        }
        __syncwarp();
    }
#pragma unroll
    for (int rd = 0; rd < C::ROUNDS; ++rd) {
        const int w = rd * 32 + lane;
        const int my_b = w / C::R1, my_k1 = w % C::R1;
        if (w < C::ITEMS && u0 + my_b < C::M) {
            const int uu = u0 + my_b;                                        // column c of T holds frequency u = c
            const int uo = (uu + C::M / 2) % C::M;
            float *dst = partial + ((size_t)fs * C::M + uo) * C::M;          // [fs][u][v]: the lanes' v are adjacent
#pragma unroll
            for (int k2 = 0; k2 < 32; ++k2) {
                const int vo = (my_k1 + C::R1 * k2 + C::M / 2) % C::M;
                dst[vo] = acc[rd][k2];
            }
        }
    }
}

// accum[v][u] += sum_k partial[k][u][v]; grid (M / 32, M / 32), block (32, 8)
__global__ void psf_fold_kernel(float *__restrict__ accum, const float *__restrict__ partial, int fsplit, int M) {
    __shared__ float tile[32][33];
    const size_t MM = (size_t)M * M;
    const int u0 = blockIdx.y * 32, v0 = blockIdx.x * 32;
    // all loads of a thread (4 rows x fsplit partials) are issued before the first add: this kernel is pure latency
    // (25 MB in 1024 small CTAs); the sum over k keeps its fixed order
    float s[4] = {0.f, 0.f, 0.f, 0.f};
    for (int k0 = 0; k0 < fsplit; k0 += 4) {
        float v[4][4];
#pragma unroll
        for (int jj = 0; jj < 4; ++jj)
#pragma unroll
            for (int kk = 0; kk < 4; ++kk)
                v[jj][kk] = (k0 + kk < fsplit) ? __ldg(partial + (size_t)(k0 + kk) * MM + (size_t)(u0 + threadIdx.y + 8 * jj) * M + v0 + threadIdx.x) : 0.f;
#pragma unroll
        for (int jj = 0; jj < 4; ++jj)
#pragma unroll
            for (int kk = 0; kk < 4; ++kk) s[jj] += v[jj][kk];
    }
#pragma unroll
    for (int jj = 0; jj < 4; ++jj) tile[threadIdx.y + 8 * jj][threadIdx.x] = s[jj];   // tile[u][v], coalesced along v
    __syncthreads();
    for (int j = threadIdx.y; j < 32; j += 8) {                       // accum[v][u], coalesced along u
        float *dst = accum + (size_t)(v0 + j) * M + u0 + threadIdx.x;
        *dst += tile[threadIdx.x][j];
    }
}

__global__ void psf_read_kernel(const float *__restrict__ accum, float *__restrict__ out, float scale, size_t MM) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < MM) out[i] = accum[i] * scale;
}

struct PsfLauncher {
    int NB, WPB, RPC;
    size_t smem;
    void (*row)(dim3, cudaStream_t, const PsfDev &, const float *, float2 *, int);
    void (*col)(dim3, cudaStream_t, const PsfDev &, const float2 *, int, int, float *, float *);
    cudaError_t (*prepare)();
    int (*col_ctas_per_sm)();       // occupancy of the column-pass kernel
};

template <class C>
void row_t(dim3 g, cudaStream_t st, const PsfDev &t, const float *ph, float2 *T, int F) {
    psf_row_kernel<C><<<g, 32 * C::WPB, C::smem, st>>>(t, ph, T, F);
}
template <class C>
void col_t(dim3 g, cudaStream_t st, const PsfDev &t, const float2 *T, int F, int fsplit, float *part, float *sr) {
    psf_col_kernel<C><<<g, 32 * C::WPB, C::smem, st>>>(t, T, F, fsplit, part, sr);
}
template <class C, class CC>
cudaError_t prepare_t() {
    cudaError_t e = cudaFuncSetAttribute(psf_row_kernel<C>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(psf_col_kernel<CC>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)CC::smem);
    return e;
}
template <class C>
int col_occ_t() {
    int n = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, psf_col_kernel<C>, 32 * C::WPB, C::smem) != cudaSuccess || n < 1) n = 1;
    return n;
}
// C: row pass; CC: column pass (same R1 and NB; 4-warp CTAs for the large grids: two CTAs per SM fill the machine better
// than one of 8 warps when a launch has only M / 8 of them)
template <class C, class CC = C>
PsfLauncher make() { return PsfLauncher{CC::NB, CC::WPB, C::RPC, C::smem, row_t<C>, col_t<CC>, prepare_t<C, CC>, col_occ_t<CC>}; }

bool find_psf_launcher(int M, PsfLauncher *out) {
    if (M % 32) return false;
    switch (M / 32) {
        case 4:  *out = make<PsfCfg<4, 8, 4>>(); return true;
        case 5:  *out = make<PsfCfg<5, 6, 4>>(); return true;
        case 6:  *out = make<PsfCfg<6, 5, 8>>(); return true;
        case 8:  *out = make<PsfCfg<8, 4, 4>>(); return true;
        case 9:  *out = make<PsfCfg<9, 3, 8>>(); return true;
        case 10: *out = make<PsfCfg<10, 3, 8>>(); return true;
        case 12: *out = make<PsfCfg<12, 2, 4>>(); return true;
        case 15: *out = make<PsfCfg<15, 2, 4>>(); return true;
        case 16: *out = make<PsfCfg<16, 2, 4>>(); return true;
        case 18: *out = make<PsfCfg<18, 1, 8>, PsfCfg<18, 1, 4>>(); return true;
        case 20: *out = make<PsfCfg<20, 1, 8>, PsfCfg<20, 1, 4>>(); return true;
        case 24: *out = make<PsfCfg<24, 1, 8>, PsfCfg<24, 1, 4>>(); return true;
        case 25: *out = make<PsfCfg<25, 1, 8>, PsfCfg<25, 1, 4>>(); return true;
        case 27: *out = make<PsfCfg<27, 1, 8>, PsfCfg<27, 1, 4>>(); return true;
        case 30: *out = make<PsfCfg<30, 1, 8>, PsfCfg<30, 1, 4>>(); return true;
        case 32: *out = make<PsfCfg<32, 1, 8>, PsfCfg<32, 1, 4>>(); return true;
        case 36: *out = make<PsfCfg<36, 1, 8>, PsfCfg<36, 1, 4>>(); return true;
        case 40: *out = make<PsfCfg<40, 1, 8>, PsfCfg<40, 1, 4>>(); return true;
        case 45: *out = make<PsfCfg<45, 1, 8>, PsfCfg<45, 1, 4>>(); return true;
        case 48: *out = make<PsfCfg<48, 1, 8>, PsfCfg<48, 1, 4>>(); return true;
        case 50: *out = make<PsfCfg<50, 1, 8>, PsfCfg<50, 1, 4>>(); return true;
        case 54: *out = make<PsfCfg<54, 1, 8>, PsfCfg<54, 1, 4>>(); return true;
        case 60: *out = make<PsfCfg<60, 1, 8>, PsfCfg<60, 1, 4>>(); return true;
        case 64: *out = make<PsfCfg<64, 1, 8>, PsfCfg<64, 1, 4>>(); return true;
        default: return false;
    }
}

int cuda_rc(cudaError_t e) { return e == cudaErrorMemoryAllocation ? PWFS_ENOMEM : PWFS_ECUDA; }

}  // namespace

struct pwfs_psf {
    int device = 0;
    PsfDev dev{};
    PsfLauncher L{};
    double sumA2 = 0.0;
    float *d_amp = nullptr;
    float2 *d_tw = nullptr;
    float *d_acc = nullptr;          // [M][M] sum over frames of |X|^2, fftshifted
    float2 *T = nullptr; size_t T_frames = 0;
    float *partial = nullptr; int partial_split = 0;
    long long count = 0;
    int num_sms = 148;
    int col_resident = 148;          // column-pass CTAs the device holds at once
    size_t scratch_budget = (size_t)2 << 30;
};

extern "C" {

int pwfs_psf_create(const pwfs_psf_params *p, pwfs_psf_t **out) {
    if (out) *out = nullptr;
    if (!p || !out || !p->pupil_amp) return PWFS_EINVAL;
    const int N = p->n_pupil, M = p->m_grid;
    if (N < 2 || M < 2 * N || !std::isfinite(p->phase_scale)) return PWFS_EINVAL;
    PsfLauncher L;
    if (!find_psf_launcher(M, &L)) return PWFS_EUNSUPPORTED;
    double sumA = 0.0, sumA2 = 0.0;
    for (size_t i = 0; i < (size_t)N * N; ++i) {
        const double a = p->pupil_amp[i];
        if (!(a >= 0.0) || !std::isfinite(a)) return PWFS_EINVAL;
        sumA += a; sumA2 += a * a;
    }
    if (!(sumA > 0.0)) return PWFS_EINVAL;
    const int R1 = M / 32;
    std::vector<float2> tw((size_t)R1 * 32);
    for (int k1 = 0; k1 < R1; ++k1)
        for (int n2 = 0; n2 < 32; ++n2) {
            const double a = -6.283185307179586476925286766559 * (double)((long long)k1 * n2 % M) / (double)M;
            tw[(size_t)k1 * 32 + n2] = make_float2((float)std::cos(a), (float)std::sin(a));
        }
    pwfs_psf *h = new (std::nothrow) pwfs_psf();
    if (!h) return PWFS_ENOMEM;
    h->device = p->device; h->L = L; h->sumA2 = sumA2;
    const size_t MM = (size_t)M * M;
    pwk::DeviceGuard dg(p->device);
    cudaError_t e = dg.err;
    if (e == cudaSuccess) e = cudaMalloc((void **)&h->d_amp, (size_t)N * N * sizeof(float));
    if (e == cudaSuccess) e = cudaMemcpy(h->d_amp, p->pupil_amp, (size_t)N * N * sizeof(float), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMalloc((void **)&h->d_tw, tw.size() * sizeof(float2));
    if (e == cudaSuccess) e = cudaMemcpy(h->d_tw, tw.data(), tw.size() * sizeof(float2), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMalloc((void **)&h->d_acc, MM * sizeof(float));
    if (e == cudaSuccess) e = cudaMemset(h->d_acc, 0, MM * sizeof(float));
    if (e == cudaSuccess) e = L.prepare();
    if (e == cudaSuccess) {
        int sms = 0;
        if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, p->device) == cudaSuccess && sms > 0) h->num_sms = sms;
        h->col_resident = h->num_sms * L.col_ctas_per_sm();
    }
    if (e != cudaSuccess) { int rc = cuda_rc(e); pwfs_psf_destroy(h); return rc; }
    PsfDev &d = h->dev;
    d.N = N; d.M = M; d.NP = (N + 31) / 32 * 32;
    d.scale = p->phase_scale;
    d.inv_sumA_sq = (float)(1.0 / (sumA * sumA));
    d.amp = h->d_amp; d.tw = h->d_tw;
    *out = h;
    return PWFS_OK;
}

int pwfs_psf_accumulate(pwfs_psf_t *h, const float *d_phase, int32_t B, float *d_sr, void *cuda_stream) {
    if (!h || B < 0) return PWFS_EINVAL;
    if (B == 0) return PWFS_OK;
    if (!d_phase) return PWFS_EINVAL;
    pwk::DeviceGuard dg(h->device);
    if (dg.err != cudaSuccess) return PWFS_ECUDA;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const PsfDev &d = h->dev;
    const PsfLauncher &L = h->L;
    const size_t MM = (size_t)d.M * d.M, per_frame = (size_t)d.M * d.NP * sizeof(float2);
    const int F = (int)std::min<size_t>((size_t)B, std::max<size_t>(1, h->scratch_budget / per_frame));
    // column pass: ~32 warps per SM in flight; the frame loop is split only as far as that needs
    const int col_ctas = (d.M + L.NB * L.WPB - 1) / (L.NB * L.WPB);
    // split of the frame loop: minimise (waves of resident CTAs) x (frames per CTA + 2 for its prologue and the
    // write of its partial PSF), at most 32 partials
    int fsplit = 1;
    {
        double best = 1e300;
        for (int c = 1; c <= std::min(F, 32); ++c) {
            const long long ctas = (long long)col_ctas * c;
            const double waves = (double)((ctas + h->col_resident - 1) / h->col_resident);
            const double cost = waves * ((F + c - 1) / c + 2.0);
            if (cost < best * (1.0 - 1e-9)) { best = cost; fsplit = c; }
        }
    }
    if ((size_t)F > h->T_frames) {
        if (h->T) cudaFree(h->T);
        h->T = nullptr; h->T_frames = 0;
        cudaError_t e = cudaMalloc((void **)&h->T, (size_t)F * per_frame);
        if (e != cudaSuccess) return cuda_rc(e);
        h->T_frames = (size_t)F;
    }
    if (fsplit > h->partial_split) {
        if (h->partial) cudaFree(h->partial);
        h->partial = nullptr; h->partial_split = 0;
        cudaError_t e = cudaMalloc((void **)&h->partial, (size_t)fsplit * MM * sizeof(float));
        if (e != cudaSuccess) return cuda_rc(e);
        h->partial_split = fsplit;
    }
    for (int f0 = 0; f0 < B; f0 += F) {
        const int Fc = std::min(F, B - f0);
        const int fsp = std::min(fsplit, Fc);
        L.row(dim3((d.NP + L.RPC - 1) / L.RPC, (Fc + kRowFrames - 1) / kRowFrames), st, d, d_phase + (size_t)f0 * d.N * d.N, h->T, Fc);
        L.col(dim3(col_ctas, fsp), st, d, h->T, Fc, fsp, h->partial, d_sr ? d_sr + f0 : nullptr);
        psf_fold_kernel<<<dim3(d.M / 32, d.M / 32), dim3(32, 8), 0, st>>>(h->d_acc, h->partial, fsp, d.M);
    }
    if (cudaGetLastError() != cudaSuccess) return PWFS_ECUDA;
    h->count += B;
    return PWFS_OK;
}

int pwfs_psf_read(pwfs_psf_t *h, float *d_psf, int64_t *frames_out, void *cuda_stream) {
    if (!h || !d_psf) return PWFS_EINVAL;
    pwk::DeviceGuard dg(h->device);
    if (dg.err != cudaSuccess) return PWFS_ECUDA;
    const size_t MM = (size_t)h->dev.M * h->dev.M;
    const double scale = h->count > 0 ? 1.0 / ((double)h->count * (double)MM * h->sumA2) : 0.0;
    psf_read_kernel<<<(unsigned)((MM + 255) / 256), 256, 0, (cudaStream_t)cuda_stream>>>(h->d_acc, d_psf, (float)scale, MM);
    if (frames_out) *frames_out = h->count;
    return cudaGetLastError() == cudaSuccess ? PWFS_OK : PWFS_ECUDA;
}

int pwfs_psf_reset(pwfs_psf_t *h, void *cuda_stream) {
    if (!h) return PWFS_EINVAL;
    pwk::DeviceGuard dg(h->device);
    if (dg.err != cudaSuccess) return PWFS_ECUDA;
    const size_t MM = (size_t)h->dev.M * h->dev.M;
    if (cudaMemsetAsync(h->d_acc, 0, MM * sizeof(float), (cudaStream_t)cuda_stream) != cudaSuccess) return PWFS_ECUDA;
    h->count = 0;
    return PWFS_OK;
}

void pwfs_psf_destroy(pwfs_psf_t *h) {
    if (!h) return;
    pwk::DeviceGuard dg(h->device);
    if (h->d_amp) cudaFree(h->d_amp);
    if (h->d_tw) cudaFree(h->d_tw);
    if (h->d_acc) cudaFree(h->d_acc);
    if (h->T) cudaFree(h->T);
    if (h->partial) cudaFree(h->partial);
    delete h;
}

}  // extern "C"
