// pwfs_small.cuh -- the whole hot path in ONE kernel for the smallest grid, M = 128.
//
// For a 64-px pupil on a 128 grid the intermediate T of one modulation point is 128 columns x 64 rows x 8 B = 64 KB: it
// fits in shared memory next to the exchange buffers, so a CTA can run the row pass of one (frame, modulation point),
// keep T on chip, run its column pass, rebin, and leave a partial detector frame.  The CTA that finishes a frame last
// adds the partial frames of the K points in a fixed order (deterministic), computes the normalisation and the slopes.
// One launch instead of four, no T / colbin round trip through L2: a closed loop's small batches (cfg 1 as specified:
// 10 frames of 12 modulation points) are launch- and latency-bound otherwise, so the unit of work is the single
// modulation point (K CTAs per frame; the row pass is NOT shared between points of equal x-tilt here: with a few
// frames the machine has SMs to spare and the critical path is what counts).
//
// grid (K, F); block 256 (8 warps); 1 CTA per SM.  Same register butterflies, size-32 stage and mask handling as the
// two-kernel path (pwfs_kernels.cuh); same arithmetic, different summation order over k (per x-tilt first).
#pragma once
#include "pwfs_kernels.cuh"

namespace pwk {

struct SmallCfg : PassCfg<4, 8, 8, 8> {
    static constexpr int WARPS = 8;
    static constexpr int PY = 65;                        // float2 pitch of a T column in shared memory (odd: conflict-free)
    static constexpr int MAXN = 64, MAXCOLS = 128, MAXD = 64, MAXCMAX = 8;
    // tables + exchange buffers + T + y-rebinned columns
    static constexpr size_t smem_q = (size_t)(1 * TAB + WARPS * WARP_BUF + MAXCOLS * PY) * sizeof(float2) + (size_t)MAXCOLS * (MAXD + 1) * sizeof(float);
    static constexpr size_t smem_t = smem_q + (size_t)TAB * sizeof(float2);
};

// part: [F][K][D][D] partial frames; counter: [F], zero between launches.
template <bool QM>
__global__ void __launch_bounds__(256, 1)
small_kernel(DevTables t, const float *__restrict__ phase, float *__restrict__ part,
             unsigned *__restrict__ counter, float *__restrict__ frames, float *__restrict__ slopes, float scale) {
    using C = SmallCfg;
    extern __shared__ float2 smem[];
    float2 *s_tw = smem;
    const float2 *s_am = smem + C::TAB;                   // unused when QM
    float2 *s_buf = smem + (QM ? 1 : 2) * C::TAB;
    float2 *s_T = s_buf + C::WARPS * C::WARP_BUF;         // [ncols][PY]
    float *s_cb = reinterpret_cast<float *>(s_T + C::MAXCOLS * C::PY);   // [ncols][D + 1]
    __shared__ float s_red[8];
    __shared__ float s_nbar;
    __shared__ int s_last;
    // rebin tables in shared memory: the rebin loops chase start -> count -> weight, three dependent loads per
    // detector bin that would each wait for L2 in a kernel every CTA runs through exactly once
    __shared__ int s_rb_start[C::MAXD], s_rb_cnt[C::MAXD], s_xc_of_x[C::M];
    __shared__ float s_rb_w[C::MAXD * C::MAXCMAX];
    const int lane = threadIdx.x & 31, wl = threadIdx.x >> 5;
    const int N = t.N, NP = t.NP, D = t.D, ncols = t.ncols;
    const int k = blockIdx.x, f = blockIdx.y;
    const int j = __ldg(t.jx + k);
    float2 *buf = s_buf + wl * C::WARP_BUF;
    // this point's y-tilt: fetched now, used after the row pass
    float2 tyv[C::NZ];
#pragma unroll
    for (int n1 = 0; n1 < C::NZ; ++n1) tyv[n1] = (32 * n1 < NP) ? __ldg(t.tyt + (size_t)k * NP + 32 * n1 + lane) : make_float2(0.f, 0.f);

    load_tables<QM, false>(s_tw, smem + C::TAB, t, C::R1);
    const int cmax = t.cmax;
    for (int i = threadIdx.x; i < D; i += blockDim.x) { s_rb_start[i] = __ldg(t.rb_start + i); s_rb_cnt[i] = __ldg(t.rb_cnt + i); }
    for (int i = threadIdx.x; i < D * cmax; i += blockDim.x) s_rb_w[i] = __ldg(t.rb_w + i);
    for (int i = threadIdx.x; i < C::M; i += blockDim.x) s_xc_of_x[i] = __ldg(t.xc_of_x + i);
    int xc_of[C::R1];                                      // compact column of this lane's x = 32 n1 + lane, -1 outside the windows
#pragma unroll
    for (int n1 = 0; n1 < C::R1; ++n1) xc_of[n1] = __ldg(t.xc_of_x + 32 * n1 + lane);
    __syncthreads();

    // ---- row pass of x-tilt j: rows y = rg * 64 + wl * 8 + b -> T[xc][y] in shared memory
    for (int rg = 0; rg * (C::WARPS * C::NB) < NP; ++rg) {
#pragma unroll
        for (int b = 0; b < C::NB; ++b) {
            const int y = (rg * C::WARPS + wl) * C::NB + b;
            float2 v[C::R1];
#pragma unroll
            for (int n1 = 0; n1 < C::NZ; ++n1) {
                const int x = 32 * n1 + lane;
                const bool ok = (y < N) && (x < N);
                const float ph = ok ? __ldg(phase + ((size_t)f * N + y) * N + x) : 0.f;
                const float am = ok ? __ldg(t.amp + (size_t)y * N + x) : 0.f;
                const float q = rintf(ph * kInv2PiHi);
                float tr = fmaf(ph, kInv2PiHi, -q);
                tr = fmaf(ph, kInv2PiLo, tr);
                float sn, cs;
                __sincosf(tr * 6.283185307179586f, &sn, &cs);
                v[n1] = cmul(make_float2(am * cs, am * sn), __ldg(t.txc + (size_t)j * t.NXP + x));
            }
            DftP<C::R1, -1, C::NZ>::run(v);
#pragma unroll
            for (int k1 = 0; k1 < C::R1; ++k1) buf[C::row_off(b * C::R1 + k1) + lane] = v[k1];
        }
        __syncwarp();
        stage32<C, QM>(buf, s_tw, s_am, lane);
        __syncwarp();
#pragma unroll
        for (int b = 0; b < C::NB; ++b) {
            const int y = (rg * C::WARPS + wl) * C::NB + b;
            float2 v[C::R1];
#pragma unroll
            for (int k1 = 0; k1 < C::R1; ++k1) v[k1] = buf[C::row_off(b * C::R1 + k1) + lane];
            apply_ipow_k1<C::R1, QM>(v);
            Dft<C::R1, +1>::run(v);
            if (y < NP) {
#pragma unroll
                for (int n1 = 0; n1 < C::R1; ++n1)
                    if (xc_of[n1] >= 0) s_T[xc_of[n1] * C::PY + y] = v[n1];
            }
        }
        __syncwarp();
    }
    __syncthreads();

    // ---- column pass of this modulation point (|E|^2 in registers) and y-rebin of every column into s_cb[xc][jy];
    // one loop over the groups of 64 columns (not unrolled: one copy of the size-32 stage in the instruction stream)
    constexpr int CPASS = C::MAXCOLS / (C::WARPS * C::NB);   // 2 groups of 64 columns
    float *colI = reinterpret_cast<float *>(buf);          // NB * M floats <= the warp's buffer
#pragma unroll 1
    for (int cp = 0; cp < CPASS; ++cp) {
        const int xc0 = (cp * C::WARPS + wl) * C::NB;
        if (xc0 >= ncols) continue;                        // warp-uniform
        float acc[C::NB][C::R1];
#pragma unroll
        for (int b = 0; b < C::NB; ++b) {
            float2 v[C::R1];
#pragma unroll
            for (int n1 = 0; n1 < C::NZ; ++n1)
                v[n1] = (32 * n1 + lane < NP && xc0 + b < ncols) ? cmul(s_T[(xc0 + b) * C::PY + 32 * n1 + lane], tyv[n1])
                                                                  : make_float2(0.f, 0.f);
            DftP<C::R1, -1, C::NZ>::run(v);
#pragma unroll
            for (int k1 = 0; k1 < C::R1; ++k1) buf[C::row_off(b * C::R1 + k1) + lane] = v[k1];
        }
        __syncwarp();
        stage32<C, QM>(buf, s_tw, s_am, lane);
        __syncwarp();
#pragma unroll
        for (int b = 0; b < C::NB; ++b) {
            float2 v[C::R1];
#pragma unroll
            for (int k1 = 0; k1 < C::R1; ++k1) v[k1] = buf[C::row_off(b * C::R1 + k1) + lane];
            apply_ipow_k1<C::R1, QM>(v);
            Dft<C::R1, +1>::run(v);
#pragma unroll
            for (int n1 = 0; n1 < C::R1; ++n1) acc[b][n1] = fmaf(v[n1].x, v[n1].x, v[n1].y * v[n1].y);
        }
        __syncwarp();
#pragma unroll
        for (int b = 0; b < C::NB; ++b)
#pragma unroll
            for (int n1 = 0; n1 < C::R1; ++n1) colI[b * C::M + 32 * n1 + lane] = acc[b][n1];
        __syncwarp();
        for (int b = 0; b < C::NB && xc0 + b < ncols; ++b)
            for (int jj = lane; jj < D; jj += 32) {
                int y = s_rb_start[jj];
                const int cnt = s_rb_cnt[jj];
                float s = 0.f;
                for (int c = 0; c < cnt; ++c) {
                    s = fmaf(s_rb_w[jj * cmax + c], colI[b * C::M + y], s);
                    if (++y == C::M) y = 0;
                }
                s_cb[(xc0 + b) * (D + 1) + jj] = s;
            }
        __syncwarp();
    }
    __syncthreads();

    // ---- x-rebin -> this x-tilt's partial frame
    float *my_part = part + ((size_t)f * gridDim.x + k) * D * D;
    for (int i = threadIdx.x; i < D * D; i += blockDim.x) {
        const int jy = i % D, jx = i / D;                  // jy fastest: conflict-free reads of s_cb
        int x = s_rb_start[jx];
        const int cnt = s_rb_cnt[jx];
        float s = 0.f;
        for (int c = 0; c < cnt; ++c) {
            s = fmaf(s_rb_w[jx * cmax + c], s_cb[s_xc_of_x[x] * (D + 1) + jy], s);
            if (++x == C::M) x = 0;
        }
        my_part[jy * D + jx] = s * scale;
    }

    // ---- the CTA that completes the frame adds the partial frames (fixed order), then normalisation and slopes
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = (atomicAdd(counter + f, 1u) == gridDim.x - 1) ? 1 : 0;
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    const int ns = t.n_sub, nv = t.n_valid;
    float *fr = frames + (size_t)f * D * D;
    float vsum = 0.f;
    for (int i = threadIdx.x; i < D * D; i += blockDim.x) {
        float s = 0.f;
        for (int g = 0; g < (int)gridDim.x; ++g) s += __ldcg(part + ((size_t)f * gridDim.x + g) * D * D + i);
        fr[i] = s;
        const int jy = i / D, jx = i - jy * D;
        const int iy = jy >= ns ? jy - ns : jy, ix = jx >= ns ? jx - ns : jx;
        if (__ldg(t.vmask + iy * ns + ix)) vsum += s;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) vsum += __shfl_xor_sync(0xffffffffu, vsum, o);
    if (lane == 0) s_red[wl] = vsum;
    __syncthreads();                                       // also: fr[] written by this CTA is visible to it
    if (threadIdx.x == 0) {
        float v = 0.f;
        for (int w = 0; w < C::WARPS; ++w) v += s_red[w];
        s_nbar = v / (float)nv;
        counter[f] = 0u;                                   // ready for the next launch
    }
    __syncthreads();
    if (slopes != nullptr) {
        const float nbar = s_nbar;
        float *out = slopes + (size_t)f * 2 * nv;
        for (int i = threadIdx.x; i < nv; i += blockDim.x) {
            const int id = __ldg(t.vidx + i), jj = id / ns, ii = id - jj * ns;
            const float a = fr[jj * D + ii], b = fr[jj * D + ns + ii];
            const float c = fr[(ns + jj) * D + ii], d = fr[(ns + jj) * D + ns + ii];
            const float den = t.slope_norm == 1 ? ((a + b) + (c + d)) : nbar;
            out[i] = ((a + c) - (b + d)) / den;
            out[nv + i] = ((a + b) - (c + d)) / den;
        }
    }
}

}  // namespace pwk
