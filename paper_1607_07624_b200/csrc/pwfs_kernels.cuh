// pwfs_kernels.cuh -- the sm_100a kernels of the pyramid-WFS hot path.
//
// Structure.  The 2-D operator IDFT2 . mask . DFT2 with the
// separable pyramid mask m(u,v) = a(u) a(v) factors into two 1-D circular
// convolutions, E = Cy (P Cx^T), C = IDFT diag(a) DFT.  So instead of four 1-D
// passes with three round trips there are two fused passes with one:
//
//   xpass (K1): for every pupil ROW y (N of them, not M) and every distinct
//               x-tilt j: phasor A exp(i(phi + tilt_x)) -> length-M DFT over x
//               -> * a(u) -> inverse DFT -> keep only the window columns ->
//               T[f][j][xc][y]  (transposed so the column pass reads coalesced).
//   ypass (K2): one warp per needed COLUMN xc, looping over its modulation
//               points k: load T[.., xc, :] * tilt_y,k(y) -> DFT over y -> * a(v)
//               -> inverse DFT -> |E|^2 accumulated in registers over k ->
//               area-weighted rebin along y -> colbin[f][ks][xc][jy].
//   xrebin (K3a), slopes (K3b): finish the detector frame and the slopes.
//
// A length-M transform, M = 32*R1, is done by ONE WARP in two register stages
// with one shared-memory exchange: lane n2 does a DFT of size R1 over
// x[32 n1 + n2] (coalesced loads), the warp exchanges through padded shared
// memory, lane k1 does a DFT of size 32 over n2.  The inverse runs the same
// graph backwards, so forward+mask+inverse needs two exchanges and no
// bit-reversal, and results come back in natural order in the lane that loaded
// them.  To keep all 32 lanes busy in the size-32 stage when R1 < 32 a warp
// works on NB transforms at once (NB*R1 ~ 32).
#pragma once
#include "pwfs_dft.cuh"

#include <type_traits>

namespace pwk {

constexpr float kInv2PiHi = 0.15915493667125702f;   // fl32(1/(2 pi))
constexpr float kInv2PiLo = 6.4206382e-09f;          // 1/(2 pi) - kInv2PiHi
constexpr int kPitch = 33;  // float2 row pitch of the exchange buffer: conflict-free LDS.64/STS.64 along rows and columns
// T is stored in blocks of kTB consecutive rows y: T[f][j][y / kTB][x][y % kTB].  A row-pass CTA that owns kTB rows
// writes, per x-tilt, one contiguous block of M * kTB float2; the column pass reads 64-byte runs.
constexpr int kTB = 8;

// Padding (float2) of the exchange buffers.  Inside a warp's buffer the NB * R1 rows are contiguous (the size-32 stage
// reads row w at w * kPitch: 16 consecutive lanes hit 16 different 64-bit banks), except that a pad TPAD may separate
// the NB transforms when R1 is a multiple of 16 (a half warp of the size-32 stage then never straddles two transforms).
// The row pass's transposed last stage reads, per instruction, 8 rows r = 8 r_hi + r_lo of the CTA (= 8 transforms,
// spread over 8 / NB warps) x 2 columns per half warp -- adjacent columns n2, n2 + 1, or (SWAP) n2, n2 + 2 with the
// other half warp taking n2 + 1, n2 + 3: the warp covers the same 8 rows x 4 columns either way.  The pad between
// warps (bits 0-7 of the result), TPAD (bits 8-15) and SWAP (bit 16) are chosen so that those 16 accesses fall in as
// many different banks as possible: all 16 for NB = 1, for R1 = 6, 10, 18, with TPAD for R1 = 16, 32, 48, 64, and with
// SWAP for odd R1 and NB = 2 (R1 = 15, 25, 27: rows r, r + 1 are an odd number of banks apart).
constexpr int pick_pads(int R1, int NB, int RPC) {
    int best_code = 0, best = 1 << 30;
    const int tmax = (R1 % 16 == 0 && NB > 1) ? 16 : 1;
    for (int swap = 0; swap < 2; ++swap)
        for (int tpad = 0; tpad < tmax; ++tpad)
            for (int pad = 0; pad < 16; ++pad) {
                const int wb = NB * R1 * kPitch + (NB - 1) * tpad + pad;
                int tot = 0;
                for (int rhi = 0; rhi < RPC / kTB; ++rhi) {
                    int cnt[16] = {};
                    int worst = 0;
                    for (int rlo = 0; rlo < kTB; ++rlo) {
                        const int r = kTB * rhi + rlo;
                        const int off = (r / NB) * wb + (r % NB) * (R1 * kPitch + tpad);
                        for (int n2 = 0; n2 < 2; ++n2) {
                            const int c = ++cnt[(off + (swap ? 2 * n2 : n2)) % 16];
                            worst = c > worst ? c : worst;
                        }
                    }
                    tot += worst;
                }
                if (tot < best) { best = tot; best_code = swap * 65536 + tpad * 256 + pad; }
            }
    return best_code;
}

// YMODE_ (column pass): bit 0 = the T column is staged in shared memory by cp.async instead of waiting in registers,
// bit 1 = the size-32 stage keeps its 32 twiddles in registers for both multiplies, bit 2 = they are read once per
// kernel and stay in registers (single-round configurations: NB * R1 <= 32).
template <int R1_, int NB_, int WPB_X_, int WPB_Y_, int MINB_X_ = 1, int MINB_Y_ = 1, int YMODE_ = 0>
struct PassCfg {
    static constexpr int R1 = R1_;           // M / 32
    static constexpr int NB = NB_;           // transforms a warp works on at once
    static constexpr int M = 32 * R1_;
    static constexpr int NZ = (R1_ + 1) / 2; // M >= 2N  =>  at most ceil(R1/2) non-zero inputs per lane
    static constexpr int ITEMS = NB_ * R1_;  // size-32 DFTs per warp batch
    static constexpr int ROUNDS = (ITEMS + 31) / 32;
    static constexpr int TPAD = (pick_pads(R1_, NB_, NB_ * WPB_X_) >> 8) & 255;     // float2 between the NB transforms
    static constexpr bool SWAP = (pick_pads(R1_, NB_, NB_ * WPB_X_) >> 16) != 0;     // column order of the transposed stage
    static constexpr int TR_BUF = R1_ * kPitch + TPAD;                               // float2 per transform
    static constexpr int WARP_BUF = ITEMS * kPitch + (NB_ - 1) * TPAD + pick_pads(R1_, NB_, NB_ * WPB_X_) % 256;   // float2 per warp
    // offset of exchange row (transform b, k1) in the warp's buffer; w = b * R1 + k1
    __host__ __device__ static constexpr int row_off(int w) { return w * kPitch + (TPAD ? (w / R1_) * TPAD : 0); }
    static constexpr int TAB = R1_ * kPitch;              // float2 per table (twiddle, mask)
    // M = 2048: the row pass's shared memory is full, the general-mask table a(u)/M is read through L1 instead
    static constexpr bool AM_GLOBAL = R1_ > 32;
    static constexpr int AM_PITCH = AM_GLOBAL ? 32 : kPitch;
    static constexpr int WPB_X = WPB_X_;     // warps per CTA, row pass
    static constexpr int WPB_Y = WPB_Y_;     // warps per CTA, column pass
    static constexpr int MINB_X = MINB_X_;   // CTAs per SM the register allocation must allow
    static constexpr int MINB_Y = MINB_Y_;
    static constexpr int RPC = NB_ * WPB_X_; // rows per CTA, row pass
    static_assert(RPC % kTB == 0, "row pass: rows per CTA must be whole y-blocks of T");
    // row pass: tables (no mask table for the quarter mask) + exchange buffers + base phasor [RPC][NZ][32]
    static constexpr size_t smem_x_q = (size_t)(WPB_X_ * WARP_BUF + 1 * TAB + RPC * NZ * 32) * sizeof(float2);
    static constexpr size_t smem_x_t = (size_t)(WPB_X_ * WARP_BUF + (AM_GLOBAL ? 1 : 2) * TAB + RPC * NZ * 32) * sizeof(float2);
    // column pass: tables + exchange buffers (+ the staged T column [NB][NZ][32] per warp when Y_ASYNC)
    static constexpr int YMODE = YMODE_;
    static constexpr bool Y_ASYNC = (YMODE_ & 1) != 0;
    static constexpr bool Y_TWKEEP = (YMODE_ & 2) != 0;
    static constexpr bool Y_TWRES = (YMODE_ & 4) != 0;     // twiddles resident in registers for the whole kernel
    static constexpr int PRE_BUF = Y_ASYNC ? NB_ * NZ * 32 : 0;
    static constexpr size_t smem_y_q = (size_t)(WPB_Y_ * (WARP_BUF + PRE_BUF) + 1 * TAB) * sizeof(float2);
    static constexpr size_t smem_y_t = (size_t)(WPB_Y_ * (WARP_BUF + PRE_BUF) + (AM_GLOBAL ? 1 : 2) * TAB) * sizeof(float2);
};

// Device-side view of a sensor's tables (all pointers are device memory).
struct DevTables {
    int N, M, NP;             // pupil px, grid, y-extent of T and tyt (N rounded up to 32; padding is zero)
    int NXP;                  // x-pitch of txc (32 * ceil(R1/2) >= N; padding is zero)
    int K, KX;                // modulation points, distinct x-tilts
    int ncols;                // pupil-plane columns computed
    int D, n_sub, cmax;       // detector size 2 n_sub, rebin support
    int n_valid, slope_norm;
    int t_frames;             // frames T holds (normally the chunk; 1 = every frame aliases slab set 0: a timing experiment)
    float *dbg_I;             // test-only (pwfs_debug_intensity): [F][ncols][M] full-resolution sum_k |E|^2, else nullptr
    const float *amp;         // [N][N]
    const float2 *txc;        // [KX][NXP] exp(i tilt_x,j(x)), zero for x >= N
    const float2 *tyt;        // [K][NP]  exp(i tilt_y,k(y)), zero for y >= N
    const int *jx;            // [K]      x-tilt index of modulation point k
    const int *korder;        // [K]      the modulation points sorted by x-tilt index
    const int2 *kj;           // [K]      (korder[i], jx[korder[i]])
    const float2 *tw;         // [R1][32] exp(-2 pi i k1 n2 / M)
    const float2 *am;         // [R1][32] a(k1 + R1 k2) / M
    const int *colx;          // [ncols]  grid x of compact column xc
    const int *xc_of_x;       // [M]      compact column of grid x (or -1)
    const int *rb_start;      // [D]      first source px (grid coordinate) of detector bin
    const int *rb_cnt;        // [D]
    const float *rb_w;        // [D][cmax] area weights
    const int *vidx;          // [n_valid] j*n_sub + i of valid subapertures, row-major
    const unsigned char *vmask;   // [n_sub][n_sub] 1 = valid subaperture
};

template <bool QM, bool AM_GLOBAL = false>
__device__ __forceinline__ void load_tables(float2 *s_tw, float2 *s_am, const DevTables &t, int R1) {
    for (int i = threadIdx.x; i < R1 * 32; i += blockDim.x) {
        int k1 = i >> 5, n2 = i & 31;
        s_tw[k1 * kPitch + n2] = t.tw[i];
        if constexpr (!QM && !AM_GLOBAL) s_am[k1 * kPitch + n2] = t.am[i];
    }
}

// Inverse DFT-32 whose inputs x[16..32) carry a run-time sign sg = +-1 (both halves of sg2):
// X = IDFT32(x[0..16), sg * x[16..32)).  Split 32 = 16 x 2: the size-2 butterflies on the pairs
// (x[p], x[p+16]) absorb the sign as FFMA2s in place of FADD2s, so it costs nothing.
__device__ __forceinline__ void idft32_signed_upper(float2 (&x)[32], float2 sg2) {
    float2 e[16], o[16];
    const float2 nsg2 = make_float2(-sg2.x, -sg2.y);
    sfor<16>([&](auto pc) {
        constexpr int p = decltype(pc)::value;
        e[p] = __ffma2_rn(x[p + 16], sg2, x[p]);
        o[p] = mul_w<p, 32, +1>(__ffma2_rn(x[p + 16], nsg2, x[p]));
    });
    Dft<16, +1>::run(e);
    Dft<16, +1>::run(o);
    sfor<16>([&](auto jc) {
        constexpr int j = decltype(jc)::value;
        x[2 * j] = e[j];
        x[2 * j + 1] = o[j];
    });
}

// Size-32 stage for the warp's current batch: for every (transform b, k1):
// twiddle, DFT over n2, mask, inverse DFT, conjugate twiddle; in place in `buf`.
//
// QM = true is the default mask s = M/4 (M % 4 == 0), whose 1-D factor is a power of i:
// a(u) = i^|u~|, i.e. i^u for u < M/2 and i^-u above.  With u = k1 + R1 k2 (k2 >= 16 <=> u >= M/2)
//   a(u) = i^k1 * i^(R1 k2)              k2 < 16
//        = i^k1 * (-1)^k1 * i^(-R1 k2)   k2 >= 16
// i^(+-R1 k2) is a compile-time swap/negate (operand modifiers, no instruction), (-1)^k1 is a
// per-lane sign absorbed by idft32_signed_upper, and i^k1 is applied where k1 is a compile-time
// register index (step A' of the callers, apply_ipow_k1).  The mask and its table cost nothing;
// the 1/M per axis moves into the final frame scale.
// TW = 1 (keep): the 32 twiddles of the lane are read once into registers and serve both multiplies (64 registers for a
// third less shared-memory traffic in this stage); TW = 0: the compiler decides whether the second multiply re-reads
// them; TW = 2 (resident, single-round configurations only: the lane's k1 never changes): the caller read them once,
// before its loop over the modulation points, and passes them in `twres`.
template <class C, bool QM, int TW = 0>
__device__ __forceinline__ void stage32(float2 *buf, const float2 *s_tw, const float2 *s_am, int lane,
                                        const float2 *twres = nullptr) {
    constexpr bool KEEP = TW == 1;
    static_assert(TW != 2 || C::ROUNDS == 1, "resident twiddles need a single round of the size-32 stage");
#pragma unroll
    for (int rd = 0; rd < C::ROUNDS; ++rd) {
        int w = rd * 32 + lane;
        if (w < C::ITEMS) {
            const int k1 = w % C::R1;
            float2 *row = buf + C::row_off(w);
            const float2 *twr = s_tw + k1 * kPitch;
            float2 u[32];
            [[maybe_unused]] float2 twv[KEEP ? 32 : 1];
#pragma unroll
            for (int n2 = 0; n2 < 32; ++n2) {
                if constexpr (KEEP) { twv[n2] = twr[n2]; u[n2] = cmul(row[n2], twv[n2]); }
                else if constexpr (TW == 2) u[n2] = cmul(row[n2], twres[n2]);
                else u[n2] = cmul(row[n2], twr[n2]);
            }
            Dft<32, -1>::run(u);
            if constexpr (QM) {
                sfor<32>([&](auto kc) {
                    constexpr int k2 = decltype(kc)::value;
                    constexpr int e = k2 < 16 ? (C::R1 * k2) % 4 : (4 - (C::R1 * k2) % 4) % 4;
                    u[k2] = mul_w<e, 4, +1>(u[k2]);
                });
                const float sg = (k1 & 1) ? -1.f : 1.f;
                idft32_signed_upper(u, make_float2(sg, sg));
            } else {
                const float2 *amr = s_am + k1 * C::AM_PITCH;      // shared memory, or t.am itself (AM_GLOBAL)
#pragma unroll
                for (int k2 = 0; k2 < 32; ++k2) u[k2] = cmul(u[k2], amr[k2]);
                Dft<32, +1>::run(u);
            }
#pragma unroll
            for (int n2 = 0; n2 < 32; ++n2) row[n2] = cmulc(u[n2], KEEP ? twv[n2] : TW == 2 ? twres[n2] : twr[n2]);
        }
    }
}

// i^k1 of the quarter mask, applied to the register that holds index k1 (free: operand modifiers).
template <int R1, bool QM>
__device__ __forceinline__ void apply_ipow_k1(float2 (&v)[R1]) {
    if constexpr (QM) {
        sfor<R1>([&](auto kc) {
            constexpr int k1 = decltype(kc)::value;
            v[k1] = mul_w<k1 % 4, 4, +1>(v[k1]);
        });
    }
}

// ------------------------------------------------------------------ K1 ------
// grid (ceil(NP/RPC), jsplit, F); block 32*WPB_X.  Warp wl of the CTA owns rows
// y0 + wl*NB + b, b < NB, of frame f and loops over its share of the distinct x-tilts j.
//
// The base phasor A exp(i phi) is computed ONCE (one range-reduced MUFU sincos per pupil
// pixel per CTA) and parked in shared memory; per x-tilt it is multiplied by the table
// exp(i tilt_x,j(x)) -- the tilt is separable, so this is the whole k-dependence of the
// row pass.  Rows N <= y < NP carry a zero phasor and come out zero.
//
// The last register stage is done "transposed": thread (r, n2) takes row r of the CTA
// (another warp's exchange buffer) and column residue n2, so that adjacent lanes hold
// adjacent rows y of the same column x = 32 n1 + n2.  T is blocked by kTB rows,
// T[f][j][y / 8][x][y % 8]: the 8 lanes (r % 8) x 4 adjacent n2 of a warp write 256 contiguous
// bytes per store, every store of a thread is a compile-time offset (n1 * 256 float2) from one
// base address, and a CTA's output per x-tilt is RPC/8 contiguous blocks of M * 64 bytes -- no
// staging pass for the transposition, no address arithmetic, no partial lines.  All M columns
// are written (T spans the whole grid); the column pass reads the window columns only.
template <class C, bool QM>
__global__ void __launch_bounds__(32 * C::WPB_X, C::MINB_X)
xpass_kernel(DevTables t, const float *__restrict__ phase, float2 *__restrict__ T, int jsplit) {
    extern __shared__ float2 smem[];
    float2 *s_tw = smem;
    const float2 *s_am = C::AM_GLOBAL ? t.am : smem + C::TAB;  // unused (zero-sized) when QM
    float2 *s_buf = smem + ((QM || C::AM_GLOBAL) ? 1 : 2) * C::TAB;
    float2 *s_p = s_buf + C::WPB_X * C::WARP_BUF;              // [RPC][NZ][32] base phasor
    const int lane = threadIdx.x & 31, wl = threadIdx.x >> 5;
    const int N = t.N;
    const int js = blockIdx.y, f = blockIdx.z;
    const int y0 = blockIdx.x * C::RPC;
    float2 *buf = s_buf + wl * C::WARP_BUF;
    float2 *pw = s_p + (size_t)wl * C::NB * C::NZ * 32 + lane;

    load_tables<QM, C::AM_GLOBAL>(s_tw, smem + C::TAB, t, C::R1);

    // a1: base phasor of this warp's rows, x = 32 n1 + lane
#pragma unroll
    for (int b = 0; b < C::NB; ++b) {
        const int y = y0 + wl * C::NB + b;
        const float *ph_row = phase + ((size_t)f * N + y) * N + lane;
        const float *a_row = t.amp + (size_t)y * N + lane;
        float ph[C::NZ], am[C::NZ];
#pragma unroll
        for (int n1 = 0; n1 < C::NZ; ++n1) {
            const bool ok = (y < N) && (32 * n1 + lane < N);
            ph[n1] = ok ? __ldg(ph_row + 32 * n1) : 0.f;
            am[n1] = ok ? __ldg(a_row + 32 * n1) : 0.f;
        }
#pragma unroll
        for (int n1 = 0; n1 < C::NZ; ++n1) {
            // phase in turns: ph/(2 pi) with 1/(2 pi) = kInv2PiHi + kInv2PiLo; q is an exact integer and
            // the FMAs keep the low bits of the product, so the reduction costs no accuracy at |ph| ~ 100 rad
            const float q = rintf(ph[n1] * kInv2PiHi);
            float tr = fmaf(ph[n1], kInv2PiHi, -q);
            tr = fmaf(ph[n1], kInv2PiLo, tr);
            float sn, cs;
            __sincosf(tr * 6.283185307179586f, &sn, &cs);
            pw[(b * C::NZ + n1) * 32] = make_float2(am[n1] * cs, am[n1] * sn);
        }
    }

    // transposed last stage: this thread's items it < NB are (row r = 8 r_hi + r_lo, column residue n2) with
    // r_lo = i % 8, n2 = (i / 8) % 32 (its two low bits exchanged when C::SWAP), r_hi = i / 256 for i = threadIdx.x + it * blockDim.x
    int item_src[C::NB];          // exchange-buffer offset of (row r, k1 = 0, n2): transform r of the CTA
    int item_dst[C::NB];          // T offset of (x = n2, y = y0 + r) within the (f, j) slab; < 0: row beyond NP
#pragma unroll
    for (int it = 0; it < C::NB; ++it) {
        const int i = threadIdx.x + it * 32 * C::WPB_X;
        const int g = (i >> 3) & 31;
        const int r = (i >> 8) * kTB + (i & 7), n2 = C::SWAP ? ((g & ~3) | ((g & 1) << 1) | ((g >> 1) & 1)) : g;
        item_src[it] = (r / C::NB) * C::WARP_BUF + (r % C::NB) * C::TR_BUF + n2;
        item_dst[it] = (y0 + r < t.NP) ? ((y0 + r) / kTB) * (C::M * kTB) + n2 * kTB + (i & 7) : -1;
    }

    const int j_lo = (int)(((long long)js * t.KX) / jsplit), j_hi = (int)(((long long)(js + 1) * t.KX) / jsplit);
    const size_t slab = (size_t)C::M * t.NP;
    __syncthreads();   // tables loaded (s_p is private to the warp that wrote it)
    // the x-tilt table row of the NEXT tilt is fetched into registers while this tilt's size-32 stage and write-out
    // run: with the shared memory this kernel uses L1 keeps ~10 KB, so a load at the point of use waits for L2
    float2 tx[C::NZ];
    {
        const float2 *txj = t.txc + (size_t)j_lo * t.NXP + lane;
#pragma unroll
        for (int n1 = 0; n1 < C::NZ; ++n1) tx[n1] = __ldg(txj + 32 * n1);
    }
    for (int j = j_lo; j < j_hi; ++j) {
        // step A: x-tilt, zero-padded DFT of size R1 over n1
#pragma unroll
        for (int b = 0; b < C::NB; ++b) {
            float2 v[C::R1];
#pragma unroll
            for (int n1 = 0; n1 < C::NZ; ++n1) v[n1] = cmul(pw[(b * C::NZ + n1) * 32], tx[n1]);
            DftP<C::R1, -1, C::NZ>::run(v);
#pragma unroll
            for (int k1 = 0; k1 < C::R1; ++k1) buf[C::row_off(b * C::R1 + k1) + lane] = v[k1];
        }
        if (j + 1 < j_hi) {
            const float2 *txj = t.txc + (size_t)(j + 1) * t.NXP + lane;
#pragma unroll
            for (int n1 = 0; n1 < C::NZ; ++n1) tx[n1] = __ldg(txj + 32 * n1);
        }
        __syncwarp();
        stage32<C, QM>(buf, s_tw, s_am, lane);
        __syncthreads();
        // step A'': inverse DFT of size R1 over k1 for item (r, n2) -> T[f][j][(y0 + r) / 8][32 n1 + n2][r % 8]
        float2 *Tj = T + ((size_t)(t.t_frames == 1 ? 0 : f) * t.KX + j) * slab;
#pragma unroll
        for (int it = 0; it < C::NB; ++it) {
            float2 v[C::R1];
            const float2 *src = s_buf + item_src[it];
#pragma unroll
            for (int k1 = 0; k1 < C::R1; ++k1) v[k1] = src[k1 * kPitch];
            apply_ipow_k1<C::R1, QM>(v);
            Dft<C::R1, +1>::run(v);
            // Under this guard ptxas moves each value to one register pair before its store, so a store is issued only
            // when the LSU has taken the previous one (ncu: those moves wait on the long scoreboard).  That pacing is
            // measured to HELP: with unguarded stores interleaved among the butterflies the same instruction mix runs
            // 5 % slower (M = 1024: 3.19 vs 3.03 ms per 100 frames; profiles/r2_tuning.md) -- bursts of stores delay
            // the shared-memory traffic of the warps that are in their size-32 stage.
            if (item_dst[it] >= 0) {
                float2 *dst = Tj + item_dst[it];
#pragma unroll
                for (int n1 = 0; n1 < C::R1; ++n1) dst[n1 * (32 * kTB)] = v[n1];
            }
        }
        __syncthreads();   // the next x-tilt overwrites the buffers
    }
}

// ------------------------------------------------------------------ K2 ------
// grid (ceil(ncols / (NB*WPB_Y)), ksplit, F); block 32*WPB_Y.  Warps are
// independent: warp -> NB adjacent columns, loops over its share of k.  The
// inputs of modulation point k+1 are fetched into registers while point k is
// being transformed (T streams from HBM/L2 once; nothing else leaves the SM).
template <class C, bool QM>
__global__ void __launch_bounds__(32 * C::WPB_Y, C::MINB_Y)
ypass_kernel(DevTables t, const float2 *__restrict__ T, float *__restrict__ colbin, int ksplit) {
    extern __shared__ float2 smem[];
    float2 *s_tw = smem;
    const float2 *s_am = C::AM_GLOBAL ? t.am : smem + C::TAB;
    float2 *s_buf = smem + ((QM || C::AM_GLOBAL) ? 1 : 2) * C::TAB;
    const int lane = threadIdx.x & 31, wl = threadIdx.x >> 5;
    const int NP = t.NP;
    const int ks = blockIdx.y, f = blockIdx.z;
    const int xc0 = (blockIdx.x * C::WPB_Y + wl) * C::NB;
    float2 *buf = s_buf + wl * C::WARP_BUF;
    [[maybe_unused]] float2 *spre = s_buf + C::WPB_Y * C::WARP_BUF + wl * C::PRE_BUF + lane;   // Y_ASYNC: [NB][NZ][32]

    load_tables<QM, C::AM_GLOBAL>(s_tw, smem + C::TAB, t, C::R1);
    __syncthreads();
    if (xc0 >= t.ncols) return;

    float acc[C::NB][C::R1];
#pragma unroll
    for (int b = 0; b < C::NB; ++b)
#pragma unroll
        for (int n1 = 0; n1 < C::R1; ++n1) acc[b][n1] = 0.f;

    const int k_lo = (int)(((long long)ks * t.K) / ksplit), k_hi = (int)(((long long)(ks + 1) * t.K) / ksplit);
    // T[f][j][y / 8][x][y % 8]: grid column x of compact column xc from the colx table (windows may leave gaps);
    // lane reads y = 32 n1 + lane, i.e. block 4 n1 + lane / 8, row lane % 8 of it: 64-byte runs
    const size_t frame_stride = (size_t)C::M * NP;
    const float2 *Tf = T + (size_t)(t.t_frames == 1 ? 0 : f) * t.KX * frame_stride + (lane >> 3) * (C::M * kTB) + (lane & 7);
    constexpr int colmul = kTB, n1_stride = 32 * C::M;
    int colofs[C::NB];
#pragma unroll
    for (int b = 0; b < C::NB; ++b) colofs[b] = (xc0 + b < t.ncols) ? __ldg(t.colx + xc0 + b) * colmul : 0;

    // The warp walks its share of the modulation points in x-tilt order (kj): points that share a slab T[f][j] come
    // one after the other and the column is fetched once for them.  The column of the NEXT slab is fetched while the
    // current point is transformed: into registers, or (Y_ASYNC) staged in shared memory by cp.async -- no registers
    // held across the size-32 stage, 12 warps per SM instead of 8; every lane writes and reads only its own slots, so
    // the only ordering needed is cp.async.wait_all in the lane.  (Staging the y-tilt row the same way was measured
    // slower: M = 1024 9.72 vs 9.54 ms per 100 frames.)
    [[maybe_unused]] float2 pre[C::Y_ASYNC ? 1 : C::NB][C::Y_ASYNC ? 1 : C::NZ];
    if constexpr (C::Y_ASYNC) {
#pragma unroll
        for (int i = 0; i < C::NB * C::NZ; ++i) spre[i * 32] = make_float2(0.f, 0.f);
    }
    auto fetch = [&](int j) {
        const float2 *src = Tf + (size_t)j * frame_stride;
#pragma unroll
        for (int b = 0; b < C::NB; ++b)
#pragma unroll
            for (int n1 = 0; n1 < C::NZ; ++n1) {
                if constexpr (C::Y_ASYNC) {
                    if (32 * n1 < NP && xc0 + b < t.ncols) {
                        const unsigned dst = (unsigned)__cvta_generic_to_shared(spre + (b * C::NZ + n1) * 32);
                        asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst), "l"(src + colofs[b] + n1 * n1_stride) : "memory");
                    }
                } else {
                    pre[b][n1] = (32 * n1 < NP && xc0 + b < t.ncols) ? __ldg(src + colofs[b] + n1 * n1_stride)
                                                                     : make_float2(0.f, 0.f);
                }
            }
    };
    [[maybe_unused]] float2 twres[C::Y_TWRES ? 32 : 1];
    if constexpr (C::Y_TWRES) {
        const float2 *twr = s_tw + (lane % C::R1) * kPitch;
#pragma unroll
        for (int n2 = 0; n2 < 32; ++n2) twres[n2] = twr[n2];
    }
    int2 kj = make_int2(0, -1), kj_next = make_int2(0, -1), kj_next2 = make_int2(0, -1);
    if (k_lo < k_hi) {
        kj_next = __ldg(t.kj + k_lo);
        if (k_lo + 1 < k_hi) kj_next2 = __ldg(t.kj + k_lo + 1);
        fetch(kj_next.y);
    }
    for (int idx = k_lo; idx < k_hi; ++idx) {
        kj = kj_next; kj_next = kj_next2;
        if (idx + 2 < k_hi) kj_next2 = __ldg(t.kj + idx + 2);
        const int k = kj.x, j = kj.y, j_next = kj_next.y;
        const float2 *ty = t.tyt + (size_t)k * NP + lane;
        float2 tyv[C::NZ];
#pragma unroll
        for (int n1 = 0; n1 < C::NZ; ++n1) tyv[n1] = (32 * n1 < NP) ? __ldg(ty + 32 * n1) : make_float2(0.f, 0.f);
        if constexpr (C::Y_ASYNC) asm volatile("cp.async.wait_all;" ::: "memory");
#pragma unroll
        for (int b = 0; b < C::NB; ++b) {
            float2 v[C::R1];
#pragma unroll
            for (int n1 = 0; n1 < C::NZ; ++n1) {
                if constexpr (C::Y_ASYNC) v[n1] = cmul(spre[(b * C::NZ + n1) * 32], tyv[n1]);
                else v[n1] = cmul(pre[b][n1], tyv[n1]);
            }
            if (b == C::NB - 1 && idx + 1 < k_hi && j_next != j) fetch(j_next);
            DftP<C::R1, -1, C::NZ>::run(v);
#pragma unroll
            for (int k1 = 0; k1 < C::R1; ++k1) buf[C::row_off(b * C::R1 + k1) + lane] = v[k1];
        }
        __syncwarp();
        stage32<C, QM, C::Y_TWRES ? 2 : C::Y_TWKEEP ? 1 : 0>(buf, s_tw, s_am, lane, twres);
        __syncwarp();
#pragma unroll
        for (int b = 0; b < C::NB; ++b) {
            float2 v[C::R1];
#pragma unroll
            for (int k1 = 0; k1 < C::R1; ++k1) v[k1] = buf[C::row_off(b * C::R1 + k1) + lane];
            apply_ipow_k1<C::R1, QM>(v);
            Dft<C::R1, +1>::run(v);
#pragma unroll
            for (int n1 = 0; n1 < C::R1; ++n1) acc[b][n1] = fmaf(v[n1].x, v[n1].x, fmaf(v[n1].y, v[n1].y, acc[b][n1]));
        }
        // next iteration's step-A stores touch only this lane's column, which only this lane read
    }
    // y-rebin: column of summed intensity -> 2 n_sub detector rows
    float *colI = reinterpret_cast<float *>(buf);          // NB*M floats <= the warp's buffer
    __syncwarp();
#pragma unroll
    for (int b = 0; b < C::NB; ++b)
#pragma unroll
        for (int n1 = 0; n1 < C::R1; ++n1) colI[b * C::M + 32 * n1 + lane] = acc[b][n1];
    __syncwarp();
    if (t.dbg_I != nullptr) {   // test-only export of the un-rebinned column (pins P2 / P7 of SURVEY.md 8(c))
        for (int b = 0; b < C::NB && xc0 + b < t.ncols; ++b)
            for (int y = lane; y < C::M; y += 32) t.dbg_I[((size_t)f * t.ncols + xc0 + b) * C::M + y] = colI[b * C::M + y];
    }
    const int D = t.D, cmax = t.cmax;
    for (int b = 0; b < C::NB; ++b) {
        const int xc = xc0 + b;
        if (xc >= t.ncols) break;
        float *out = colbin + (((size_t)f * ksplit + ks) * t.ncols + xc) * D;
        for (int jj = lane; jj < D; jj += 32) {
            int y = __ldg(t.rb_start + jj);
            const int cnt = __ldg(t.rb_cnt + jj);
            const float *w = t.rb_w + (size_t)jj * cmax;
            float s = 0.f;
            for (int c = 0; c < cnt; ++c) {
                s = fmaf(__ldg(w + c), colI[b * C::M + y], s);
                if (++y == C::M) y = 0;
            }
            out[jj] = s;
        }
    }
}

// ------------------------------------------------------------------ K3a -----
// frame[f][jy][jx] = (1/K) sum_ks sum_c wx[jx][c] colbin[f][ks][xc(jx,c)][jy], and this detector column's share of
// the slope normalisation: nsum[f][jx] = sum over jy of the pixels that belong to valid subapertures.
// grid (D (jx), F); block covers jy.  Source columns are taken four at a time so that their loads are in flight
// together (a single frame in a closed loop is latency-bound here).
static __global__ void xrebin_kernel(DevTables t, const float *__restrict__ colbin, float *__restrict__ frames,
                                     float *__restrict__ nsum, int ksplit, float scale) {
    __shared__ float red[8];
    const int jx = blockIdx.x, f = blockIdx.y;
    const int D = t.D, ns = t.n_sub;
    const int x = __ldg(t.rb_start + jx);
    const int cnt = __ldg(t.rb_cnt + jx);
    const float *w = t.rb_w + (size_t)jx * t.cmax;
    const int ix = jx >= ns ? jx - ns : jx;
    float part = 0.f;
    for (int jy = threadIdx.x; jy < D; jy += blockDim.x) {
        float s = 0.f;
        for (int c0 = 0; c0 < cnt; c0 += 4) {
            int xc[4];
            float wc[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const bool ok = c0 + u < cnt;
                int xx = x + c0 + u;
                if (xx >= t.M) xx -= t.M;
                xc[u] = ok ? __ldg(t.xc_of_x + xx) : 0;
                wc[u] = ok ? __ldg(w + c0 + u) : 0.f;
            }
            if (ksplit < 3) {                                  // batches: one or two k-splits, four loads in flight
                for (int ks = 0; ks < ksplit; ++ks) {
                    const float *src = colbin + ((size_t)f * ksplit + ks) * t.ncols * D + jy;
                    float v[4];
#pragma unroll
                    for (int u = 0; u < 4; ++u) v[u] = c0 + u < cnt ? __ldg(src + (size_t)xc[u] * D) : 0.f;
#pragma unroll
                    for (int u = 0; u < 4; ++u) s = fmaf(wc[u], v[u], s);
                }
                continue;
            }
            // four k-splits x four columns = up to 16 loads in flight (a single frame has 6-12 k-splits and this kernel
            // is nothing but load latency); absent entries add an exact zero, the order of the sum stays ks-major
            for (int ks0 = 0; ks0 < ksplit; ks0 += 4) {
                float v[4][4];
#pragma unroll
                for (int kk = 0; kk < 4; ++kk) {
                    const float *src = colbin + ((size_t)f * ksplit + min(ks0 + kk, ksplit - 1)) * t.ncols * D + jy;
#pragma unroll
                    for (int u = 0; u < 4; ++u)
                        v[kk][u] = (ks0 + kk < ksplit && c0 + u < cnt) ? __ldg(src + (size_t)xc[u] * D) : 0.f;
                }
#pragma unroll
                for (int kk = 0; kk < 4; ++kk)
#pragma unroll
                    for (int u = 0; u < 4; ++u) s = fmaf(wc[u], v[kk][u], s);
            }
        }
        s *= scale;
        frames[((size_t)f * D + jy) * D + jx] = s;
        const int iy = jy >= ns ? jy - ns : jy;
        if (__ldg(t.vmask + iy * ns + ix)) part += s;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = part;
    __syncthreads();
    if (threadIdx.x == 0) {
        float v = 0.f;
        for (int i = 0; i < (int)((blockDim.x + 31) >> 5); ++i) v += red[i];
        nsum[(size_t)f * D + jx] = v;
    }
}

// test-only: dbg[f][xc][y] (corner-placed grid, unscaled) -> I[f][(y + o) % M][(x + o) % M] * scale, the oracle's
// centred coordinates; columns that were not computed stay zero (I is cleared by the caller).  grid (ncols, F).
static __global__ void debug_scatter_kernel(DevTables t, const float *__restrict__ dbg, float *__restrict__ I, int o,
                                            float scale) {
    const int xc = blockIdx.x, f = blockIdx.y, M = t.M;
    const int x = (__ldg(t.colx + xc) + o) % M;
    const float *src = dbg + ((size_t)f * t.ncols + xc) * M;
    for (int y = threadIdx.x; y < M; y += blockDim.x) I[((size_t)f * M + (y + o) % M) * M + x] = src[y] * scale;
}

// ------------------------------------------------------------------ K3b -----
// grid (ceil(n_valid / 256), F); block 256.  nbar = (1 / n_valid) sum_jx nsum[f][jx], added in one fixed order by
// every CTA of the frame (same value everywhere, no second pass over the frame), then the slopes of 256 subapertures.
static __global__ void slopes_kernel(DevTables t, const float *__restrict__ frames, const float *__restrict__ nsum,
                                     float *__restrict__ slopes) {
    __shared__ float s_nbar;
    const int f = blockIdx.y, D = t.D, ns = t.n_sub, nv = t.n_valid;
    if (threadIdx.x < 32) {
        float v = 0.f;
        for (int j = threadIdx.x; j < D; j += 32) v += __ldg(nsum + (size_t)f * D + j);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (threadIdx.x == 0) s_nbar = v / (float)nv;
    }
    __syncthreads();
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nv) return;
    const float nbar = s_nbar;
    const float *fr = frames + (size_t)f * D * D;
    const int id = __ldg(t.vidx + i), jj = id / ns, ii = id - jj * ns;
    const float a = fr[jj * D + ii], b = fr[jj * D + ns + ii];
    const float c = fr[(ns + jj) * D + ii], d = fr[(ns + jj) * D + ns + ii];
    const float den = t.slope_norm == 1 ? ((a + b) + (c + d)) : nbar;
    float *out = slopes + (size_t)f * 2 * nv;
    out[i] = ((a + c) - (b + d)) / den;
    out[nv + i] = ((a + b) - (c + d)) / den;
}

}  // namespace pwk
