// rec_tc.cu -- f2, modal reconstructor for a BATCH of frames on the 5th-generation
// tensor cores: modes[b][m] = sum_j recmat[m][j] slopes[b][j] (reading F2g).
//
// This is the one dense contraction of the chain (n_modes x n_slopes x B).  The FP32 bar of the
// parity tests (|d| <= 1e-5 sum |R||s|) rules out single-pass TF32 (2^-11 per operand), so every
// operand is split into two TF32-representable planes, x = hi + lo + O(2^-22 |x|), and the product is
//   R S^T ~= Rhi Shi^T + Rhi Slo^T + Rlo Shi^T        (dropped terms <= 3 * 2^-22 |R||S| = 7e-7)
// accumulated in FP32 in tensor memory: three tcgen05.mma.kind::tf32 per K step, same accumulator.
// recmat is streamed from HBM as it is (FP32, 4 bytes per element) and split INSIDE the pipeline; the
// (small) slope planes are written by a split kernel per call.
//
// Kernel (TWO neighbouring 128 x 128 output tiles of one K split per CTA, 320 threads):
//   warp 0 (one lane)  TMA producer: four 128 x 32 FP32 boxes per stage (two raw recmat tiles, Shi, Slo; 128-byte
//                      swizzle) into a 3-stage ring of 64 KB, completion on the stage's "full" mbarrier;
//   warps 2-9          converters: two warps per TMEM lane quarter, thread = (row of a recmat tile, half of its 32 K
//                      values); reads its 16 raw values of each tile (undoing the swizzle in the address),
//                      hi = tf32(x), lo = tf32(x - hi), and writes both planes into one of two slots of TENSOR MEMORY
//                      (tcgen05.st 32x32b.x16: lane = row, column = k) once the MMAs that read the slot last have
//                      retired ("tfree" mbarrier), then arrives on the slot's "conv" mbarrier;
//   warp 1 (one lane)  MMA issuer: waits for "conv", per stage 4 K steps x 2 tiles x 3 UMMAs (M 128, N = frames
//                      rounded up to 16, K 8), A (recmat hi / lo) from tensor memory, B (slope planes) from
//                      shared-memory descriptors, into two accumulators of 128 TMEM columns; tcgen05.commit
//                      releases the stage ("empty") and the slot ("tfree") and, after the last one, signals the
//                      epilogue;
//   warps 2-9 again    epilogue: tcgen05.ld 32 lanes x 32 columns at a time, rows = modes so that a
//                      column store is one coalesced 128-byte line of modes[b][m0..m0+32).
// Tile pairs x K splits ~ number of SMs; the split-K partial sums are added in a fixed order by a second
// kernel (deterministic, no atomics).  Per stage the CTA needs 32 KB from HBM and 32 KB of slope planes out of L2
// and issues 24 UMMAs; measured, the kernel runs at the rate those short UMMAs issue at (~97 cycles each, tensor pipe
// 61 %; DESIGN.md 11 f2, profiles/r2_tuning.md section 11).
#include "rec_tc.cuh"

#include <cuda.h>

#include <algorithm>
#include <cstdint>
#include <cstdlib>
#include <new>

#include "../../include/pwfs.h"

namespace {

constexpr int BM = 128, BN = 128, BK = 32, UK = 8, STAGES = 3;
constexpr int TM = 2;                                 // m tiles (of 128 modes) per CTA: they share the slope planes of a stage
constexpr int TSLOTS = 2;                             // slots of converted recmat planes in tensor memory
constexpr int kTileBytes = BM * BK * 4;               // 16 KB, one operand plane of one stage
constexpr int kStageBytes = (TM + 2) * kTileBytes;    // TM raw recmat tiles, Shi, Slo
constexpr int kThreads = 320;                         // warp 0 TMA, warp 1 MMA, warps 2..9 converters / epilogue
constexpr uint32_t kAccCols = 128 * TM;               // accumulators: TMEM columns [0, 128 TM)
constexpr uint32_t kTmemCols = 512;                   // + per slot and m tile 32 columns of recmat hi and 32 of lo: 256 + 2 * 2 * 64
static_assert(kAccCols + TSLOTS * TM * 64 <= kTmemCols, "tensor memory budget");
constexpr int kLoadBytes = kStageBytes;               // what TMA brings per stage
constexpr int kConvThreads = 256;                     // warps 2..9: two per TMEM lane quarter, 16 K values each
constexpr size_t kSmemBytes = (size_t)STAGES * kStageBytes + 1024 /* alignment slack */ + 256 /* barriers */;
static_assert(BK * 4 == 128, "one K block is one 128-byte swizzle row");

// tcgen05 instruction descriptor, kind::tf32: D = F32 (bits 4-5 = 1), A = B = TF32 (bits 7-9, 10-12 = 2),
// both K-major (bits 15, 16 = 0), N >> 3 at bits 17-22, M >> 4 at bits 24-28.
// N is the frames of the tile rounded up to 16 (B = 100: N = 112, an eighth fewer tensor cycles than the full tile).
__host__ __device__ constexpr uint32_t idesc_for(int n) {
    return (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(BM >> 4) << 24);
}

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
// Nearest TF32 value (10 mantissa bits, low 13 bits zero) by integer arithmetic: add half a TF32 ulp to the magnitude
// and clear the low bits.  Two ALU instructions; cvt.rna.tf32.f32 is emulated on sm_100a with ~6 (ncu: the converter
// warps were the pipeline's bottleneck with it).  Differs from cvt.rna only on exact ties (away from zero both) and
// leaves Inf / NaN what they are.
__device__ __forceinline__ uint32_t to_tf32(float x) { return (__float_as_uint(x) + 0x1000u) & 0xFFFFE000u; }
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    uint32_t done;
    do {
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n" : "=r"(done) : "r"(bar), "r"(parity) : "memory");
    } while (!done);
}
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap *map, uint32_t bar, int c0, int c1) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
        ::"r"(dst), "l"((uint64_t)map), "r"(bar), "r"(c0), "r"(c1) : "memory");
}
// Shared-memory matrix descriptor, K-major operand in the canonical 128-byte-swizzle layout (what TMA
// SWIZZLE_128B writes for a box of 32 floats x rows): start >> 4 at bits 0-13, leading offset unused for
// swizzled K-major (1), stride offset = 8 rows x 128 B = 1024 >> 4 at bits 32-45, descriptor version 1
// at bit 46, layout type SWIZZLE_128B = 2 at bits 61-63.
__device__ __forceinline__ uint64_t smem_desc(uint32_t saddr) {
    return (uint64_t)((saddr & 0x3FFFFu) >> 4) | (1ull << 16) | ((uint64_t)(1024 >> 4) << 32) | (1ull << 46) | (2ull << 61);
}
// A operand in tensor memory (lane = row of the 128 x 8 tile, one TF32 value per 32-bit column), B from shared memory
__device__ __forceinline__ void umma_tf32_ts(uint32_t tmem_d, uint32_t tmem_a, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::1.kind::tf32 [%0], [%1], %2, %3, p;\n"
        "}\n" ::"r"(tmem_d), "r"(tmem_a), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void tmem_st_32x16(uint32_t taddr, const uint32_t (&r)[16]) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], "
        "{%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};"
        ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]),
          "r"(r[8]), "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15])
        : "memory");
}
__device__ __forceinline__ void umma_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void tmem_ld_32x32(uint32_t taddr, uint32_t (&r)[32]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
          "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]),
          "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]),
          "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
        : "r"(taddr));
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}

// grid (ceil(m_tiles / TM), ksplit, n_tiles); block 320; dynamic smem kSmemBytes.
// dst: modes [B][n_modes] when ksplit == 1, else partials [ksplit][B][n_modes].
//
// A CTA works on TM = 2 neighbouring m tiles of one K range and frame tile, so that one copy of the slope planes in
// shared memory serves both: per stage 2 x 16 KB of recmat + 32 KB of slope planes instead of 16 + 32.  The kernel is
// bound by what comes out of L2 (every byte TMA delivers to an SM passes through it: 3 bytes per recmat byte with one
// m tile per CTA = 576 MB in 63 us = 9.1 TB/s of the ~12 TB/s the L2 slices deliver; ncu: tensor pipe 60 %, DRAM 40 %,
// the converters waiting for TMA), so the ratio is what counts: now 2 bytes per recmat byte.  (Clusters of two CTAs
// with the slope planes multicast gave nothing: at cluster sizes up to 4 a multicast costs L2 what two loads cost.)
// Tensor memory: two accumulators of 128 columns, and TSLOTS = 2 slots of converted recmat planes (2 m tiles x (32 hi
// + 32 lo) columns each) that the converters fill one stage ahead of the MMA warp.
__global__ void __launch_bounds__(kThreads, 1)
rec_tc_kernel(const __grid_constant__ CUtensorMap mR,
              const __grid_constant__ CUtensorMap mShi, const __grid_constant__ CUtensorMap mSlo,
              float *__restrict__ dst, int n_modes, int B, int nkb, int ksplit, int m_tiles) {
    extern __shared__ uint8_t smem_raw[];
    const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;          // 128-byte swizzle needs 1024-byte tiles
    const uint32_t bars = base + STAGES * kStageBytes;
    // barriers: full[s] at +8 s, empty[s] at +8 (STAGES + s), conv[ts] at +8 (2 STAGES + ts), tfree[ts] at
    // +8 (2 STAGES + TSLOTS + ts), accumulator-ready after them; then the TMEM address
    const uint32_t bar_conv = bars + 8 * (2 * STAGES), bar_tfree = bar_conv + 8 * TSLOTS, bar_acc = bar_tfree + 8 * TSLOTS;
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(smem_raw + (bar_acc + 8 - smem_u32(smem_raw)));
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int m_pair = blockIdx.x, ks = blockIdx.y, n_tile = blockIdx.z;
    const int kb_lo = (int)(((long long)ks * nkb) / ksplit), kb_hi = (int)(((long long)(ks + 1) * nkb) / ksplit);

    if (threadIdx.x == 0) {
        for (int s = 0; s < STAGES; ++s) {
            mbar_init(bars + 8 * s, 1);
            mbar_init(bars + 8 * (STAGES + s), 1);
        }
        for (int ts = 0; ts < TSLOTS; ++ts) {
            mbar_init(bar_conv + 8 * ts, kConvThreads);
            mbar_init(bar_tfree + 8 * ts, 1);
        }
        mbar_init(bar_acc, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 2) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "n"(kTmemCols) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem = *tmem_slot;

    if (warp == 0) {
        if (lane == 0) {                                                  // ---- TMA producer
            int it = 0;
            for (int kb = kb_lo; kb < kb_hi; ++kb, ++it) {
                const int s = it % STAGES;
                const uint32_t full = bars + 8 * s, empty = bars + 8 * (STAGES + s), st = base + s * kStageBytes;
                mbar_wait(empty, ((it / STAGES) & 1) ^ 1);
                mbar_expect_tx(full, kLoadBytes);
#pragma unroll
                for (int t = 0; t < TM; ++t) {                            // raw FP32 recmat; a tile beyond the matrix re-reads the last one
                    const int mt = min(m_pair * TM + t, m_tiles - 1);
                    tma_load_2d(st + t * kTileBytes, &mR, full, kb * BK, mt * BM);
                }
                tma_load_2d(st + TM * kTileBytes, &mShi, full, kb * BK, n_tile * BN);
                tma_load_2d(st + (TM + 1) * kTileBytes, &mSlo, full, kb * BK, n_tile * BN);
            }
        }
    } else if (warp == 1) {
        if (lane == 0) {                                                  // ---- MMA issuer
            const int n_here = min(BN, (B - n_tile * BN + 15) / 16 * 16);
            const uint32_t idesc = idesc_for(n_here);
            int it = 0;
            for (int kb = kb_lo; kb < kb_hi; ++kb, ++it) {
                const int s = it % STAGES, ts = it % TSLOTS;
                const uint32_t conv = bar_conv + 8 * ts, tfree = bar_tfree + 8 * ts, empty = bars + 8 * (STAGES + s);
                const uint32_t st = base + s * kStageBytes;
                mbar_wait(conv, (it / TSLOTS) & 1);                       // TMA landed AND recmat has been split
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
#pragma unroll
                for (int k = 0; k < BK / UK; ++k) {
                    const uint32_t ko = k * UK * 4;                      // 32 bytes along the swizzled row
                    const uint64_t shi = smem_desc(st + TM * kTileBytes + ko), slo = smem_desc(st + (TM + 1) * kTileBytes + ko);
#pragma unroll
                    for (int t = 0; t < TM; ++t) {
                        const uint32_t acc = tmem + (uint32_t)t * 128u;
                        const uint32_t a_hi = tmem + kAccCols + (uint32_t)(ts * TM + t) * 64u, a_lo = a_hi + 32u;
                        umma_tf32_ts(acc, a_lo + k * UK, shi, idesc, (it > 0 || k > 0) ? 1u : 0u);   // small terms first
                        umma_tf32_ts(acc, a_hi + k * UK, slo, idesc, 1u);
                        umma_tf32_ts(acc, a_hi + k * UK, shi, idesc, 1u);
                    }
                }
                umma_commit(empty);                                       // frees the stage when these UMMAs retire
                umma_commit(tfree);                                       // ... and the slot of converted planes
            }
            umma_commit(bar_acc);
        }
    } else {                                                              // ---- warps 2..9: converters, then epilogue
        // A warp may touch the TMEM lanes 32 (warp % 4) .. + 32 only; the two warps of a lane quarter (warp, warp + 4)
        // share its rows: `half` 0 takes the K values 0..15 of a row, `half` 1 the values 16..31.
        const int q = warp & 3, half = (warp - 2) >> 2;
        {
            int it = 0;
            for (int kb = kb_lo; kb < kb_hi; ++kb, ++it) {
                const int s = it % STAGES, ts = it % TSLOTS;
                mbar_wait(bars + 8 * s, (it / STAGES) & 1);               // the stage has landed
                mbar_wait(bar_tfree + 8 * ts, ((it / TSLOTS) & 1) ^ 1);   // the MMAs that read this slot have retired
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                // thread = (row of the tile = TMEM lane 32 q + lane, half); a row's 32 K values are 8 chunks of 16 bytes
                // that TMA's 128-byte swizzle has stored at chunk position c ^ (row % 8)
                const int row = q * 32 + lane;
#pragma unroll
                for (int t = 0; t < TM; ++t) {
                    const uint8_t *tile = smem_raw + (base - smem_u32(smem_raw)) + s * kStageBytes + t * kTileBytes + row * 128;
                    uint32_t hi[16], lo[16];
#pragma unroll
                    for (int c = 0; c < 4; ++c) {
                        const float4 x = *reinterpret_cast<const float4 *>(tile + (((4 * half + c) ^ (row & 7)) << 4));
                        const float xv[4] = {x.x, x.y, x.z, x.w};
#pragma unroll
                        for (int e = 0; e < 4; ++e) {
                            hi[4 * c + e] = to_tf32(xv[e]);
                            lo[4 * c + e] = to_tf32(xv[e] - __uint_as_float(hi[4 * c + e]));
                        }
                    }
                    const uint32_t t_hi = tmem + ((uint32_t)(q * 32) << 16) + kAccCols + (uint32_t)(ts * TM + t) * 64u + (uint32_t)half * 16u;
                    tmem_st_32x16(t_hi, hi);
                    tmem_st_32x16(t_hi + 32u, lo);
                }
                asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
                asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
                mbar_arrive(bar_conv + 8 * ts);
            }
        }
        mbar_wait(bar_acc, 0);
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        float *out = dst + (size_t)ks * B * n_modes;
#pragma unroll
        for (int t = 0; t < TM; ++t) {
            const int m = (m_pair * TM + t) * BM + q * 32 + lane;
            for (int c0 = 32 * half; c0 < BN; c0 += 64) {                // the quarter's two warps alternate over the columns
                const int n0 = n_tile * BN + c0;
                if (n0 >= B) break;                                       // warp-uniform
                uint32_t r[32];
                tmem_ld_32x32(tmem + ((uint32_t)(q * 32) << 16) + (uint32_t)t * 128u + (uint32_t)c0, r);
                if (m < n_modes) {
#pragma unroll
                    for (int j = 0; j < 32; ++j)
                        if (n0 + j < B) out[(size_t)(n0 + j) * n_modes + m] = __uint_as_float(r[j]);
                }
            }
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 2)
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(kTmemCols) : "memory");
}

// x -> hi = tf32(x), lo = tf32(x - hi) (round to nearest, low 13 mantissa bits zero), zero beyond `cols`.
// grid (ceil(ldp / 256), rows)
__global__ void split_tf32_kernel(const float *__restrict__ src, size_t src_pitch, int cols, int ldp,
                                  float *__restrict__ hi, float *__restrict__ lo) {
    const int c = blockIdx.x * blockDim.x + threadIdx.x, r = blockIdx.y;
    if (c >= ldp) return;
    const float x = c < cols ? __ldg(src + (size_t)r * src_pitch + c) : 0.f;
    uint32_t h, l;
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(h) : "f"(x));
    const float rest = x - __uint_as_float(h);
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(l) : "f"(rest));
    hi[(size_t)r * ldp + c] = __uint_as_float(h);
    lo[(size_t)r * ldp + c] = __uint_as_float(l);
}

// out[i] = sum_ks part[ks][i], fixed order
__global__ void splitk_sum_kernel(const float *__restrict__ part, size_t n, int ksplit, float *__restrict__ out) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    float s = 0.f;
    for (int ks = 0; ks < ksplit; ++ks) s += __ldg(part + (size_t)ks * n + i);
    out[i] = s;
}

using EncodeTiledFn = CUresult (*)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                   const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                   CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_tiled_fn() {
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) != cudaSuccess ||
        q != cudaDriverEntryPointSuccess)
        return nullptr;
    return reinterpret_cast<EncodeTiledFn>(fn);
}

// [rows][ldp] FP32 plane, box 32 (K) x 128 (rows), 128-byte swizzle; rows beyond `rows` read as zero
bool make_map(EncodeTiledFn enc, CUtensorMap *map, const float *plane, int rows, int ldp) {
    const cuuint64_t dims[2] = {(cuuint64_t)ldp, (cuuint64_t)rows};
    const cuuint64_t strides[1] = {(cuuint64_t)ldp * sizeof(float)};
    const cuuint32_t box[2] = {(cuuint32_t)BK, (cuuint32_t)BM};
    const cuuint32_t estr[2] = {1, 1};
    return enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<float *>(plane), dims, strides, box, estr,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

int cuda_rc(cudaError_t e) { return e == cudaErrorMemoryAllocation ? PWFS_ENOMEM : PWFS_ECUDA; }

}  // namespace

struct RecTc {
    int device = 0, n_modes = 0, n_slopes = 0, ldp = 0, num_sms = 148;
    EncodeTiledFn enc = nullptr;
    float *d_Shi = nullptr, *d_Slo = nullptr, *d_part = nullptr;
    int b_cap = 0;                  // frames the slope planes / partials are sized for
    int ksplit_env = 0;             // PWFS_REC_KSPLIT (tuning builds only), read once at create; 0 = heuristic
    size_t part_cap = 0;            // floats in d_part
    CUtensorMap mR, mShi, mSlo;
};

int rec_tc_create(RecTc **out, const float *d_R, int n_modes, int n_slopes, int ldk, int device, int num_sms) {
    *out = nullptr;
    RecTc *h = new (std::nothrow) RecTc();
    if (!h) return PWFS_ENOMEM;
    h->device = device; h->n_modes = n_modes; h->n_slopes = n_slopes; h->num_sms = num_sms;
    h->ldp = (n_slopes + BK - 1) / BK * BK;
    h->enc = encode_tiled_fn();
    if (!h->enc) { delete h; return PWFS_EUNSUPPORTED; }
#ifdef PWFS_TUNING   // tuning builds only (libpwfs_tuning.so): K split forced from the environment, read once here
    if (const char *e = std::getenv("PWFS_REC_KSPLIT")) h->ksplit_env = std::max(0, std::atoi(e));
#endif
    // recmat itself is the TMA source: [n_modes][ldk] FP32, ldk % 4 == 0 (16-byte row pitch), zero padded; K blocks
    // beyond ldk are filled with zeros by TMA
    cudaError_t e = cudaFuncSetAttribute(rec_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes);
    if (e != cudaSuccess) { int rc = cuda_rc(e); rec_tc_destroy(h); return rc; }
    if (!make_map(h->enc, &h->mR, d_R, n_modes, ldk)) {
        rec_tc_destroy(h);
        return PWFS_ECUDA;
    }
    *out = h;
    return PWFS_OK;
}

// K split for a batch that fills n_tiles frame tiles (a function of the tile count, not of B itself)
static int rec_tc_ksplit_tiles(const RecTc *h, int n_tiles) {
    const int m_tiles = (h->n_modes + BM - 1) / BM, nkb = h->ldp / BK;
    int ksplit = h->num_sms / ((m_tiles + TM - 1) / TM * n_tiles);
    if (h->ksplit_env > 0) ksplit = h->ksplit_env;
    if (ksplit > nkb / 4) ksplit = nkb / 4;                               // at least 4 K blocks per split
    return ksplit < 1 ? 1 : ksplit;
}

static int rec_tc_ksplit(const RecTc *h, int B) { return rec_tc_ksplit_tiles(h, (B + BN - 1) / BN); }

// floats of split-K partials a batch of n_tiles frame tiles writes
static size_t rec_tc_part_need(const RecTc *h, int n_tiles) {
    const int ksplit = rec_tc_ksplit_tiles(h, n_tiles);
    return ksplit > 1 ? (size_t)ksplit * ((size_t)n_tiles * BN) * h->n_modes : 0;
}

// Makes the slope planes hold B frames and the partials hold part_need floats (allocates; synchronises `st` first
// when it has to replace buffers that may be in use).
static int rec_tc_size(RecTc *h, int B, size_t part_need, cudaStream_t st) {
    if (B <= h->b_cap && part_need <= h->part_cap) return PWFS_OK;
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(st, &cs) == cudaSuccess && cs != cudaStreamCaptureStatusNone) return PWFS_EINVAL;
    if (cudaStreamSynchronize(st) != cudaSuccess) return PWFS_ECUDA;
    if (B > h->b_cap) {
        const int cap = (B + BN - 1) / BN * BN;
        cudaFree(h->d_Shi); cudaFree(h->d_Slo);
        h->d_Shi = h->d_Slo = nullptr; h->b_cap = 0;
        const size_t bytes = (size_t)cap * h->ldp * sizeof(float);
        cudaError_t e = cudaMalloc((void **)&h->d_Shi, bytes);
        if (e == cudaSuccess) e = cudaMalloc((void **)&h->d_Slo, bytes);
        if (e == cudaSuccess) e = cudaMemset(h->d_Shi, 0, bytes);
        if (e == cudaSuccess) e = cudaMemset(h->d_Slo, 0, bytes);
        if (e != cudaSuccess) return cuda_rc(e);
        if (!make_map(h->enc, &h->mShi, h->d_Shi, cap, h->ldp) || !make_map(h->enc, &h->mSlo, h->d_Slo, cap, h->ldp))
            return PWFS_ECUDA;
        h->b_cap = cap;
    }
    if (part_need > h->part_cap) {
        cudaFree(h->d_part);
        h->d_part = nullptr; h->part_cap = 0;
        cudaError_t e = cudaMalloc((void **)&h->d_part, part_need * sizeof(float));
        if (e != cudaSuccess) return cuda_rc(e);
        h->part_cap = part_need;
    }
    return PWFS_OK;
}

// Sizes the slope planes and the split-K partials for every batch of 1..B frames: a smaller batch fills fewer frame
// tiles, is split further along K, and can need MORE partials than B itself (148 x 128 floats per mode for one tile
// against 49 x 384 for three), so the need is the largest over the tile counts up to B's.
int rec_tc_reserve(RecTc *h, int B, cudaStream_t st) {
    size_t part_need = 0;
    for (int nt = 1; nt <= (B + BN - 1) / BN; ++nt) part_need = std::max(part_need, rec_tc_part_need(h, nt));
    return rec_tc_size(h, B, part_need, st);
}

int rec_tc_run(RecTc *h, const float *d_slopes, int B, float *d_modes, cudaStream_t st) {
    const int m_tiles = (h->n_modes + BM - 1) / BM, n_tiles = (B + BN - 1) / BN, nkb = h->ldp / BK;
    const int ksplit = rec_tc_ksplit(h, B);
    if (int rc = rec_tc_size(h, B, rec_tc_part_need(h, n_tiles), st)) return rc;   // no-op once sized (pwfs_rec_reserve)
    split_tf32_kernel<<<dim3((h->ldp + 255) / 256, B), 256, 0, st>>>(d_slopes, (size_t)h->n_slopes, h->n_slopes, h->ldp,
                                                                    h->d_Shi, h->d_Slo);
    rec_tc_kernel<<<dim3((m_tiles + TM - 1) / TM, ksplit, n_tiles), kThreads, kSmemBytes, st>>>(
        h->mR, h->mShi, h->mSlo, ksplit > 1 ? h->d_part : d_modes, h->n_modes, B, nkb, ksplit, m_tiles);
    if (ksplit > 1) {
        const size_t n = (size_t)B * h->n_modes;
        splitk_sum_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(h->d_part, n, ksplit, d_modes);
    }
    return cudaGetLastError() == cudaSuccess ? PWFS_OK : PWFS_ECUDA;
}

void rec_tc_destroy(RecTc *h) {
    if (!h) return;
    cudaFree(h->d_Shi); cudaFree(h->d_Slo); cudaFree(h->d_part);
    delete h;
}
