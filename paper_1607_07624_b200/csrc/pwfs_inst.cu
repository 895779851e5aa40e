// pwfs_inst.cu -- the row-pass / column-pass kernels of ONE grid size, M = 32 * PWFS_INST_R1, both
// mask variants.  build.py compiles this file once per R1 of PWFS_FOR_EACH_R1 (pwfs_launch.cuh).
#include "pwfs_launch.cuh"
#include "pwfs_small.cuh"

#ifndef PWFS_INST_R1
#define PWFS_INST_R1 4   // a bare `nvcc -c` of this file still gives a valid object
#endif

namespace pwk {
namespace {

// Tuning hook: -DPWFS_TX_NB / _TX_WPB / _TX_MINB (row pass) and -DPWFS_TY_NB / _TY_WPB / _TY_MINB / _TY_MODE (column pass)
// replace the configuration of this translation unit's grid size; used to build experimental variants of the
// library, the shipped build sets none of them.
using C0 = CfgFor<PWFS_INST_R1>::type;
using CY0 = CfgForY<PWFS_INST_R1>::type;
#ifndef PWFS_TX_NB
#define PWFS_TX_NB C0::NB
#endif
#ifndef PWFS_TX_WPB
#define PWFS_TX_WPB C0::WPB_X
#endif
#ifndef PWFS_TX_MINB
#define PWFS_TX_MINB C0::MINB_X
#endif
#ifndef PWFS_TY_NB
#define PWFS_TY_NB CY0::NB
#endif
#ifndef PWFS_TY_WPB
#define PWFS_TY_WPB CY0::WPB_Y
#endif
#ifndef PWFS_TY_MINB
#define PWFS_TY_MINB CY0::MINB_Y
#endif
#ifndef PWFS_TY_MODE
#define PWFS_TY_MODE CY0::YMODE
#endif
using C = PassCfg<PWFS_INST_R1, PWFS_TX_NB, PWFS_TX_WPB, C0::WPB_Y, PWFS_TX_MINB, C0::MINB_Y>;      // row pass
using CY = PassCfg<PWFS_INST_R1, PWFS_TY_NB, CY0::WPB_X, PWFS_TY_WPB, CY0::MINB_X, PWFS_TY_MINB, PWFS_TY_MODE>;   // column pass

template <bool QM>
void launch_x_t(dim3 grid, cudaStream_t st, const DevTables &t, const float *phase, float2 *T, int jsplit) {
    xpass_kernel<C, QM><<<grid, 32 * C::WPB_X, QM ? C::smem_x_q : C::smem_x_t, st>>>(t, phase, T, jsplit);
}
template <bool QM>
void launch_y_t(dim3 grid, cudaStream_t st, const DevTables &t, const float2 *T, float *colbin, int ksplit) {
    ypass_kernel<CY, QM><<<grid, 32 * CY::WPB_Y, QM ? CY::smem_y_q : CY::smem_y_t, st>>>(t, T, colbin, ksplit);
}
template <bool QM>
void launch_s_t(dim3 grid, cudaStream_t st, const DevTables &t, const float *phase, float *part, unsigned *counter,
                float *frames, float *slopes, float scale) {
    small_kernel<QM><<<grid, 256, QM ? SmallCfg::smem_q : SmallCfg::smem_t, st>>>(t, phase, part, counter, frames, slopes, scale);
}
template <bool QM>
Launcher make() {
    Launcher l;
    l.R1 = C::R1; l.NB = CY::NB; l.WPB_X = C::WPB_X; l.WPB_Y = CY::WPB_Y; l.RPC = C::RPC;
    l.smem_x = QM ? C::smem_x_q : C::smem_x_t; l.smem_y = QM ? CY::smem_y_q : CY::smem_y_t;
    l.xfn = (const void *)xpass_kernel<C, QM>;
    l.yfn = (const void *)ypass_kernel<CY, QM>;
    l.launch_x = launch_x_t<QM>;
    l.launch_y = launch_y_t<QM>;
#if PWFS_INST_R1 == 4
    l.sfn = (const void *)small_kernel<QM>;
    l.smem_s = QM ? SmallCfg::smem_q : SmallCfg::smem_t;
    l.launch_s = launch_s_t<QM>;
#endif
    return l;
}

}  // namespace

template <>
Launcher launcher_for<PWFS_INST_R1>(bool quarter) { return quarter ? make<true>() : make<false>(); }

}  // namespace pwk
