// pwfs_launch.cuh -- the kernel configuration of every supported grid size M = 32 R1 and the
// launcher record pwfs_api.cu dispatches through.  launcher_for<R1>() is defined once per R1 in
// pwfs_inst.cu (one translation unit per grid size).
#pragma once
#include "pwfs_kernels.cuh"

namespace pwk {

// R1 = M / 32 of the built grids: every 2/3/5-smooth multiple of 32 from M = 128 to M = 2048
// (M >= 128 keeps at least four register points per lane; 64 is the most a lane's registers hold)
#define PWFS_FOR_EACH_R1(X) X(4) X(5) X(6) X(8) X(9) X(10) X(12) X(15) X(16) X(18) X(20) X(24) X(25) X(27) X(30) X(32) \
    X(36) X(40) X(45) X(48) X(50) X(54) X(60) X(64)

// PassCfg<R1, NB, warps/CTA row pass, warps/CTA column pass, min CTAs/SM row pass, column pass>.  CfgFor is the row
// pass; the column pass takes its NB from CfgForY below.  Row pass (measured on B200, profiles/r2_tuning.md): small
// CTAs -- 4 warps x NB rows = 8 (or 16, 24) rows -- with a register budget that leaves no spills beat 8-warp CTAs
// capped at 128 registers (M = 1024: 3.65 -> 3.20 ms per 100 frames; M = 320: 1.96 -> 1.81; M = 480: 3.53 -> 3.14;
// M = 800: 11.8 -> 11.5): fewer warps wait at each of the two CTA barriers per x-tilt, and the 14-17 spilled registers
// of the 128-register build went through the same LSU queue that limits the kernel.  NB * R1 fills whole rounds of 32
// lanes in the size-32 stage as far as shared memory allows (NB * R1 * 264 bytes per warp + the parked phasor).
template <int R1> struct CfgFor;
template <> struct CfgFor<4>  { using type = PassCfg<4, 8, 4, 4>; };          // M = 128
template <> struct CfgFor<5>  { using type = PassCfg<5, 6, 4, 4>; };          // M = 160
template <> struct CfgFor<6>  { using type = PassCfg<6, 5, 8, 4>; };          // M = 192
template <> struct CfgFor<8>  { using type = PassCfg<8, 4, 4, 4>; };          // M = 256
template <> struct CfgFor<9>  { using type = PassCfg<9, 3, 8, 4>; };          // M = 288
template <> struct CfgFor<10> { using type = PassCfg<10, 6, 4, 4, 2, 1>; };   // M = 320
template <> struct CfgFor<12> { using type = PassCfg<12, 5, 8, 4>; };         // M = 384
template <> struct CfgFor<15> { using type = PassCfg<15, 2, 4, 4, 4, 1>; };   // M = 480
template <> struct CfgFor<16> { using type = PassCfg<16, 2, 4, 4, 4, 1>; };   // M = 512
template <> struct CfgFor<18> { using type = PassCfg<18, 3, 8, 4, 2, 1>; };   // M = 576
template <> struct CfgFor<20> { using type = PassCfg<20, 2, 4, 4, 2, 1>; };   // M = 640
template <> struct CfgFor<24> { using type = PassCfg<24, 2, 4, 4, 2, 1>; };   // M = 768
template <> struct CfgFor<25> { using type = PassCfg<25, 2, 4, 4, 2, 1>; };   // M = 800
template <> struct CfgFor<27> { using type = PassCfg<27, 2, 4, 4, 2, 1>; };   // M = 864
template <> struct CfgFor<30> { using type = PassCfg<30, 2, 4, 4, 2, 1>; };   // M = 960
template <> struct CfgFor<32> { using type = PassCfg<32, 2, 4, 4, 2, 2>; };   // M = 1024
// R1 > 32: the size-32 stage runs in two rounds (the second with R1 - 32 lanes), one CTA per SM in both passes
template <> struct CfgFor<36> { using type = PassCfg<36, 1, 8, 4, 1, 1>; };   // M = 1152
template <> struct CfgFor<40> { using type = PassCfg<40, 1, 8, 4, 1, 1>; };   // M = 1280
template <> struct CfgFor<45> { using type = PassCfg<45, 1, 8, 4, 1, 1>; };   // M = 1440
template <> struct CfgFor<48> { using type = PassCfg<48, 1, 8, 4, 1, 1>; };   // M = 1536
template <> struct CfgFor<50> { using type = PassCfg<50, 1, 8, 4, 1, 1>; };   // M = 1600
template <> struct CfgFor<54> { using type = PassCfg<54, 1, 8, 4, 1, 1>; };   // M = 1728
template <> struct CfgFor<60> { using type = PassCfg<60, 1, 8, 4, 1, 1>; };   // M = 1920
template <> struct CfgFor<64> { using type = PassCfg<64, 1, 8, 4, 1, 1>; };   // M = 2048

// The column pass may batch more transforms per warp than the row pass (whose shared memory also parks the base
// phasor): more of the 32 lanes busy in the size-32 stage.  Default: the same configuration.  (R1 = 25 with NB = 5,
// 125 items, was tried: the exchange buffers then allow only 6 warps per SM and the column pass ran 1.6x slower.)
// YMODE (last argument; measured on B200, profiles/r2_tuning.md): 2 = twiddles kept in registers through the size-32
// stage (left to the compiler, an unrelated source change moved M = 800 between 33.3 and 40.3 ms per 600 frames);
// 1 = T column staged by cp.async, 168 registers, 3 CTAs per SM (M = 1024: 9.74 -> 9.69 ms per 100 frames; M = 320:
// 5.09 -> 5.04; slower on M = 480 and 800); 5 = staged T column AND the twiddles resident in registers for the whole
// kernel, still 168 registers (M = 800: 33.05 -> 31.84; slower on M = 1024: 10.16, and M = 320: 5.16).  R1 > 32 keeps
// the compiler's choice (64 register points per lane already).
template <int R1> struct CfgForY {
    using B = typename CfgFor<R1>::type;
    using type = PassCfg<R1, B::NB, B::WPB_X, B::WPB_Y, B::MINB_X, B::MINB_Y, R1 <= 32 ? 2 : 0>;
};
template <> struct CfgForY<10> { using type = PassCfg<10, 3, 8, 4, 2, 3, 1>; };   // 30 items
template <> struct CfgForY<15> { using type = PassCfg<15, 2, 8, 4, 2, 2, 2>; };   // 30 items, 250 registers, no spill (NB = 4: 60 items, 120 B of spill, 9.86 -> 8.99 ms per 500 frames)
template <> struct CfgForY<16> { using type = PassCfg<16, 2, 8, 4, 2, 1, 2>; };
template <> struct CfgForY<20> { using type = PassCfg<20, 3, 8, 4, 2, 1, 2>; };   // 60 items (was 20 of 32)
template <> struct CfgForY<24> { using type = PassCfg<24, 1, 8, 4, 2, 1, 2>; };
template <> struct CfgForY<25> { using type = PassCfg<25, 1, 8, 4, 2, 3, 5>; };   // staged T + resident twiddles, 12 warps/SM: 33.05 -> 31.84 ms per 600 frames
template <> struct CfgForY<27> { using type = PassCfg<27, 1, 8, 4, 2, 1, 2>; };
template <> struct CfgForY<30> { using type = PassCfg<30, 1, 8, 4, 2, 1, 2>; };
template <> struct CfgForY<32> { using type = PassCfg<32, 1, 8, 4, 2, 3, 1>; };

struct Launcher {
    int R1, NB, WPB_X, WPB_Y, RPC;   // NB, WPB_Y: column pass; WPB_X, RPC: row pass
    size_t smem_x, smem_y;
    const void *xfn, *yfn;
    void (*launch_x)(dim3, cudaStream_t, const DevTables &, const float *, float2 *, int);
    void (*launch_y)(dim3, cudaStream_t, const DevTables &, const float2 *, float *, int);
    // M = 128 only (else nullptr): the whole path in one kernel, pwfs_small.cuh.  grid (K, F)
    const void *sfn = nullptr;
    size_t smem_s = 0;
    void (*launch_s)(dim3, cudaStream_t, const DevTables &, const float *, float *, unsigned *, float *, float *, float) = nullptr;
};

// quarter = the mask shift is exactly M/4 and there is no field stop: kernels with the table-free
// power-of-i mask; otherwise the table-mask kernels
template <int R1> Launcher launcher_for(bool quarter);
#define PWFS_DECL(R) template <> Launcher launcher_for<R>(bool quarter);
PWFS_FOR_EACH_R1(PWFS_DECL)
#undef PWFS_DECL

}  // namespace pwk
