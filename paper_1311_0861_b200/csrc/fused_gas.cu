// Fused hydro step of the gas (fused_impl.cuh): footprint of 32 x 16 cells, eight Eulerian warps with two adjacent
// footprint rows per thread and twelve single-row Lagrangian warps (640 threads launched at 96 registers each,
// re-split with setmaxnreg to 128 / 64: nothing spills).
#ifndef GP_GAS_FY
#define GP_GAS_FY 16
#define GP_GAS_NDW 12
#endif
#ifndef GP_GAS_REG_E
#if defined(GP_GAS_EROWS) && GP_GAS_EROWS == 1
#define GP_GAS_REG_E 80
#define GP_GAS_REG_D 56
#else
#define GP_GAS_REG_E 128
#define GP_GAS_REG_D 64
#endif
#endif
#ifndef GP_GAS_NS
#define GP_GAS_NS 6
#endif
#define GP_NS GP_GAS_NS
#define GP_FY GP_GAS_FY
#define GP_NDW GP_GAS_NDW
#define GP_REG_E GP_GAS_REG_E
#define GP_REG_D GP_GAS_REG_D
// w*_x, w*_y of the last two planes stay in registers for the z-averaged face-velocity plane: 5.87 -> 5.54 ms
#ifndef GP_GAS_TZREG
#define GP_GAS_TZREG 1
#endif
#define GP_TZREG GP_GAS_TZREG
// stage E publishes the primitives of the next plane before its z face solve: 5.53 -> 5.43 ms
#ifndef GP_GAS_EARLYPUB
#define GP_GAS_EARLYPUB 1
#endif
#define GP_EARLYPUB GP_GAS_EARLYPUB
// two footprint rows per Eulerian thread: the y face between them stays in registers, half as many row hand-offs
// (5.46 -> 5.20 ms; one row per thread with 16 + 12 warps and 80 / 56 registers: -DGP_GAS_EROWS=1)
#ifndef GP_GAS_EROWS
#define GP_GAS_EROWS 2
#endif
#define GP_EROWS GP_GAS_EROWS
#define GP_FUSED_NS fgas
#define GP_FUSED_GAS 1
#include "fused_impl.cuh"
