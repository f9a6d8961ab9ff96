// Fused hydro step of the gas carrying the overdetermined system (GP_OD contexts; fused_impl.cuh with GP_OVERDET):
// six fields (rho*eps paired with the energy).  Footprint of 32 x 12 cells, twelve Eulerian and eight Lagrangian warps
// (640 threads launched at 96 registers, re-split 104 / 80: nothing spills), four ring slots, 41 planes = 123 KB.
// Measured at 512^3: 7.0 ms; the 32 x 16 footprint of the plain gas kernel needs 200 KB here (five slots), spills at
// 72 registers and leaves the spills almost no L1: 12.3 ms.
#ifndef GP_GASOD_FY
#define GP_GASOD_FY 12
#define GP_GASOD_NDW 8
#define GP_GASOD_NS 4
#endif
#ifndef GP_GASOD_REG_E
#define GP_GASOD_REG_E 104
#define GP_GASOD_REG_D 80
#endif
#define GP_OVERDET 1
#define GP_NS GP_GASOD_NS
#define GP_FY GP_GASOD_FY
#define GP_NDW GP_GASOD_NDW
#define GP_REG_E GP_GASOD_REG_E
#define GP_REG_D GP_GASOD_REG_D
#ifndef GP_GASOD_TZREG
#define GP_GASOD_TZREG 0
#endif
#define GP_TZREG GP_GASOD_TZREG
#ifndef GP_GASOD_EROWS
#define GP_GASOD_EROWS 1
#endif
#define GP_EROWS GP_GASOD_EROWS
#define GP_FUSED_NS fgasod
#define GP_FUSED_GAS 1
#include "fused_impl.cuh"
