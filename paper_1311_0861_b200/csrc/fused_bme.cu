// Fused hydro step of the collisionless component (fused_impl.cuh): footprint of 32 x 12 cells, twelve
// Eulerian warps and eight Lagrangian warps (640 threads, launched at 96 registers each and re-split with
// setmaxnreg: the Eulerian warps carry 20 doubles of state per column).
#ifndef GP_BME_FY
#define GP_BME_FY 12
#define GP_BME_NDW 8
#endif
#ifndef GP_BME_REG_E
#define GP_BME_REG_E 104
#define GP_BME_REG_D 80
#endif
#define GP_NS 4
#define GP_FY GP_BME_FY
#define GP_NDW GP_BME_NDW
#define GP_REG_E GP_BME_REG_E
#define GP_REG_D GP_BME_REG_D
#ifndef GP_BME_TZREG
#define GP_BME_TZREG 0
#endif
#define GP_TZREG GP_BME_TZREG
#define GP_FUSED_NS fbme
#define GP_FUSED_BME 1
#include "fused_impl.cuh"
