// Fused hydro step of the collisionless component (fused_impl.cuh): footprint of 32 x 12 cells, twelve
// Eulerian warps and four Lagrangian warps (512 threads, launched at 128 registers each and re-split with
// setmaxnreg: the Eulerian warps carry 20 doubles of state per column and both face solvers of stage B in
// one basic block).
#define GP_FY 12
#ifndef GP_REG_E
#define GP_REG_E 136
#define GP_REG_D 96
#endif
#define GP_FUSED_NS fbme
#define GP_FUSED_BME 1
#include "fused_impl.cuh"
