// Fused hydro step of the gas (fused_impl.cuh): footprint of 32 x 16 cells, sixteen Eulerian warps and four
// Lagrangian warps (640 threads, 96 registers each).
#define GP_FY 16
#define GP_FUSED_NS fgas
#define GP_FUSED_GAS 1
#include "fused_impl.cuh"
