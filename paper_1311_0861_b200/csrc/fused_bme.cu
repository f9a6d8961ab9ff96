// Fused hydro step of the collisionless component (fused_impl.cuh): footprint of 32 x 12 threads,
// which leaves 168 registers per thread (no spills; measured 4 % faster than 32 x 16 at 128 with
// spills) and room to run both face solvers of stage B in one basic block (another 1.5 %).
#define GP_FY 12
#define GP_BME_MERGE 1
#define GP_FUSED_NS fbme
#define GP_FUSED_BME 1
#include "fused_impl.cuh"
