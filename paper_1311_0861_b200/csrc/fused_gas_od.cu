// Fused hydro step of the gas carrying the overdetermined system (GP_OD contexts; fused_impl.cuh with GP_OVERDET):
// six fields (rho*eps paired with the energy), footprint of 32 x 16 cells, five ring slots so that the 50 planes fit
// in shared memory (200 KB).
#define GP_OVERDET 1
#define GP_NS 5
#define GP_FY 16
#define GP_NDW 12
#define GP_REG_E 80
#define GP_REG_D 56
#define GP_FUSED_NS fgasod
#define GP_FUSED_GAS 1
#include "fused_impl.cuh"
