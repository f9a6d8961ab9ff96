// Fused hydro step of the collisionless component carrying the overdetermined system (GP_OD contexts;
// fused_impl.cuh with GP_OVERDET): sixteen fields (Pi_ij as three more pairs).  The ring alone takes 64 planes, so the
// footprint is 32 x 8 cells (95 planes, 190 KB): eight Eulerian warps and four Lagrangian warps (384 threads launched
// at 168 registers, re-split with setmaxnreg).
#ifndef GP_BMEOD_FY
#define GP_BMEOD_FY 8
#define GP_BMEOD_NDW 4
#endif
#ifndef GP_BMEOD_REG_E
#define GP_BMEOD_REG_E 200
#define GP_BMEOD_REG_D 104
#endif
#define GP_OVERDET 1
#define GP_NS 4
#define GP_FY GP_BMEOD_FY
#define GP_NDW GP_BMEOD_NDW
#define GP_REG_E GP_BMEOD_REG_E
#define GP_REG_D GP_BMEOD_REG_D
#ifndef GP_BMEOD_TZREG
#define GP_BMEOD_TZREG 0
#endif
#define GP_TZREG GP_BMEOD_TZREG
#define GP_FUSED_NS fbmeod
#define GP_FUSED_BME 1
#include "fused_impl.cuh"
