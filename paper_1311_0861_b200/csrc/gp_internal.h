// Internal declarations shared by the translation units of libgpupegas.so (CUDA path only;
// nothing here is seen by oracle/).
#pragma once

#include <cuda.h>
#include <cuda_runtime.h>
#include <cufft.h>

#include <cstddef>
#include <cstdio>

#include "../../include/gpupegas.h"

namespace gp {

constexpr int NGAS = 5;
constexpr int NBME = 10;
constexpr int NHYD = NGAS + NBME;
// Carried fields of the overdetermined system (GP_OD; PAPER.md:41 4th equation): rho*eps, Pi_ij (6).
// Internal field index = public id - 1 (the public enum has GP_PHI between the two groups).
constexpr int NODG = 1, NODB = 6;
constexpr int F_EPS = NHYD, F_PI = NHYD + 1;
constexpr int NALL = NHYD + NODG + NODB;
inline int field_index(int public_id) { return public_id < NHYD ? public_id : public_id - 1; }
// The state lives in HBM as arrays of field PAIRS, one double2 per cell: gas (rho,m_x) (m_y,m_z),
// collisionless (n,nu_x) (nu_y,nu_z) (nE_xx,nE_xy) (nE_xz,nE_yy) (nE_yz,nE_zz), so that the fused
// kernels stage and store 16 bytes per access straight into their paired shared-memory layout.
// U[f] of a paired field points at its member of the pair and consecutive cells are BSTR doubles
// apart.  The gas energy and Phi are plain arrays (stride 1) -- except in a GP_OD context, where the energy
// is paired with the carried internal energy, (rho*E, rho*eps), and the carried Pi_ij form three more pairs
// (Pi_xx,Pi_xy) (Pi_xz,Pi_yy) (Pi_yz,Pi_zz).  Indices below are internal (field_index).
constexpr int BSTR = 2;
constexpr int NGASP = 4;          // gas fields 0..3 are always paired
inline bool field_paired(int f, bool od) { return f < NGASP || (f >= NGAS && f < NHYD) || (od && (f == NGAS - 1 || f >= NHYD)); }
// the first member of the pair field f belongs to
inline int pair_base(int f) {
    if (f == NGAS - 1 || f == F_EPS) return NGAS - 1;
    if (f > F_EPS) return F_PI + ((f - F_PI) & ~1);
    return f < NGAS ? (f & ~1) : NGAS + ((f - NGAS) & ~1);
}

// Grid geometry handed to kernels by value.
struct Geo {
    int nx, ny, nz;
    int bcx, bcy, bcz;
};

// Field pointer bundles (kernel arguments).
template <int NF>
struct Fields {
    double* p[NF];
};
template <int NF>
struct ConstFields {
    const double* p[NF];
};

// Phi lives in an array padded by TWO ghost layers per side: cell (i,j,k), i in [-2, nx+1] etc., sits at
// p[(i+2) + pitch*((j+2) + py*(k+2))], pitch >= nx+4 (phi_pitch below), py = ny+4.
// Layer 1 holds the ghost values of the Poisson mode (periodic solve: wrapped; isolated solve: the padded
// convolution at indices -1 and n; user-set Phi: the hydro rule per axis); layer 2, edges and corners are
// index maps of the same rule (wrap, or clamp for the isolated solve) and are only ever read for the U* of
// periodic ghost cells.  The fused kernels therefore stage Phi rows without any case analysis.
struct PhiPad {
    const double* p;
    int pitch, py;
};
// The array is laid out so that the interior rows (the rows the inverse transform writes and the kernels read most)
// start on 128-byte boundaries: the first ghost column sits PHI_XOFF - 2 doubles into a 256-byte aligned allocation,
// the pitch is a multiple of 16 doubles.  gp_ctx::phip points at the first ghost column.
constexpr int PHI_XOFF = 16;
inline int phi_pitch(int nx) { return (nx + PHI_XOFF + 2 + 15) & ~15; }
inline size_t phi_pad_elems(int nx, int ny, int nz) { return (size_t)phi_pitch(nx) * (ny + 4) * (nz + 4) + PHI_XOFF; }

void set_error(const char* fmt, ...);

// Kernels (and cuFFT executions) that can be timed one by one with CUDA events.
enum KernelId { K_CFL = 0, K_SOURCE, K_FFT_FWD, K_GREEN, K_FFT_INV, K_PHI_GHOST, K_PAD_SOURCE, K_MUL_KERNEL, K_EXTRACT,
                K_FUSED_GAS, K_FUSED_BME, K_ZPASS, K_ISO_YFWD, K_ISO_ZFUSED, K_ISO_YINV, K_OD_AUX, K_NUM };

struct Timing {
    bool on = false;
    cudaEvent_t* ev = nullptr;   // pairs: ev[2*i] start, ev[2*i+1] stop
    int* kid = nullptr;
    size_t cap = 0, used = 0;
    double ms[K_NUM] = {};
    long long cnt[K_NUM] = {};
};

}  // namespace gp

namespace gp {
// Tensor maps of one fused kernel, kept per context: nothing in them changes from step to step except the base
// addresses, which alternate between the two halves of the double buffer, so two sets cover every launch.
constexpr int TM_MAX = 9;      // 8 pair maps of the 16-field collisionless kernel + Phi
struct TmCache {
    const void* key_u[2];      // U[first field] the set was encoded for (null: empty)
    const void* key_phi[2];
    int ok[2];                 // TMA can describe the grid (else the kernel stages cell by cell)
    int next;                  // set to overwrite next
    alignas(64) CUtensorMap tm[2][TM_MAX];
};
}  // namespace gp

struct gp_ctx {
    gp_grid g;
    double gamma;
    gp_bc bc;
    cudaStream_t stream;
    size_t N;

    // storage
    char* base;
    size_t bytes;
    bool owns;
    bool ready;
    bool od;                // GP_OD: the overdetermined system is carried (fields NHYD.. exist, the energy is paired)
    int estr;               // stride of the gas energy array in doubles (1, or BSTR with GP_OD)
    double* U[gp::NALL];    // state U^n (internal field index)
    double* Us[gp::NALL];   // target of the fused step (U^{n+1}); swapped with U after every step
    double* phip;                   // Phi, padded by two ghost layers (PhiPad above)
    double* d_dt;                   // [0] = dt of the last gp_max_dt
    unsigned long long* d_smax;     // bit pattern of the running max signal speed
    int* d_flag;                    // != 0: bad state seen by the CFL reduction
    unsigned long long* d_smax_next;   // max signal speed of U^{n+1}, folded by the fused step kernels
    int* d_flag_next;
    double* d_kappa;                // GP_OD: [0..1] kappa_gas, kappa_bme folded by the last step (before its balance), [2..3] of gp_kappa
    bool kappa_cached;
    unsigned od_stale;              // GP_OD: bit (f - F_EPS) set = carried field f has not followed the conserved fields
                                    // (fresh storage, or a conserved field written since); see api.cu
    bool cfl_cached;                // d_smax_next / d_flag_next describe the current state

    // Poisson
    bool fft_ready;
    cufftHandle plan_fwd, plan_inv;
    cufftDoubleComplex* spec;       // half-spectrum work array
    double* padded;                 // isolated: (2nx)(2ny)(2nz) real array
    double* kspec;                  // isolated: real spectrum of the 1/r kernel
    double* tabx; double* taby; double* tabz;   // periodic: 1 - (2/3) sin^2(pi k/N) per axis
    bool isofast;                   // isolated: pruned transforms of isofft.cu (else full (2N)^3 cuFFT plans)
    double* isoA;                   // isolated, pruned: x spectra of the data lines / of the kept lines
    double* itwy; double* itwz;     // isolated, pruned: exp(-2 pi i k/2ny), exp(-2 pi i k/2nz)
    double* ztw;                    // periodic, fused z pass: exp(-2 pi i k/nz), nz complex values
    bool zfused;                    // periodic: 2-D batched cuFFT plans + the fused z pass (zpass.cu)
    double* src;                    // periodic, gas + stars: rho + n assembled here (by the fused step or k_source)
    bool src_cached;                // src holds rho + n of the current state (written by the fused step)

    gp::TmCache* tmc[2];            // tensor-map sets of the gas / collisionless fused kernel (fused_impl.cuh)
    long long n_own, n_fft;
    gp::Timing* tim;
};

namespace gp {

// api.cu: bracket one launch with events when timing is on
void tic(gp_ctx* c, int kid);
void toc(gp_ctx* c);

// hydro.cu
int launch_cfl(gp_ctx* c, double cfl);
int launch_cfl_from_cache(gp_ctx* c, double cfl);
int launch_cfl_reset_next(gp_ctx* c);
// fill the ghost layers of Phi by wrap (GP_BC_PERIODIC) or clamp (GP_BC_OUTFLOW) per axis; keep_faces: leave the
// six layer-1 faces as they are (the isolated solve has written them)
int launch_phi_ghost_bc(gp_ctx* c, int bcx, int bcy, int bcz, bool keep_faces = false);
inline PhiPad phipad_of(const gp_ctx* c) { return PhiPad{c->phip, phi_pitch(c->g.nx), c->g.ny + 4}; }
inline double* phi_interior(const gp_ctx* c) {      // address of cell (0,0,0)
    return c->phip + 2 + (size_t)phi_pitch(c->g.nx) * (2 + (size_t)(c->g.ny + 4) * 2);
}
// dst[i * dstride] = src[i * sstride], i < n (field copies between the plain and the paired layout)
int launch_strided_copy(gp_ctx* c, double* dst, int dstride, const double* src, int sstride, size_t n);

// fused_gas.cu, fused_bme.cu (fused_impl.cuh)
// src_out != nullptr: also write rho + n of the new state there (src_in = the new n, or nullptr)
int launch_fused_gas(gp_ctx* c, double dt, const double* d_dt, const double* src_in, double* src_out);
int launch_fused_bme(gp_ctx* c, double dt, const double* d_dt);
// fused_gas_od.cu, fused_bme_od.cu: the same kernels carrying the overdetermined system (GP_OD)
int launch_fused_gas_od(gp_ctx* c, double dt, const double* d_dt, const double* src_in, double* src_out, int balance);
int launch_fused_bme_od(gp_ctx* c, double dt, const double* d_dt, int balance);

// od.cu: cell-local passes of the overdetermined system
int launch_od_derive(gp_ctx* c);
int launch_od_balance(gp_ctx* c);
int launch_od_kappa(gp_ctx* c, double* d_out);
int math_selftest(int n, const double* x, double* rcp, double* rsq);

// selftest.cu
int fp64_rate_selftest(double* thread_inst_per_s, double* ms_out);

// poisson.cu
int poisson_setup(gp_ctx* c);
void poisson_teardown(gp_ctx* c);
int poisson_solve(gp_ctx* c);
size_t poisson_storage_bytes(const gp_grid* g);

// isofft.cu
bool iso_pruned_supported(const gp_grid* g);
size_t iso_pruned_storage_bytes(const gp_grid* g);
int iso_pruned_setup(gp_ctx* c);
int iso_pruned_solve(gp_ctx* c);

// zpass.cu
bool zpass_supported(int nz);
int launch_zpass(gp_ctx* c, double coef6);

}  // namespace gp

#define GP_CUDA(call)                                                                          \
    do {                                                                                       \
        cudaError_t e_ = (call);                                                               \
        if (e_ != cudaSuccess) {                                                               \
            gp::set_error("%s:%d: %s: %s", __FILE__, __LINE__, #call, cudaGetErrorString(e_)); \
            return GP_ERR_CUDA;                                                                \
        }                                                                                      \
    } while (0)

#define GP_CUFFT(call)                                                             \
    do {                                                                           \
        cufftResult r_ = (call);                                                   \
        if (r_ != CUFFT_SUCCESS) {                                                 \
            gp::set_error("%s:%d: %s: cufft error %d", __FILE__, __LINE__, #call, (int)r_); \
            return GP_ERR_CUFFT;                                                   \
        }                                                                          \
    } while (0)
