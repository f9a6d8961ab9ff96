/*
 * oracle/oracle.h — C ABI of the CPU oracle (TEST INFRASTRUCTURE ONLY).
 *
 * A plain, slow, fp64 CPU implementation of one explicit timestep of the
 * operator-split Godunov + FIIC scheme of GPUPEGAS (Kulikov, arXiv:1311.0861),
 * written from the paper with the readings listed in DESIGN.md.
 * It shares no code, header, table or helper with the CUDA path under
 * paper_1311_0861_b200/csrc/.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may load this library.
 *
 * Arrays handed across this ABI are host pointers to nx*ny*nz contiguous
 * doubles, x fastest (c = i + nx*(j + ny*k)), interior cells only.
 */
#ifndef GPUPEGAS_ORACLE_H
#define GPUPEGAS_ORACLE_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct orc_ctx orc_ctx;

enum { ORC_OK = 0, ORC_ERR_ARG = 1, ORC_ERR_ALLOC = 2, ORC_ERR_STATE = 5, ORC_ERR_UNSUPPORTED = 6 };
enum { ORC_GAS = 1, ORC_STARS = 2 };
enum { ORC_POISSON_NONE = 0, ORC_POISSON_PERIODIC = 1, ORC_POISSON_ISOLATED = 2 };
enum { ORC_BC_PERIODIC = 0, ORC_BC_OUTFLOW = 1 };
/* field order: gas rho, rho*v (3), rho*E; collisionless
 * n, n*u (3), nE_xx, nE_xy, nE_xz, nE_yy, nE_yz, nE_zz; potential Phi+Phi0. */
enum { ORC_RHO = 0, ORC_MX, ORC_MY, ORC_MZ, ORC_E,
       ORC_N, ORC_NUX, ORC_NUY, ORC_NUZ, ORC_EXX, ORC_EXY, ORC_EXZ, ORC_EYY, ORC_EYZ, ORC_EZZ,
       ORC_PHI, ORC_NFIELDS,
       /* carried fields of the overdetermined system (orc_od_*): rho*eps, Pi_ij */
       ORC_EPS = ORC_NFIELDS, ORC_PXX, ORC_PXY, ORC_PXZ, ORC_PYY, ORC_PYZ, ORC_PZZ };

orc_ctx* orc_create(int nx, int ny, int nz, double h, int components, int poisson, double G,
                    double gamma, int bcx, int bcy, int bcz);
void orc_destroy(orc_ctx*);
void orc_set_threads(int nthreads);          /* OpenMP threads used by the outer loops */
int  orc_get_threads(void);

int orc_set_field(orc_ctx*, int field, const double* src);
int orc_get_field(orc_ctx*, int field, double* dst);
int orc_get_star_field(orc_ctx*, int field, double* dst);   /* U* left by the last Eulerian stage */

int orc_eulerian(orc_ctx*, double dt);         /* S1 + S2: U^n -> U*                         */
int orc_lagrangian(orc_ctx*, double dt);       /* ghost fill of U* + S3: U* -> U^{n+1}       */
int orc_lagrangian_only(orc_ctx*, double dt);  /* U* := U^n, then orc_lagrangian (stage pin) */
int orc_step(orc_ctx*, double dt);             /* orc_eulerian then orc_lagrangian           */
int orc_max_dt(orc_ctx*, double cfl, double* dt);
int orc_solve_poisson(orc_ctx*);
/* Phi including its one-cell ghost ring, (nx+2)(ny+2)(nz+2) doubles, x fastest. */
int orc_get_phi_padded(orc_ctx*, double* dst);

/* ---- overdetermined system and correctness check ----
 * orc_od_enable allocates rho*eps and Pi_ij and derives them from the current conserved state; afterwards
 * orc_set_field / orc_get_field / orc_get_star_field accept ORC_EPS and ORC_PXX..ORC_PZZ.  The orc_od_* stages take
 * the pressure and the dispersion tensor from the CARRIED fields and update them by their own equations.
 * orc_kappa: out[0] = kappa_gas, out[1] = kappa_bme.  orc_od_balance is the build's own reading
 * of the "energy balance procedure" the paper only cites (G15). */
int orc_od_enable(orc_ctx*);
int orc_od_eulerian(orc_ctx*, double dt);
int orc_od_lagrangian(orc_ctx*, double dt);
int orc_od_lagrangian_only(orc_ctx*, double dt);
int orc_od_step(orc_ctx*, double dt, int balance);
int orc_od_balance(orc_ctx*);
int orc_kappa(orc_ctx*, double* out);

/* ---- stateless pieces, exported so tests can pin them one by one ---- */
/* PAPER.md:112,114 */
void orc_gas_face(double gamma, double rhoL, double vL, double pL, double rhoR, double vR, double pR,
                  double* V, double* P);
/* PAPER.md:170-178 for a face normal to axis d; in: n, u[3], Pi[6] (xx,xy,xz,yy,yz,zz) of L and R;
 * out: ustar[3] (x,y,z) and Pid[3] = Pi*_{x d}, Pi*_{y d}, Pi*_{z d}. */
void orc_bme_face(int d, double nL, const double* uL, const double* PiL,
                  double nR, const double* uR, const double* PiR, double* ustar, double* Pid);
/* in-place complex radix-2 FFT of length n (power of two); sign -1 forward, +1 inverse (unscaled) */
int orc_fft1d(double* re, double* im, int n, int sign);
/* O(N^2) direct summation of the isolated potential (reading G3): phi over the index box
 * [lo, hi) per axis (may reach outside the grid, e.g. lo=-1, hi=n+1 for the ghost ring). */
int orc_poisson_direct(int nx, int ny, int nz, double h, double G, const double* dens,
                       int lo_x, int hi_x, int lo_y, int hi_y, int lo_z, int hi_z, double* phi);
double orc_kernel_self(void);   /* K(0)*h: potential at the centre of a uniform unit cube of unit mass */

#ifdef __cplusplus
}
#endif
#endif
