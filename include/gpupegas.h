/*
 * include/gpupegas.h — C ABI of libgpupegas.so: the B200 (sm_100a) hot path of GPUPEGAS
 * (I. Kulikov, arXiv:1311.0861): one explicit fp64 timestep of the operator-split
 * Godunov + FIIC (fluids-in-cell) scheme on a uniform 3-D Cartesian grid, for a gas and a
 * collisionless component, with an FFT Poisson solve and a CFL reduction.
 *
 * Everything behind these calls runs in hand-written CUDA kernels (plus cuFFT for the
 * transforms).  There is no CPU fallback: without a CUDA device gp_create fails.
 *
 * Conventions
 *   - Every int-returning call returns GP_OK or an error code and never throws; the text of
 *     the last error of the calling thread is available from gp_last_error().
 *   - A field is nx*ny*nz contiguous doubles, x fastest (c = i + nx*(j + ny*k)), interior
 *     cells only: ghost cells never cross the ABI (they are index maps inside the kernels).
 *   - Pointers passed in stay owned by the caller; the library copies.  `*_on_device` says
 *     whether such a pointer is device memory (non-zero) or host memory (0).
 *   - Work is issued asynchronously on the context's stream (default: the legacy default
 *     stream; see gp_set_stream).  Calls that hand a result to the host (gp_get_state to a
 *     host pointer, gp_max_dt with dt != NULL) synchronise that stream.
 *   - Cubic cells only (one h).  nx, ny, nz >= 4.  With a Poisson mode, nx, ny, nz even.
 *     GP_POISSON_ISOLATED needs GP_BC_OUTFLOW on every axis (gp_create fails otherwise).
 *   - One "full timestep" of the metric = gp_max_dt + gp_solve_poisson (if gravity) + gp_step.
 */
#ifndef GPUPEGAS_H
#define GPUPEGAS_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct gp_ctx gp_ctx;   /* opaque; created by gp_create, freed by gp_destroy */

enum { GP_OK = 0, GP_ERR_ARG = 1, GP_ERR_ALLOC = 2, GP_ERR_CUDA = 3, GP_ERR_CUFFT = 4,
       GP_ERR_STATE = 5 /* NaN/Inf, or rho, n, p or Pi_dd <= 0 seen */, GP_ERR_UNSUPPORTED = 6 };

/* components bit mask.  GP_OD: carry the overdetermined system of the paper as well (see below). */
enum { GP_GAS = 1, GP_STARS = 2, GP_OD = 4 };
enum { GP_POISSON_NONE = 0, GP_POISSON_PERIODIC = 1, GP_POISSON_ISOLATED = 2 };
enum { GP_BC_PERIODIC = 0, GP_BC_OUTFLOW = 1 };

/* Conserved fields.  Gas: rho, rho*v (3), rho*E.  Collisionless component
 * (PAPER.md:57, 63): n, n*u (3), n*E_ij (6, symmetric: xx xy xz yy yz zz).  Potential
 * (PAPER.md:186): Phi + Phi0, one field for the summed density.  gp_set_state / gp_get_state take any of these
 * ids (GP_EPS ... GP_PZZ only on a GP_OD context). */
enum { GP_RHO = 0, GP_MX, GP_MY, GP_MZ, GP_E,
       GP_N, GP_NUX, GP_NUY, GP_NUZ, GP_EXX, GP_EXY, GP_EXZ, GP_EYY, GP_EYZ, GP_EZZ,
       GP_PHI, GP_NFIELDS,
       /* Carried fields of the overdetermined system (contexts created with GP_OD only): the internal energy
        * rho*eps of the gas (4th equation) and the velocity-dispersion tensor Pi_ij of the
        * collisionless component (xx xy xz yy yz zz). */
       GP_EPS = GP_NFIELDS, GP_PXX, GP_PXY, GP_PXZ, GP_PYY, GP_PYZ, GP_PZZ, GP_NFIELDS_OD };

typedef struct {
    int nx, ny, nz;      /* interior cells per axis */
    double h;            /* cell size (with h_x = h_y = h_z) */
    int components;      /* GP_GAS | GP_STARS [| GP_OD] */
    int poisson;         /* GP_POISSON_* */
    double G;            /* gravitational constant multiplying the source of PAPER.md:186 */
} gp_grid;

typedef struct { int x, y, z; } gp_bc;   /* GP_BC_* per axis, applied to the hydro fields */

/* Create a context for `grid`, adiabatic index `gamma` and boundary rule `bc`.
 * Allocates nothing large: device storage is taken at the first call that needs it, from the
 * region bound with gp_bind_storage if there is one, else with cudaMalloc.  Returns NULL on
 * failure (bad arguments, no CUDA device). */
gp_ctx* gp_create(const gp_grid* grid, double gamma, const gp_bc* bc);
void gp_destroy(gp_ctx* ctx);

/* Copy one field in / out.  `field` must belong to an enabled component (or be GP_PHI), else
 * GP_ERR_ARG.  Setting GP_PHI also fills its ghost faces by the hydro boundary rule. */
int gp_set_state(gp_ctx* ctx, int field, const double* src, int src_on_device);
int gp_get_state(gp_ctx* ctx, int field, double* dst, int dst_on_device);

/* Phi <- solution of the Poisson equation for (rho + n) of the current state.
 * Periodic mode: PAPER.md:190 (exact inverse of the 27-point Laplacian, zero-mean Phi).
 * Isolated mode: zero-padded (2N)^3 convolution with the -G/r kernel (Hockney & Eastwood); the
 * six ghost faces of Phi are taken from padded indices 2N-1 and N.  The first isolated solve of a
 * context also builds the kernel spectrum, for which it allocates (and frees before returning)
 * temporary device scratch of about 128 bytes per cell with cudaMalloc: GP_ERR_ALLOC if that fails.
 * Any even nx, ny, nz is accepted; power-of-two sizes (nz in [8, 1024] periodic; ny, nz <= 512
 * isolated) take the fused / pruned transforms, other sizes plain cuFFT 3-D plans.
 * With both components and the periodic mode the source rho + n is normally the one the last
 * gp_step wrote; after a gp_set_state it is reassembled from the stored densities.
 * GP_POISSON_NONE: GP_ERR_UNSUPPORTED. */
int gp_solve_poisson(gp_ctx* ctx);

/* CFL reduction: dt = cfl*h / max over cells and axes of (|v_d| + sqrt(gamma p/rho)) and
 * (|u_d| + sqrt(3 Pi_dd/n)) (wave speeds PAPER.md:86, 140).  The result stays on the device
 * for gp_step(ctx, 0).  If `dt` is not NULL the call also copies it to *dt (host pointer),
 * synchronises, and returns GP_ERR_STATE if the state holds NaN/Inf or a non-positive
 * rho, n, p or Pi_dd.  In a GP_OD context p and Pi_dd are those of the CARRIED fields, the ones the stages
 * use: p = (gamma-1) rho*eps and the carried Pi_dd (reading G16); a cell whose total-energy description
 * is unphysical but whose carried fields are positive (gas-vacuum border) is then not an error. */
int gp_max_dt(gp_ctx* ctx, double cfl, double* dt);

/* One timestep: Eulerian stage (face values PAPER.md:112-114 and
 * 170-178, pressure and gravity sources from the stored Phi) then Lagrangian stage (upwind
 * flux-form advection), for every enabled component.  dt > 0: use it; dt <= 0: use the
 * device-resident dt of the last gp_max_dt. */
int gp_step(gp_ctx* ctx, double dt);

/* ---- overdetermined system and correctness check (contexts created with GP_OD) ----
 * Besides rho*E and n*E_ij the scheme carries rho*eps (4th equation) and Pi_ij by their
 * own equations.  In a GP_OD context both stages take the pressure p = (gamma-1) rho*eps and the dispersion tensor
 * from the CARRIED fields; the Eulerian stage also updates them,
 *     (rho eps)* = rho eps - tau (gamma-1) rho eps  sum_d (V_{d+1/2} - V_{d-1/2}) / h,
 *     Pi_ij*     = Pi_ij   - tau sum_k [Pi_jk (u*_i|_{k+1/2} - u*_i|_{k-1/2}) + Pi_ik (u*_j|_{k+1/2} - u*_j|_{k-1/2})] / h
 * with the face values V, u* of PAPER.md:112 and 170-172, and the Lagrangian stage advects them like every other
 * field.  All other GP_OD calls return GP_ERR_UNSUPPORTED on a context created without GP_OD.
 *
 * gp_od_derive: carried fields := what the conserved fields imply (rho eps = rho E - rho v^2/2, PAPER.md:41 last
 *   line; Pi_ij = n E_ij - n u_i u_j).  Call it after setting the conserved fields, unless the
 *   carried fields are set explicitly with gp_set_state(GP_EPS ... GP_PZZ).
 * gp_od_step: one timestep as above; dt as in gp_step.  balance != 0 applies the energy balance (below) to the new
 *   state inside the same kernels.  gp_step on a GP_OD context is gp_od_step(ctx, dt, 1).
 * gp_od_balance: the "energy balance procedure" (PAPER.md:202 only cites it; reading G15 -- this build's
 *   own design), cell by cell on the current state: where rho E - rho v^2/2 > 0 (all three Pi_dd of
 *   n E_ij - n u_i u_j > 0) the total-energy description wins and the carried field is reset from it; elsewhere the
 *   carried field wins: |v| is rescaled, direction kept, so that rho v^2/2 = rho E - rho eps (v := 0 and
 *   rho E := rho eps if even that is not positive), and n E_ij := Pi_ij + n u_i u_j.
 * gp_kappa: out[0] = kappa_gas = sum |rho E - rho eps - rho v^2/2| h^3, out[1] = kappa_bme = sum over the six
 *   components of |n E_ij - Pi_ij - n u_i u_j| h^3 of the CURRENT state (host pointer;
 *   synchronises).  A component that is not enabled reports 0.
 * gp_od_last_kappa: the same two sums for the state the last gp_od_step / gp_step produced BEFORE its balance was
 *   applied, folded by the step kernels at no extra pass (the paper's per-step check); GP_ERR_STATE if no step has
 *   run since the state was last set.  The blocks of the step kernels add their partial sums with one fp64
 *   atomicAdd each, in scheduling order: unlike gp_kappa (fixed-order sum, bit-reproducible) the last digits of
 *   these two numbers may differ from run to run (relative 1e-15 or so); the state itself is deterministic.
 * Stale carried fields: writing a conserved field of a GP_OD context with gp_set_state leaves the carried fields of
 *   that component behind (and fresh storage holds none at all).  Until gp_od_derive has run, or the carried fields
 *   have been set as well, gp_step / gp_od_step, gp_max_dt and gp_od_balance return GP_ERR_STATE instead of
 *   computing with the pressure of some other state. */
int gp_od_derive(gp_ctx* ctx);
int gp_od_step(gp_ctx* ctx, double dt, int balance);
int gp_od_balance(gp_ctx* ctx);
int gp_kappa(gp_ctx* ctx, double* out);
int gp_od_last_kappa(gp_ctx* ctx, double* out);

/* ---- the correctness check for callers who cannot let the library allocate ----
 * gp_kappa needs a context, and a context takes device storage of about twice the state (cudaMalloc at first use,
 * or a region the caller binds).  Some callers have no memory to give and cannot tolerate an allocation: a run
 * whose grids fill the card, a PyTorch process whose caching allocator already holds the free HBM (a cudaMalloc
 * from in here then fails, or starves that allocator later), a multi-stream time loop (cudaMalloc / cudaFree stall
 * the whole device), or a tool that merely holds the fields of some snapshot and wants the two sums.  For them:
 *
 * gp_kappa_noalloc: out_device[0] = kappa_gas, out_device[1] = kappa_bme, the sums defined under gp_kappa, of the
 *   fields the caller passes.  No context; the call never calls cudaMalloc, cudaFree or any allocating library
 *   routine, and copies nothing.
 *   n_cells   number of cells, 1 ... GP_KAPPA_NOALLOC_MAX_CELLS (512^3); more: GP_ERR_ARG (a larger grid can be
 *             summed slab by slab, adding the results).
 *   h         cell size (> 0); the sums are multiplied by h^3.
 *   gas       HOST array of 6 DEVICE pointers, each to n_cells contiguous doubles: rho, rho v_x, rho v_y, rho v_z,
 *             rho E, rho eps; or NULL (kappa_gas = 0).
 *   stars     HOST array of 16 DEVICE pointers: n, n u_x, n u_y, n u_z, n E_ij (xx xy xz yy yz zz), Pi_ij (same
 *             order); or NULL (kappa_bme = 0).  Not both NULL.  The fields are only read and stay the caller's.
 *   out_device  DEVICE pointer to 2 doubles, written by the last kernel of the call.
 *   cuda_stream a cudaStream_t of the current device (NULL: default stream).  The two kernels are issued on it and
 *             the call returns without synchronising; the result is ready when work queued behind it runs.
 *   Scratch: the per-block partial sums sit in a 512 KiB array compiled into the library (one pair of doubles per
 *   4096 cells, which is where the limit comes from).  Every GPU that has loaded the library holds that array
 *   until the process ends.  All calls on a GPU share it: calls issued on ONE stream are safe back to back (each
 *   call rewrites every slot it later reads, so nothing needs to start at zero), but two calls that can overlap on
 *   the GPU -- different streams without an event between them, or two host threads -- race on it and may both
 *   return garbage.  The first call on each device looks up the array's device address (which may make the driver
 *   load the module); make that first call outside any stream capture.  The result is bit-reproducible for given
 *   inputs; it differs from gp_kappa's only by the rounding of a different summation order.
 *   Errors: GP_ERR_ARG as above (also a NULL pointer inside gas / stars), GP_ERR_CUDA if the address look-up or a
 *   launch fails, GP_ERR_UNSUPPORTED for a device ordinal >= 64. */
#define GP_KAPPA_NOALLOC_MAX_CELLS 134217728
int gp_kappa_noalloc(size_t n_cells, double h, const double* const* gas, const double* const* stars,
                     double* out_device, void* cuda_stream);

const char* gp_last_error(void);   /* thread-local static text; never freed by the caller */

/* ---- optional: let the caller (e.g. PyTorch) own the stream and the device memory ---- */
int gp_set_stream(gp_ctx* ctx, void* cuda_stream);          /* a cudaStream_t; NULL = default stream */
size_t gp_storage_bytes(const gp_grid* grid);               /* size of the state + work storage */
/* Hand the context a device region of at least gp_storage_bytes(grid) bytes, 256-byte aligned.
 * Must be called before the first call that touches device state.  The caller keeps ownership
 * and must keep it alive until gp_destroy. */
int gp_bind_storage(gp_ctx* ctx, void* device_ptr, size_t bytes);
int gp_synchronize(gp_ctx* ctx);                            /* wait for the context's stream */
/* Number of kernel launches (own kernels and cuFFT executions counted separately) issued by this
 * context so far; for the bench's gpu_launches claim. */
int gp_launch_counts(gp_ctx* ctx, long long* own_kernels, long long* cufft_execs);

/* ---- optional: per-kernel timing with CUDA events on the context's stream ----
 * gp_timing_enable(ctx, 1) zeroes the totals and brackets every later kernel launch (and cuFFT
 * execution) with an event pair; gp_timing_enable(ctx, 0) stops.  gp_timing_read synchronises
 * the stream and returns, per kernel kind that ran, its name (static string), the summed
 * elapsed milliseconds and the number of launches; at most max_entries entries are written. */
int gp_timing_enable(gp_ctx* ctx, int on);
int gp_timing_read(gp_ctx* ctx, int max_entries, int* n_entries, const char** names, double* total_ms,
                   long long* launches);

/* ---- optional: self test of the device arithmetic helpers ----
 * The hydro kernels replace fp64 divisions and square roots by a reciprocal and a reciprocal
 * square root built from the hardware seed plus one cubically convergent correction.  This call
 * evaluates both on n host-supplied positive normal numbers x (host pointers, n >= 1) so a test
 * can bound their error: rcp[i] ~ 1/x[i], rsqrt_out[i] ~ 1/sqrt(x[i]).  Allocates and frees its
 * own scratch; uses the default stream; synchronises. */
int gp_math_selftest(int n, const double* x, double* rcp, double* rsqrt_out);

/* ---- optional: self test of the fp64 issue rate of the device ----
 * Runs a kernel of independent DFMA chains on every SM of the current device (default stream, synchronises) and
 * returns the achieved fp64 thread-instructions per second (host pointer) and, if ms is not NULL, the best kernel
 * time in milliseconds.  bench.py reports it beside the nominal fp64 peak of its ALU roofline. */
int gp_fp64_rate_selftest(double* thread_inst_per_s, double* ms);

#ifdef __cplusplus
}
#endif
#endif
