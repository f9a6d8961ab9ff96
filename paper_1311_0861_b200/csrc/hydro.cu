// Hydro kernels of libgpupegas.so: Eulerian stage, Lagrangian
// stage, CFL reduction, Phi ghost faces.  fp64 throughout.
//
// Ghost cells are index maps: a neighbour index outside the grid is wrapped (periodic) or
// clamped (outflow) per axis, which equals filling one ghost layer axis by axis (edges and
// corners included).  U* ghosts are copies of the nearest interior U* (outflow) because the
// Lagrangian kernel reads the stored interior U* through the same map.
#include "gp_internal.h"

namespace gp {

__device__ __forceinline__ int map_index(int i, int n, int bc) {
    if (bc == GP_BC_PERIODIC) {
        if (i < 0) i += n;
        else if (i >= n) i -= n;
    } else {
        i = i < 0 ? 0 : (i >= n ? n - 1 : i);
    }
    return i;
}

__device__ __forceinline__ size_t cell(const Geo& g, int i, int j, int k) {
    return (size_t)i + (size_t)g.nx * ((size_t)j + (size_t)g.ny * (size_t)k);
}

// Centred difference of Phi (reading G5) using the ghost faces at the grid boundary.
__device__ __forceinline__ void grad_phi(const Geo& g, const Phi& P, int i, int j, int k, double inv2h, double gr[3]) {
    const size_t c = cell(g, i, j, k);
    const double xm = i > 0 ? P.c[c - 1] : P.gx0[j + (size_t)g.ny * k];
    const double xp = i < g.nx - 1 ? P.c[c + 1] : P.gx1[j + (size_t)g.ny * k];
    const double ym = j > 0 ? P.c[c - g.nx] : P.gy0[i + (size_t)g.nx * k];
    const double yp = j < g.ny - 1 ? P.c[c + g.nx] : P.gy1[i + (size_t)g.nx * k];
    const size_t sz = (size_t)g.nx * g.ny;
    const double zm = k > 0 ? P.c[c - sz] : P.gz0[i + (size_t)g.nx * j];
    const double zp = k < g.nz - 1 ? P.c[c + sz] : P.gz1[i + (size_t)g.nx * j];
    gr[0] = (xp - xm) * inv2h;
    gr[1] = (yp - ym) * inv2h;
    gr[2] = (zp - zm) * inv2h;
}

// --------------------------------------------------------------------------------------------
// Gas
// --------------------------------------------------------------------------------------------
struct GasPrim { double rho, v[3], p; };

__device__ __forceinline__ GasPrim gas_prim(const ConstFields<NGAS>& U, size_t c, double gm1) {
    GasPrim w;
    w.rho = U.p[0][c];
    const double ir = 1.0 / w.rho;
    w.v[0] = U.p[1][c] * ir;
    w.v[1] = U.p[2][c] * ir;
    w.v[2] = U.p[3][c] * ir;
    w.p = gm1 * (U.p[4][c] - 0.5 * w.rho * (w.v[0] * w.v[0] + w.v[1] * w.v[1] + w.v[2] * w.v[2]));
    return w;
}

// PAPER.md:112, 114
__device__ __forceinline__ void gas_face(double gamma, double rl, double vl, double pl, double rr, double vr, double pr,
                                         double& V, double& P) {
    const double Z = sqrt(rl * rr * gamma * (pl + pr) / (rl + rr));
    V = 0.5 * (vl + vr) + 0.5 * (pl - pr) / Z;
    P = 0.5 * (pl + pr) + 0.5 * (vl - vr) * Z;
}

__global__ void __launch_bounds__(256)
k_eulerian_gas(Geo g, ConstFields<NGAS> U, Fields<NGAS> Us, Fields<3> W, Phi phi, double gamma, double h,
               double dt_val, const double* __restrict__ dt_ptr) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = blockIdx.z * blockDim.z + threadIdx.z;
    if (i >= g.nx || j >= g.ny || k >= g.nz) return;
    const double tau = dt_ptr ? *dt_ptr : dt_val;
    const double gm1 = gamma - 1.0;
    const size_t c = cell(g, i, j, k);
    const GasPrim w0 = gas_prim(U, c, gm1);
    double gr[3];
    grad_phi(g, phi, i, j, k, 0.5 / h, gr);

    const int n[3] = {g.nx, g.ny, g.nz};
    const int bc[3] = {g.bcx, g.bcy, g.bcz};
    const int ijk[3] = {i, j, k};
    double dP[3], dPV = 0.0;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        int a[3] = {i, j, k};
        a[d] = map_index(ijk[d] - 1, n[d], bc[d]);
        const GasPrim wm = gas_prim(U, cell(g, a[0], a[1], a[2]), gm1);
        a[d] = map_index(ijk[d] + 1, n[d], bc[d]);
        const GasPrim wp = gas_prim(U, cell(g, a[0], a[1], a[2]), gm1);
        double Vm, Pm, Vp, Pp;
        gas_face(gamma, wm.rho, wm.v[d], wm.p, w0.rho, w0.v[d], w0.p, Vm, Pm);
        gas_face(gamma, w0.rho, w0.v[d], w0.p, wp.rho, wp.v[d], wp.p, Vp, Pp);
        dP[d] = Pp - Pm;
        dPV += Pp * Vp - Pm * Vm;
    }
    const double th = tau / h;
    Us.p[0][c] = w0.rho;
    double work = 0.0;
    const double ir = 1.0 / w0.rho;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const double m = U.p[1 + d][c];
        const double ms = m - th * dP[d] - tau * w0.rho * gr[d];
        Us.p[1 + d][c] = ms;
        W.p[d][c] = ms * ir;
        work += (m - 0.5 * tau * w0.rho * gr[d]) * gr[d];
    }
    Us.p[4][c] = U.p[4][c] - th * dPV - tau * work;
}

// --------------------------------------------------------------------------------------------
// Collisionless component (Boltzmann moment equations)
// --------------------------------------------------------------------------------------------
// sym(i,j) -> index in (xx,xy,xz,yy,yz,zz)
__device__ __forceinline__ constexpr int sym(int i, int j) {
    return i == 0 ? j : (j == 0 ? i : (i == 1 ? (j == 1 ? 3 : 4) : (j == 1 ? 4 : 5)));
}

// What a d-face needs from a cell: n, u[3], Pi_dd, Pi_dt1, Pi_dt2 -> Pd[3] = Pi_{x d}, Pi_{y d}, Pi_{z d}.
struct BmeHalf { double n, u[3], Pd[3]; };

template <int D>
__device__ __forceinline__ BmeHalf bme_half(const ConstFields<NBME>& U, size_t c) {
    BmeHalf w;
    w.n = U.p[0][c];
    const double in = 1.0 / w.n;
#pragma unroll
    for (int a = 0; a < 3; ++a) w.u[a] = U.p[1 + a][c] * in;
#pragma unroll
    for (int a = 0; a < 3; ++a) w.Pd[a] = U.p[4 + sym(a, D)][c] - w.n * w.u[a] * w.u[D];
    return w;
}

// PAPER.md:170-178 for a face normal to axis D, bracketed parameters averaged:
// harmonic mean of n, arithmetic means of Pi_dd and Pi_dt.  us[3] = u*, Ps[3] = Pi*_{. D}.
template <int D>
__device__ __forceinline__ void bme_face(const BmeHalf& L, const BmeHalf& R, double us[3], double Ps[3]) {
    const double s3 = 1.7320508075688772935;
    const double nb = 2.0 * L.n * R.n / (L.n + R.n);
    const double a = 0.5 * (L.Pd[D] + R.Pd[D]);
    const double Z1 = sqrt(nb * a);
    const double Z3 = s3 * Z1;
    const double dPdd = 0.5 * (L.Pd[D] - R.Pd[D]);
    const double dud = 0.5 * (L.u[D] - R.u[D]);
    us[D] = 0.5 * (L.u[D] + R.u[D]) + dPdd / Z3;
    Ps[D] = a + dud * Z3;
#pragma unroll
    for (int q = 1; q <= 2; ++q) {
        const int t = (D + q) % 3;
        const double b = 0.5 * (L.Pd[t] + R.Pd[t]);
        us[t] = 0.5 * (L.u[t] + R.u[t]) + 0.5 * (L.Pd[t] - R.Pd[t]) / Z1 + dPdd * (b * (1.0 - s3) / (a * Z3));
        Ps[t] = b + 0.5 * (L.u[t] - R.u[t]) * Z1 + dud * (b * nb * (s3 - 1.0) / Z1);
    }
}

template <int D>
__device__ __forceinline__ void bme_axis(const Geo& g, const ConstFields<NBME>& U, int i, int j, int k,
                                         double dnu[3], double dE[6]) {
    const int n[3] = {g.nx, g.ny, g.nz};
    const int bc[3] = {g.bcx, g.bcy, g.bcz};
    int a[3] = {i, j, k};
    const BmeHalf w0 = bme_half<D>(U, cell(g, i, j, k));
    a[D] = map_index((D == 0 ? i : (D == 1 ? j : k)) - 1, n[D], bc[D]);
    const BmeHalf wm = bme_half<D>(U, cell(g, a[0], a[1], a[2]));
    a[D] = map_index((D == 0 ? i : (D == 1 ? j : k)) + 1, n[D], bc[D]);
    const BmeHalf wp = bme_half<D>(U, cell(g, a[0], a[1], a[2]));
    double um[3], Pm[3], up[3], Pp[3];
    bme_face<D>(wm, w0, um, Pm);
    bme_face<D>(w0, wp, up, Pp);
    // d/dx_D of Pi_{iD} and of (Pi_{jD} u_i + Pi_{iD} u_j)
#pragma unroll
    for (int p = 0; p < 3; ++p) dnu[p] += Pp[p] - Pm[p];
#pragma unroll
    for (int p = 0; p < 3; ++p)
#pragma unroll
        for (int q = p; q < 3; ++q)
            dE[sym(p, q)] += (Pp[q] * up[p] + Pp[p] * up[q]) - (Pm[q] * um[p] + Pm[p] * um[q]);
}

__global__ void __launch_bounds__(256)
k_eulerian_bme(Geo g, ConstFields<NBME> U, Fields<NBME> Us, Fields<3> W, Phi phi, double h,
               double dt_val, const double* __restrict__ dt_ptr) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = blockIdx.z * blockDim.z + threadIdx.z;
    if (i >= g.nx || j >= g.ny || k >= g.nz) return;
    const double tau = dt_ptr ? *dt_ptr : dt_val;
    const size_t c = cell(g, i, j, k);
    double gr[3];
    grad_phi(g, phi, i, j, k, 0.5 / h, gr);
    double dnu[3] = {0.0, 0.0, 0.0}, dE[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    bme_axis<0>(g, U, i, j, k, dnu, dE);
    bme_axis<1>(g, U, i, j, k, dnu, dE);
    bme_axis<2>(g, U, i, j, k, dnu, dE);
    const double nn = U.p[0][c];
    const double in = 1.0 / nn;
    const double th = tau / h;
    double u[3];
    Us.p[0][c] = nn;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const double m = U.p[1 + a][c];
        u[a] = m * in;
        const double ms = m - th * dnu[a] - tau * nn * gr[a];
        Us.p[1 + a][c] = ms;
        W.p[a][c] = ms * in;
    }
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = a; b < 3; ++b) {
            const double src = (u[a] - 0.5 * tau * gr[a]) * gr[b] + (u[b] - 0.5 * tau * gr[b]) * gr[a];
            Us.p[4 + sym(a, b)][c] = U.p[4 + sym(a, b)][c] - th * dE[sym(a, b)] - tau * nn * src;
        }
}

// --------------------------------------------------------------------------------------------
// Lagrangian stage, PAPER.md:124 with the face flux of PAPER.md:128 (reading G2): face velocity
// = mean of the 4 face-vertex velocities, each the mean of the 8 cells around the vertex, i.e.
// a (1/4,1/2,1/4)x(1/4,1/2,1/4) transverse average of the two-cell mean; upwind f+.
// --------------------------------------------------------------------------------------------
template <int NF>
__global__ void __launch_bounds__(256)
k_lagrangian(Geo g, ConstFields<NF> Us, Fields<NF> Un, ConstFields<3> W, double h,
             double dt_val, const double* __restrict__ dt_ptr) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = blockIdx.z * blockDim.z + threadIdx.z;
    if (i >= g.nx || j >= g.ny || k >= g.nz) return;
    const double tau = dt_ptr ? *dt_ptr : dt_val;
    const int ii[3] = {map_index(i - 1, g.nx, g.bcx), i, map_index(i + 1, g.nx, g.bcx)};
    const int jj[3] = {map_index(j - 1, g.ny, g.bcy), j, map_index(j + 1, g.ny, g.bcy)};
    const int kk[3] = {map_index(k - 1, g.nz, g.bcz), k, map_index(k + 1, g.nz, g.bcz)};
    const double om[3] = {0.25, 0.5, 0.25};
    double wm[3], wp[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        double line[3] = {0.0, 0.0, 0.0};   // transverse average at offsets -1, 0, +1 along d
#pragma unroll
        for (int a = 0; a < 3; ++a)
#pragma unroll
            for (int b = 0; b < 3; ++b)
#pragma unroll
                for (int s = 0; s < 3; ++s) {
                    // (s along d, a along t1=(d+1)%3, b along t2=(d+2)%3)
                    int o[3];
                    o[d] = s; o[(d + 1) % 3] = a; o[(d + 2) % 3] = b;
                    line[s] += om[a] * om[b] * W.p[d][cell(g, ii[o[0]], jj[o[1]], kk[o[2]])];
                }
        wm[d] = 0.5 * (line[0] + line[1]);
        wp[d] = 0.5 * (line[1] + line[2]);
    }
    const size_t c = cell(g, i, j, k);
    const size_t cxm = cell(g, ii[0], j, k), cxp = cell(g, ii[2], j, k);
    const size_t cym = cell(g, i, jj[0], k), cyp = cell(g, i, jj[2], k);
    const size_t czm = cell(g, i, j, kk[0]), czp = cell(g, i, j, kk[2]);
    const double th = tau / h;
#pragma unroll
    for (int f = 0; f < NF; ++f) {
        const double* __restrict__ fs = Us.p[f];
        const double f0 = fs[c];
        double div = 0.0;
        div += wp[0] * (wp[0] >= 0.0 ? f0 : fs[cxp]) - wm[0] * (wm[0] >= 0.0 ? fs[cxm] : f0);
        div += wp[1] * (wp[1] >= 0.0 ? f0 : fs[cyp]) - wm[1] * (wm[1] >= 0.0 ? fs[cym] : f0);
        div += wp[2] * (wp[2] >= 0.0 ? f0 : fs[czp]) - wm[2] * (wm[2] >= 0.0 ? fs[czm] : f0);
        Un.p[f][c] = f0 - th * div;
    }
}

// --------------------------------------------------------------------------------------------
// CFL reduction (reading G4): max over cells and axes of |v_d| + sqrt(gamma p/rho) and
// |u_d| + sqrt(3 Pi_dd/n).  Speeds are non-negative, so their bit patterns order like the
// values and one atomicMax on the 64-bit pattern finishes the reduction.
// --------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_cfl(size_t N, int has_gas, int has_stars, ConstFields<NGAS> Ug, ConstFields<NBME> Ub, double gamma,
      unsigned long long* __restrict__ smax_bits, int* __restrict__ flag) {
    double smax = 0.0;
    int bad = 0;
    const double gm1 = gamma - 1.0;
    for (size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x; c < N; c += (size_t)gridDim.x * blockDim.x) {
        if (has_gas) {
            const GasPrim w = gas_prim(Ug, c, gm1);
            if (!(w.rho > 0.0) || !(w.p > 0.0)) bad = 1;
            const double cs = sqrt(gamma * w.p / w.rho);
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                const double s = fabs(w.v[d]) + cs;
                if (!(s <= 1.7976931348623157e308)) bad = 1;   // NaN or Inf
                smax = fmax(smax, s);
            }
        }
        if (has_stars) {
            const double nn = Ub.p[0][c];
            if (!(nn > 0.0)) bad = 1;
            const double in = 1.0 / nn;
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                const double u = Ub.p[1 + d][c] * in;
                const double Pdd = Ub.p[4 + sym(d, d)][c] - nn * u * u;
                if (!(Pdd > 0.0)) bad = 1;
                const double s = fabs(u) + sqrt(3.0 * Pdd * in);
                if (!(s <= 1.7976931348623157e308)) bad = 1;
                smax = fmax(smax, s);
            }
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        smax = fmax(smax, __shfl_xor_sync(0xffffffffu, smax, o));
        bad |= __shfl_xor_sync(0xffffffffu, bad, o);
    }
    __shared__ double s_max[8];
    __shared__ int s_bad[8];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0) { s_max[warp] = smax; s_bad[warp] = bad; }
    __syncthreads();
    if (warp == 0) {
        smax = lane < (blockDim.x >> 5) ? s_max[lane] : 0.0;
        bad = lane < (blockDim.x >> 5) ? s_bad[lane] : 0;
#pragma unroll
        for (int o = 4; o > 0; o >>= 1) {
            smax = fmax(smax, __shfl_xor_sync(0xffffffffu, smax, o));
            bad |= __shfl_xor_sync(0xffffffffu, bad, o);
        }
        if (lane == 0) {
            atomicMax(smax_bits, (unsigned long long)__double_as_longlong(smax));
            if (bad) atomicOr(flag, 1);
        }
    }
}

__global__ void k_cfl_begin(unsigned long long* smax_bits, int* flag) {
    *smax_bits = 0ull;
    *flag = 0;
}

__global__ void k_cfl_finish(const unsigned long long* smax_bits, int* flag, double cfl, double h, double* dt) {
    const double s = __longlong_as_double((long long)*smax_bits);
    if (!(s > 0.0)) *flag = 1;
    *dt = cfl * h / s;
}

// Phi ghost faces by a boundary rule (wrap or copy of the nearest interior value).
__global__ void k_phi_ghost(Geo g, const double* __restrict__ phi, double* gx0, double* gx1, double* gy0,
                            double* gy1, double* gz0, double* gz1) {
    const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const size_t nyz = (size_t)g.ny * g.nz, nxz = (size_t)g.nx * g.nz, nxy = (size_t)g.nx * g.ny;
    if (t < nyz) {
        const int j = (int)(t % g.ny), k = (int)(t / g.ny);
        gx0[t] = phi[cell(g, g.bcx == GP_BC_PERIODIC ? g.nx - 1 : 0, j, k)];
        gx1[t] = phi[cell(g, g.bcx == GP_BC_PERIODIC ? 0 : g.nx - 1, j, k)];
    }
    if (t < nxz) {
        const int i = (int)(t % g.nx), k = (int)(t / g.nx);
        gy0[t] = phi[cell(g, i, g.bcy == GP_BC_PERIODIC ? g.ny - 1 : 0, k)];
        gy1[t] = phi[cell(g, i, g.bcy == GP_BC_PERIODIC ? 0 : g.ny - 1, k)];
    }
    if (t < nxy) {
        const int i = (int)(t % g.nx), j = (int)(t / g.nx);
        gz0[t] = phi[cell(g, i, j, g.bcz == GP_BC_PERIODIC ? g.nz - 1 : 0)];
        gz1[t] = phi[cell(g, i, j, g.bcz == GP_BC_PERIODIC ? 0 : g.nz - 1)];
    }
}

// --------------------------------------------------------------------------------------------
// launches
// --------------------------------------------------------------------------------------------
static Geo geo_of(const gp_ctx* c) {
    return Geo{c->g.nx, c->g.ny, c->g.nz, c->bc.x, c->bc.y, c->bc.z};
}

static Phi phi_of(const gp_ctx* c) {
    return Phi{c->phi, c->phig[0], c->phig[1], c->phig[2], c->phig[3], c->phig[4], c->phig[5]};
}

static void grid3(const gp_ctx* c, dim3& grid, dim3& block) {
    block = dim3(64, 2, 2);
    grid = dim3((c->g.nx + block.x - 1) / block.x, (c->g.ny + block.y - 1) / block.y, (c->g.nz + block.z - 1) / block.z);
}

int launch_eulerian_gas(gp_ctx* c, double dt, const double* d_dt) {
    ConstFields<NGAS> U; Fields<NGAS> Us; Fields<3> W;
    for (int f = 0; f < NGAS; ++f) { U.p[f] = c->U[f]; Us.p[f] = c->Us[f]; }
    for (int d = 0; d < 3; ++d) W.p[d] = c->W[d];
    dim3 grid, block;
    grid3(c, grid, block);
    tic(c, K_EUL_GAS);
    k_eulerian_gas<<<grid, block, 0, c->stream>>>(geo_of(c), U, Us, W, phi_of(c), c->gamma, c->g.h, dt, d_dt);
    toc(c);
    c->n_own++;
    GP_CUDA(cudaGetLastError());
    return GP_OK;
}

int launch_eulerian_bme(gp_ctx* c, double dt, const double* d_dt) {
    ConstFields<NBME> U; Fields<NBME> Us; Fields<3> W;
    for (int f = 0; f < NBME; ++f) { U.p[f] = c->U[NGAS + f]; Us.p[f] = c->Us[NGAS + f]; }
    for (int d = 0; d < 3; ++d) W.p[d] = c->W[d];
    dim3 grid, block;
    grid3(c, grid, block);
    tic(c, K_EUL_BME);
    k_eulerian_bme<<<grid, block, 0, c->stream>>>(geo_of(c), U, Us, W, phi_of(c), c->g.h, dt, d_dt);
    toc(c);
    c->n_own++;
    GP_CUDA(cudaGetLastError());
    return GP_OK;
}

template <int NF>
static int launch_lagrangian_t(gp_ctx* c, int f0, double dt, const double* d_dt) {
    ConstFields<NF> Us; Fields<NF> Un; ConstFields<3> W;
    for (int f = 0; f < NF; ++f) { Us.p[f] = c->Us[f0 + f]; Un.p[f] = c->U[f0 + f]; }
    for (int d = 0; d < 3; ++d) W.p[d] = c->W[d];
    dim3 grid, block;
    grid3(c, grid, block);
    tic(c, NF == NGAS ? K_LAG_GAS : K_LAG_BME);
    k_lagrangian<NF><<<grid, block, 0, c->stream>>>(geo_of(c), Us, Un, W, c->g.h, dt, d_dt);
    toc(c);
    c->n_own++;
    GP_CUDA(cudaGetLastError());
    return GP_OK;
}

int launch_lagrangian(gp_ctx* c, int f0, int nf, double dt, const double* d_dt) {
    return nf == NGAS ? launch_lagrangian_t<NGAS>(c, f0, dt, d_dt) : launch_lagrangian_t<NBME>(c, f0, dt, d_dt);
}

int launch_cfl(gp_ctx* c, double cfl) {
    ConstFields<NGAS> Ug; ConstFields<NBME> Ub;
    for (int f = 0; f < NGAS; ++f) Ug.p[f] = c->U[f];
    for (int f = 0; f < NBME; ++f) Ub.p[f] = c->U[NGAS + f];
    tic(c, K_CFL);
    k_cfl_begin<<<1, 1, 0, c->stream>>>(c->d_smax, c->d_flag);
    size_t blocks = (c->N + 255) / 256;
    if (blocks > 148 * 16) blocks = 148 * 16;
    k_cfl<<<(unsigned)blocks, 256, 0, c->stream>>>(c->N, (c->g.components & GP_GAS) != 0, (c->g.components & GP_STARS) != 0,
                                                   Ug, Ub, c->gamma, c->d_smax, c->d_flag);
    k_cfl_finish<<<1, 1, 0, c->stream>>>(c->d_smax, c->d_flag, cfl, c->g.h, c->d_dt);
    toc(c);
    c->n_own += 3;
    GP_CUDA(cudaGetLastError());
    return GP_OK;
}

int launch_phi_ghost_bc(gp_ctx* c, int bcx, int bcy, int bcz) {
    Geo g = geo_of(c);
    g.bcx = bcx; g.bcy = bcy; g.bcz = bcz;
    size_t m = (size_t)g.ny * g.nz;
    if ((size_t)g.nx * g.nz > m) m = (size_t)g.nx * g.nz;
    if ((size_t)g.nx * g.ny > m) m = (size_t)g.nx * g.ny;
    tic(c, K_PHI_GHOST);
    k_phi_ghost<<<(unsigned)((m + 255) / 256), 256, 0, c->stream>>>(g, c->phi, c->phig[0], c->phig[1], c->phig[2],
                                                                   c->phig[3], c->phig[4], c->phig[5]);
    toc(c);
    c->n_own++;
    GP_CUDA(cudaGetLastError());
    return GP_OK;
}

}  // namespace gp
