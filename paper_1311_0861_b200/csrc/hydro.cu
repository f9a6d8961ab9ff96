// Stand-alone CFL reduction (used when the state was set from outside; after a step the fused
// kernels of fused_impl.cuh have already folded the max signal speed of the new state) and the Phi
// ghost faces.  fp64 throughout.
#include "gp_internal.h"

namespace gp {

__device__ __forceinline__ size_t cell(const Geo& g, int i, int j, int k) {
    return (size_t)i + (size_t)g.nx * ((size_t)j + (size_t)g.ny * (size_t)k);
}

// sym(i,j) -> index in (xx,xy,xz,yy,yz,zz)
__device__ __forceinline__ constexpr int sym(int i, int j) {
    return i == 0 ? j : (j == 0 ? i : (i == 1 ? (j == 1 ? 3 : 4) : (j == 1 ? 4 : 5)));
}

struct GasPrim { double rho, v[3], p; };

__device__ __forceinline__ GasPrim gas_prim(const ConstFields<NGAS>& U, size_t c, double gm1) {
    GasPrim w;
    w.rho = U.p[0][BSTR * c];
    const double ir = 1.0 / w.rho;
    w.v[0] = U.p[1][BSTR * c] * ir;
    w.v[1] = U.p[2][BSTR * c] * ir;
    w.v[2] = U.p[3][BSTR * c] * ir;
    w.p = gm1 * (U.p[4][c] - 0.5 * w.rho * (w.v[0] * w.v[0] + w.v[1] * w.v[1] + w.v[2] * w.v[2]));
    return w;
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
            const double nn = Ub.p[0][BSTR * c];
            if (!(nn > 0.0)) bad = 1;
            const double in = 1.0 / nn;
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                const double u = Ub.p[1 + d][BSTR * c] * in;
                const double Pdd = Ub.p[4 + sym(d, d)][BSTR * c] - nn * u * u;
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

__global__ void k_cfl_finish(const unsigned long long* smax_bits, const int* flag_in, int* flag_out, double cfl, double h,
                             double* dt) {
    const double s = __longlong_as_double((long long)*smax_bits);
    *flag_out = (*flag_in != 0 || !(s > 0.0)) ? 1 : 0;
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

__global__ void __launch_bounds__(256)
k_strided_copy(size_t n, double* __restrict__ dst, int dstride, const double* __restrict__ src, int sstride) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
        dst[i * dstride] = src[i * sstride];
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
    k_cfl_finish<<<1, 1, 0, c->stream>>>(c->d_smax, c->d_flag, c->d_flag, cfl, c->g.h, c->d_dt);
    toc(c);
    c->n_own += 3;
    GP_CUDA(cudaGetLastError());
    return GP_OK;
}

// dt from the max signal speed the fused step kernels folded for the current state
int launch_cfl_from_cache(gp_ctx* c, double cfl) {
    tic(c, K_CFL);
    k_cfl_finish<<<1, 1, 0, c->stream>>>(c->d_smax_next, c->d_flag_next, c->d_flag, cfl, c->g.h, c->d_dt);
    toc(c);
    c->n_own += 1;
    GP_CUDA(cudaGetLastError());
    return GP_OK;
}

int launch_cfl_reset_next(gp_ctx* c) {
    k_cfl_begin<<<1, 1, 0, c->stream>>>(c->d_smax_next, c->d_flag_next);
    c->n_own += 1;
    GP_CUDA(cudaGetLastError());
    return GP_OK;
}

int launch_strided_copy(gp_ctx* c, double* dst, int dstride, const double* src, int sstride, size_t n) {
    size_t blocks = (n + 255) / 256;
    if (blocks > 148 * 16) blocks = 148 * 16;
    k_strided_copy<<<(unsigned)blocks, 256, 0, c->stream>>>(n, dst, dstride, src, sstride);
    c->n_own++;
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
