// Stand-alone CFL reduction (used when the state was set from outside; after a step the fused
// kernels of fused_impl.cuh have already folded the max signal speed of the new state) and the ghost
// layers of the padded Phi.  fp64 throughout.
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

// estr: stride of the energy array (1, or BSTR in a GP_OD context where it is paired with rho*eps)
__device__ __forceinline__ GasPrim gas_prim(const ConstFields<NGAS>& U, size_t c, double gm1, int estr) {
    GasPrim w;
    w.rho = U.p[0][BSTR * c];
    const double ir = 1.0 / w.rho;
    w.v[0] = U.p[1][BSTR * c] * ir;
    w.v[1] = U.p[2][BSTR * c] * ir;
    w.v[2] = U.p[3][BSTR * c] * ir;
    w.p = gm1 * (U.p[4][estr * c] - 0.5 * w.rho * (w.v[0] * w.v[0] + w.v[1] * w.v[1] + w.v[2] * w.v[2]));
    return w;
}

// --------------------------------------------------------------------------------------------
// CFL reduction (reading G4): max over cells and axes of |v_d| + sqrt(gamma p/rho) and
// |u_d| + sqrt(3 Pi_dd/n); in a GP_OD context p and Pi_dd are the carried ones (reading G16).  Speeds are
// non-negative, so their bit patterns order like the values and one atomicMax on the 64-bit pattern finishes
// the reduction.
// --------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_cfl(size_t N, int has_gas, int has_stars, ConstFields<NGAS> Ug, int estr, ConstFields<NBME> Ub, double gamma,
      const double* __restrict__ eps, ConstFields<3> Pdd_carried,
      unsigned long long* __restrict__ smax_bits, int* __restrict__ flag) {
    double smax = 0.0;
    int bad = 0;
    const double gm1 = gamma - 1.0;
    for (size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x; c < N; c += (size_t)gridDim.x * blockDim.x) {
        if (has_gas) {
            GasPrim w = gas_prim(Ug, c, gm1, estr);
            if (eps) w.p = gm1 * eps[BSTR * c];        // GP_OD (reading G16): the pressure the stages use
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
                const double Pdd = Pdd_carried.p[d] ? Pdd_carried.p[d][BSTR * c]      // GP_OD (reading G16)
                                                    : Ub.p[4 + sym(d, d)][BSTR * c] - nn * u * u;
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

// Ghost layers of the padded Phi (gp_internal.h, PhiPad) by a boundary rule per axis: wrap (GP_BC_PERIODIC) or
// copy of the nearest interior value (GP_BC_OUTFLOW).  Per-axis index maps equal filling x, then y over the
// x-extended range, then z: edges and corners included.  keep_faces: positions with exactly one coordinate
// outside by one (the six ghost faces) already hold their values (isolated solve) and are left alone.
__device__ __forceinline__ int ghost_map(int i, int n, int bc) {
    if (bc == GP_BC_PERIODIC) return i < 0 ? i + n : (i >= n ? i - n : i);
    return i < 0 ? 0 : (i >= n ? n - 1 : i);
}

__global__ void __launch_bounds__(256)
k_phi_ghost(Geo g, double* __restrict__ pad, int pitch, int keep_faces) {
    const int px = g.nx + 4, py = g.ny + 4;
    // enumerate the ghost cells only: four z slabs, then four y rows of every interior plane, then four x columns
    const size_t nzs = (size_t)4 * px * py, nys = (size_t)4 * px * g.nz, nxs = (size_t)4 * g.ny * g.nz;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < nzs + nys + nxs; q += (size_t)gridDim.x * blockDim.x) {
        int I, J, K;      // padded coordinates
        if (q < nzs) {
            I = (int)(q % px); J = (int)(q / px % py); const int s = (int)(q / ((size_t)px * py));
            K = s < 2 ? s : g.nz + s;
        } else if (q < nzs + nys) {
            const size_t r = q - nzs;
            I = (int)(r % px); const int s = (int)(r / px % 4); K = 2 + (int)(r / ((size_t)4 * px));
            J = s < 2 ? s : g.ny + s;
        } else {
            const size_t r = q - nzs - nys;
            const int s = (int)(r % 4); J = 2 + (int)(r / 4 % g.ny); K = 2 + (int)(r / ((size_t)4 * g.ny));
            I = s < 2 ? s : g.nx + s;
        }
        const int i = I - 2, j = J - 2, k = K - 2;
        if (keep_faces) {
            const int ox = i < 0 ? -i : (i >= g.nx ? i - g.nx + 1 : 0), oy = j < 0 ? -j : (j >= g.ny ? j - g.ny + 1 : 0),
                      oz = k < 0 ? -k : (k >= g.nz ? k - g.nz + 1 : 0);
            if (ox + oy + oz == 1) continue;
        }
        const int im = ghost_map(i, g.nx, g.bcx), jm = ghost_map(j, g.ny, g.bcy), km = ghost_map(k, g.nz, g.bcz);
        pad[(size_t)I + (size_t)pitch * (J + (size_t)py * K)] = pad[(size_t)(im + 2) + (size_t)pitch * ((jm + 2) + (size_t)py * (km + 2))];
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

int launch_cfl(gp_ctx* c, double cfl) {
    ConstFields<NGAS> Ug; ConstFields<NBME> Ub;
    for (int f = 0; f < NGAS; ++f) Ug.p[f] = c->U[f];
    for (int f = 0; f < NBME; ++f) Ub.p[f] = c->U[NGAS + f];
    // GP_OD: signal speeds and the bad-state flag from the carried rho*eps and Pi_xx, Pi_yy, Pi_zz
    const double* eps = (c->od && (c->g.components & GP_GAS)) ? c->U[F_EPS] : nullptr;
    ConstFields<3> Pc;
    const int diag[3] = {0, 3, 5};
    for (int d = 0; d < 3; ++d) Pc.p[d] = (c->od && (c->g.components & GP_STARS)) ? c->U[F_PI + diag[d]] : nullptr;
    tic(c, K_CFL);
    k_cfl_begin<<<1, 1, 0, c->stream>>>(c->d_smax, c->d_flag);
    size_t blocks = (c->N + 255) / 256;
    if (blocks > 148 * 16) blocks = 148 * 16;
    k_cfl<<<(unsigned)blocks, 256, 0, c->stream>>>(c->N, (c->g.components & GP_GAS) != 0, (c->g.components & GP_STARS) != 0,
                                                   Ug, c->estr, Ub, c->gamma, eps, Pc, c->d_smax, c->d_flag);
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

int launch_phi_ghost_bc(gp_ctx* c, int bcx, int bcy, int bcz, bool keep_faces) {
    Geo g = geo_of(c);
    g.bcx = bcx; g.bcy = bcy; g.bcz = bcz;
    const size_t m = (size_t)4 * (g.nx + 4) * (g.ny + 4) + (size_t)4 * (g.nx + 4) * g.nz + (size_t)4 * g.ny * g.nz;
    size_t blocks = (m + 255) / 256;
    if (blocks > 148 * 16) blocks = 148 * 16;
    tic(c, K_PHI_GHOST);
    k_phi_ghost<<<(unsigned)blocks, 256, 0, c->stream>>>(g, c->phip, phi_pitch(g.nx), keep_faces ? 1 : 0);
    toc(c);
    c->n_own++;
    GP_CUDA(cudaGetLastError());
    return GP_OK;
}

}  // namespace gp
