// Cell-local passes of the overdetermined system (GP_OD contexts; PAPER.md:41 last line, 57, 194-202):
// derive the carried fields from the conserved ones, the energy balance (reading G15) as a pass of its
// own, and the correctness check kappa of the current state.  The step itself carries rho*eps and Pi_ij inside
// the fused kernels (fused_gas_od.cu, fused_bme_od.cu); these passes serve set-up, checks and tests.  fp64.
#include "gp_internal.h"

namespace gp {

namespace {

struct OdFields {
    double* g[NGAS + NODG];   // rho, m (3), rho E, rho eps            (null without gas)
    double* b[NBME + NODB];   // n, nu (3), nE (6), Pi (6)             (null without the collisionless component)
};

__device__ __forceinline__ constexpr int sym(int i, int j) {
    return i == 0 ? j : (j == 0 ? i : (i == 1 ? (j == 1 ? 3 : 4) : (j == 1 ? 4 : 5)));
}

// every field of a GP_OD context is a member of a pair: stride BSTR
__device__ __forceinline__ double& at(double* p, size_t c) { return p[BSTR * c]; }

// MODE 0: derive; 1: balance
template <int MODE>
__global__ void __launch_bounds__(256) k_od_cell(size_t N, OdFields F) {
    for (size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x; c < N; c += (size_t)gridDim.x * blockDim.x) {
        if (F.g[0]) {
            const double rho = at(F.g[0], c);
            double m[3], v[3];
#pragma unroll
            for (int d = 0; d < 3; ++d) { m[d] = at(F.g[1 + d], c); v[d] = m[d] / rho; }
            const double E = at(F.g[4], c);
            const double kin = 0.5 * rho * (v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
            const double e_tot = E - kin;                 // rho eps as the total energy implies it
            if (MODE == 0 || e_tot > 0.0) {
                at(F.g[5], c) = e_tot;
            } else {
                const double eps = at(F.g[5], c);
                const double kin_new = E - eps;           // what rho v^2/2 has to be
                if (kin_new > 0.0 && kin > 0.0) {
                    const double s = sqrt(kin_new / kin); // |v| rescaled, direction kept
#pragma unroll
                    for (int d = 0; d < 3; ++d) at(F.g[1 + d], c) = m[d] * s;
                } else {
#pragma unroll
                    for (int d = 0; d < 3; ++d) at(F.g[1 + d], c) = 0.0;
                    at(F.g[4], c) = eps;
                }
            }
        }
        if (F.b[0]) {
            const double n = at(F.b[0], c);
            double u[3], Pi[6];
#pragma unroll
            for (int d = 0; d < 3; ++d) u[d] = at(F.b[1 + d], c) / n;
#pragma unroll
            for (int i = 0; i < 3; ++i)
#pragma unroll
                for (int j = i; j < 3; ++j) Pi[sym(i, j)] = at(F.b[4 + sym(i, j)], c) - n * u[i] * u[j];
            if (MODE == 0 || (Pi[0] > 0.0 && Pi[3] > 0.0 && Pi[5] > 0.0)) {
#pragma unroll
                for (int s = 0; s < 6; ++s) at(F.b[10 + s], c) = Pi[s];
            } else {
#pragma unroll
                for (int i = 0; i < 3; ++i)
#pragma unroll
                    for (int j = i; j < 3; ++j) at(F.b[4 + sym(i, j)], c) = at(F.b[10 + sym(i, j)], c) + n * u[i] * u[j];
            }
        }
    }
}

// kappa of the current state: per-block partial sums in a fixed order, then one block adds the
// partials in a fixed order: the result does not depend on the scheduling.
constexpr int KB = 148 * 4;

__global__ void __launch_bounds__(256) k_od_kappa_partial(size_t N, OdFields F, double* __restrict__ part) {
    double kg = 0.0, kb = 0.0;
    for (size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x; c < N; c += (size_t)gridDim.x * blockDim.x) {
        if (F.g[0]) {
            const double rho = at(F.g[0], c);
            double v2 = 0.0;
#pragma unroll
            for (int d = 0; d < 3; ++d) { const double v = at(F.g[1 + d], c) / rho; v2 += v * v; }
            kg += fabs(at(F.g[4], c) - at(F.g[5], c) - 0.5 * rho * v2);
        }
        if (F.b[0]) {
            const double n = at(F.b[0], c);
            double u[3];
#pragma unroll
            for (int d = 0; d < 3; ++d) u[d] = at(F.b[1 + d], c) / n;
#pragma unroll
            for (int i = 0; i < 3; ++i)
#pragma unroll
                for (int j = i; j < 3; ++j) kb += fabs(at(F.b[4 + sym(i, j)], c) - at(F.b[10 + sym(i, j)], c) - n * u[i] * u[j]);
        }
    }
    __shared__ double sg[256], sb[256];
    sg[threadIdx.x] = kg; sb[threadIdx.x] = kb;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) { sg[threadIdx.x] += sg[threadIdx.x + o]; sb[threadIdx.x] += sb[threadIdx.x + o]; }
        __syncthreads();
    }
    if (threadIdx.x == 0) { part[2 * blockIdx.x] = sg[0]; part[2 * blockIdx.x + 1] = sb[0]; }
}

__global__ void __launch_bounds__(256) k_od_kappa_final(int nb, const double* __restrict__ part, double h3, double* __restrict__ out) {
    __shared__ double sg[256], sb[256];
    double kg = 0.0, kb = 0.0;
    for (int i = threadIdx.x; i < nb; i += 256) { kg += part[2 * i]; kb += part[2 * i + 1]; }
    sg[threadIdx.x] = kg; sb[threadIdx.x] = kb;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) { sg[threadIdx.x] += sg[threadIdx.x + o]; sb[threadIdx.x] += sb[threadIdx.x + o]; }
        __syncthreads();
    }
    if (threadIdx.x == 0) { out[0] = sg[0] * h3; out[1] = sb[0] * h3; }
}

OdFields fields_of(const gp_ctx* c) {
    OdFields F;
    const bool gas = (c->g.components & GP_GAS) != 0, stars = (c->g.components & GP_STARS) != 0;
    for (int f = 0; f < NGAS; ++f) F.g[f] = gas ? c->U[f] : nullptr;
    F.g[NGAS] = gas ? c->U[F_EPS] : nullptr;
    for (int f = 0; f < NBME; ++f) F.b[f] = stars ? c->U[NGAS + f] : nullptr;
    for (int s = 0; s < NODB; ++s) F.b[NBME + s] = stars ? c->U[F_PI + s] : nullptr;
    return F;
}

unsigned blocks_for(size_t N) {
    size_t b = (N + 255) / 256;
    return (unsigned)(b > 148 * 16 ? 148 * 16 : b);
}

}  // namespace

int launch_od_derive(gp_ctx* c) {
    tic(c, K_OD_AUX);
    k_od_cell<0><<<blocks_for(c->N), 256, 0, c->stream>>>(c->N, fields_of(c));
    toc(c);
    c->n_own++;
    GP_CUDA(cudaGetLastError());
    return GP_OK;
}

int launch_od_balance(gp_ctx* c) {
    tic(c, K_OD_AUX);
    k_od_cell<1><<<blocks_for(c->N), 256, 0, c->stream>>>(c->N, fields_of(c));
    toc(c);
    c->n_own++;
    GP_CUDA(cudaGetLastError());
    return GP_OK;
}

// d_out[0..1] = kappa_gas, kappa_bme.  The partial sums live in the step target of the density pair, which is free
// between steps (as for the field copies of gp_set_state / gp_get_state).
int launch_od_kappa(gp_ctx* c, double* d_out) {
    double* part = (c->g.components & GP_GAS) ? c->Us[0] : c->Us[NGAS];
    size_t nb = (c->N + 255) / 256;
    if (nb > KB) nb = KB;
    if (2 * nb > 2 * c->N) nb = c->N;      // the scratch holds 2 N doubles
    tic(c, K_OD_AUX);
    k_od_kappa_partial<<<(unsigned)nb, 256, 0, c->stream>>>(c->N, fields_of(c), part);
    k_od_kappa_final<<<1, 256, 0, c->stream>>>((int)nb, part, c->g.h * c->g.h * c->g.h, d_out);
    toc(c);
    c->n_own += 2;
    GP_CUDA(cudaGetLastError());
    return GP_OK;
}

}  // namespace gp
