// Poisson step of libgpupegas.so: cuFFT real transforms plus hand-written
// source-assembly, Green's-function and ghost-face kernels.
//
// Periodic mode: PAPER.md:190 with a negative sign and the k = 0 mode set to zero, i.e. the exact
// inverse of the 27-point Laplacian PAPER.md:188 names (reading G3).
// Isolated mode: cyclic convolution on the zero-padded (2N)^3 grid with K(r) = 1/|r|,
// K(0) = (3 ln((sqrt3+1)/(sqrt3-1)) - pi/2)/h (potential at the centre of a uniform cube);
// Phi = -G * sum_j m_j K.  The six ghost faces of Phi are read from padded indices 2N-1 and N,
// where the convolution is still exact.  Phi is written straight into the interior of its ghost-padded
// array (gp_internal.h, PhiPad): cuFFT's inverse transforms through an output embedding, the isolated
// solves by their extraction kernels; k_phi_ghost then fills the ghost layers.
#include <cmath>
#include <vector>

#include "gp_internal.h"

namespace gp {

static inline size_t align256(size_t b) { return (b + 255) & ~(size_t)255; }

size_t poisson_storage_bytes(const gp_grid* g) {
    const size_t nx = g->nx, ny = g->ny, nz = g->nz;
    if (g->poisson == GP_POISSON_PERIODIC) {
        size_t b = align256((nx / 2 + 1) * ny * nz * sizeof(cufftDoubleComplex)) + 3 * align256((nx + ny + nz) * sizeof(double));
        b += align256(2 * nz * sizeof(double));                                   // twiddles of the fused z pass
        b += align256(nx * ny * nz * sizeof(double));   // rho + n (the densities are paired in the state)
        return b;
    }
    if (g->poisson == GP_POISSON_ISOLATED && iso_pruned_supported(g)) return iso_pruned_storage_bytes(g);
    if (g->poisson == GP_POISSON_ISOLATED) {
        const size_t half = (nx + 1) * (2 * ny) * (2 * nz);
        return align256(half * sizeof(cufftDoubleComplex)) + align256(half * sizeof(double)) +
               align256(8 * nx * ny * nz * sizeof(double));
    }
    return 0;
}

// s = rho + n, written where the transform reads it.
__global__ void __launch_bounds__(256)
k_source(size_t N, const double* __restrict__ rho, const double* __restrict__ n, double* __restrict__ s) {
    for (size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x; c < N; c += (size_t)gridDim.x * blockDim.x) {
        double v = 0.0;
        if (rho) v += rho[BSTR * c];
        if (n) v += n[BSTR * c];
        s[c] = v;
    }
}

// Multiply the half spectrum by -4 pi G h^2 / (6 (1 - prod_d (1 - 2/3 sin^2(pi k_d/N_d)))) / N,
// zero at k = 0.  tab_d[k] = 1 - 2/3 sin^2(pi k/N_d).
__global__ void __launch_bounds__(256)
k_green_periodic(int nxh, int ny, int nz, const double* __restrict__ tx, const double* __restrict__ ty,
                 const double* __restrict__ tz, double coef, cufftDoubleComplex* __restrict__ spec) {
    const size_t total = (size_t)nxh * ny * nz;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < total; q += (size_t)gridDim.x * blockDim.x) {
        const int i = (int)(q % nxh);
        const size_t r = q / nxh;
        const int j = (int)(r % ny), k = (int)(r / ny);
        double f = 0.0;
        if (q != 0) f = coef / (6.0 * (1.0 - tx[i] * ty[j] * tz[k]));
        cufftDoubleComplex v = spec[q];
        v.x *= f; v.y *= f;
        spec[q] = v;
    }
}

// ---- isolated mode ----
__global__ void __launch_bounds__(256)
k_pad_source(int nx, int ny, int nz, const double* __restrict__ rho, const double* __restrict__ n, double h3,
             double* __restrict__ padded) {
    const size_t mx = 2 * (size_t)nx, my = 2 * (size_t)ny, mz = 2 * (size_t)nz;
    const size_t total = mx * my * mz;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < total; q += (size_t)gridDim.x * blockDim.x) {
        const size_t i = q % mx, r = q / mx, j = r % my, k = r / my;
        double v = 0.0;
        if (i < (size_t)nx && j < (size_t)ny && k < (size_t)nz) {
            const size_t c = i + (size_t)nx * (j + (size_t)ny * k);
            if (rho) v += rho[BSTR * c];
            if (n) v += n[BSTR * c];
            v *= h3;
        }
        padded[q] = v;
    }
}

__global__ void __launch_bounds__(256)
k_kernel_fill(int nx, int ny, int nz, double h, double kself, double* __restrict__ padded) {
    const size_t mx = 2 * (size_t)nx, my = 2 * (size_t)ny, mz = 2 * (size_t)nz;
    const size_t total = mx * my * mz;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < total; q += (size_t)gridDim.x * blockDim.x) {
        const long long i = q % mx, r = q / mx, j = r % my, k = r / my;
        const double dx = (double)(i < nx ? i : i - (long long)mx);
        const double dy = (double)(j < ny ? j : j - (long long)my);
        const double dz = (double)(k < nz ? k : k - (long long)mz);
        const double r2 = dx * dx + dy * dy + dz * dz;
        padded[q] = r2 == 0.0 ? kself / h : 1.0 / (h * sqrt(r2));
    }
}

__global__ void __launch_bounds__(256)
k_take_real(size_t total, const cufftDoubleComplex* __restrict__ spec, double* __restrict__ out) {
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < total; q += (size_t)gridDim.x * blockDim.x)
        out[q] = spec[q].x;
}

__global__ void __launch_bounds__(256)
k_mul_real(size_t total, const double* __restrict__ ks, double scale, cufftDoubleComplex* __restrict__ spec) {
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < total; q += (size_t)gridDim.x * blockDim.x) {
        const double f = ks[q] * scale;
        cufftDoubleComplex v = spec[q];
        v.x *= f; v.y *= f;
        spec[q] = v;
    }
}

// Interior of the (2N)^3 result -> Phi; its indices 2N-1 and N -> the six ghost faces (cells -1 and n).
// phi points at cell (0,0,0) of the ghost-padded Phi array (row pitch `pitch`, py rows per plane).
__global__ void __launch_bounds__(256)
k_extract(int nx, int ny, int nz, const double* __restrict__ padded, double* __restrict__ phi, int pitch, int py) {
    const size_t mx = 2 * (size_t)nx, my = 2 * (size_t)ny;
    const size_t N = (size_t)nx * ny * nz;
    auto P = [&](size_t i, size_t j, size_t k) { return padded[i + mx * (j + my * k)]; };
    auto F = [&](long long i, long long j, long long k) -> double& { return phi[i + (long long)pitch * (j + (long long)py * k)]; };
    for (size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x; c < N; c += (size_t)gridDim.x * blockDim.x) {
        const size_t i = c % nx, r = c / nx, j = r % ny, k = r / ny;
        F(i, j, k) = P(i, j, k);
        if (i == 0) { F(-1, j, k) = P(2 * (size_t)nx - 1, j, k); F(nx, j, k) = P(nx, j, k); }
        if (j == 0) { F(i, -1, k) = P(i, 2 * (size_t)ny - 1, k); F(i, ny, k) = P(i, ny, k); }
        if (k == 0) { F(i, j, -1) = P(i, j, 2 * (size_t)nz - 1); F(i, j, nz) = P(i, j, nz); }
    }
}

static unsigned blocks_for(size_t n) {
    size_t b = (n + 255) / 256;
    const size_t cap = 148 * 32;
    return (unsigned)(b > cap ? cap : (b ? b : 1));
}

int poisson_setup(gp_ctx* c) {
    if (c->fft_ready) return GP_OK;
    const int nx = c->g.nx, ny = c->g.ny, nz = c->g.nz;
    const int pitch = phi_pitch(nx), py = ny + 4;      // the inverse transform writes into the padded Phi
    if (c->g.poisson == GP_POISSON_PERIODIC) {
        c->zfused = zpass_supported(nz);
        // The table uploads come first: a failure here returns before any plan exists, so nothing is left
        // behind for a retry to leak (the plans are created last and cleaned up by the rc path below).
        const double pi = 3.14159265358979323846;
        std::vector<double> t((size_t)nx + ny + nz);
        for (int k = 0; k < nx; ++k) { const double s = std::sin(pi * k / nx); t[k] = 1.0 - 2.0 / 3.0 * s * s; }
        for (int k = 0; k < ny; ++k) { const double s = std::sin(pi * k / ny); t[nx + k] = 1.0 - 2.0 / 3.0 * s * s; }
        for (int k = 0; k < nz; ++k) { const double s = std::sin(pi * k / nz); t[nx + ny + k] = 1.0 - 2.0 / 3.0 * s * s; }
        GP_CUDA(cudaMemcpyAsync(c->tabx, t.data(), t.size() * sizeof(double), cudaMemcpyHostToDevice, c->stream));
        GP_CUDA(cudaStreamSynchronize(c->stream));
        if (c->zfused) {
            std::vector<double> w(2 * (size_t)nz);
            for (int k = 0; k < nz; ++k) {
                const long double a = 2.0L * 3.14159265358979323846264338327950288L * (long double)k / (long double)nz;
                w[2 * k] = (double)cosl(a);
                w[2 * k + 1] = (double)-sinl(a);
            }
            GP_CUDA(cudaMemcpyAsync(c->ztw, w.data(), w.size() * sizeof(double), cudaMemcpyHostToDevice, c->stream));
            GP_CUDA(cudaStreamSynchronize(c->stream));
        }
        if (c->zfused) {
            // batched 2-D real transforms over the xy planes; the z direction is zpass.cu's
            int n[2] = {ny, nx}, rembed[2] = {ny, nx}, cembed[2] = {ny, nx / 2 + 1}, pembed[2] = {py, pitch};
            GP_CUFFT(cufftPlanMany(&c->plan_fwd, 2, n, rembed, 1, ny * nx, cembed, 1, ny * (nx / 2 + 1), CUFFT_D2Z, nz));
            if (cufftPlanMany(&c->plan_inv, 2, n, cembed, 1, ny * (nx / 2 + 1), pembed, 1, py * pitch, CUFFT_Z2D, nz) != CUFFT_SUCCESS) {
                cufftDestroy(c->plan_fwd);
                set_error("gp_solve_poisson: cufftPlanMany (inverse, padded output) failed");
                return GP_ERR_CUFFT;
            }
        } else {
            int n[3] = {nz, ny, nx}, cembed[3] = {nz, ny, nx / 2 + 1}, pembed[3] = {nz + 4, py, pitch};
            GP_CUFFT(cufftPlan3d(&c->plan_fwd, nz, ny, nx, CUFFT_D2Z));
            if (cufftPlanMany(&c->plan_inv, 3, n, cembed, 1, nz * ny * (nx / 2 + 1), pembed, 1, (nz + 4) * py * pitch, CUFFT_Z2D, 1) != CUFFT_SUCCESS) {
                cufftDestroy(c->plan_fwd);
                set_error("gp_solve_poisson: cufftPlanMany (inverse 3-D, padded output) failed");
                return GP_ERR_CUFFT;
            }
        }
    } else if (c->g.poisson == GP_POISSON_ISOLATED && c->isofast) {
        return iso_pruned_setup(c);
    } else if (c->g.poisson == GP_POISSON_ISOLATED) {
        GP_CUFFT(cufftPlan3d(&c->plan_fwd, 2 * nz, 2 * ny, 2 * nx, CUFFT_D2Z));
        if (cufftPlan3d(&c->plan_inv, 2 * nz, 2 * ny, 2 * nx, CUFFT_Z2D) != CUFFT_SUCCESS) {
            cufftDestroy(c->plan_fwd);
            set_error("gp_solve_poisson: cufftPlan3d (inverse) failed");
            return GP_ERR_CUFFT;
        }
    } else {
        set_error("gp_solve_poisson: context was created with GP_POISSON_NONE");
        return GP_ERR_UNSUPPORTED;
    }
    // From here on a failure must not leave half-built plans behind, and fft_ready is set only once the
    // kernel spectrum exists: a retry after a failed set-up repeats it instead of convolving with zeros.
    int rc = GP_OK;
    if (cufftSetStream(c->plan_fwd, c->stream) != CUFFT_SUCCESS || cufftSetStream(c->plan_inv, c->stream) != CUFFT_SUCCESS) {
        set_error("gp_solve_poisson: cufftSetStream failed");
        rc = GP_ERR_CUFFT;
    }
    if (rc == GP_OK && c->g.poisson == GP_POISSON_ISOLATED) {
        // spectrum of the kernel, once: real because the kernel is even in every axis
        const size_t total = 8 * c->N, half = ((size_t)nx + 1) * (2 * (size_t)ny) * (2 * (size_t)nz);
        const double s3 = std::sqrt(3.0), pi = 3.14159265358979323846;
        const double kself = 3.0 * std::log((s3 + 1.0) / (s3 - 1.0)) - pi / 2.0;
        k_kernel_fill<<<blocks_for(total), 256, 0, c->stream>>>(nx, ny, nz, c->g.h, kself, c->padded);
        if (cufftExecD2Z(c->plan_fwd, c->padded, c->spec) != CUFFT_SUCCESS) {
            set_error("gp_solve_poisson: kernel-spectrum transform failed");
            rc = GP_ERR_CUFFT;
        }
        k_take_real<<<blocks_for(half), 256, 0, c->stream>>>(half, c->spec, c->kspec);
        c->n_own += 2; c->n_fft += 1;
        const cudaError_t e = cudaStreamSynchronize(c->stream);
        if (rc == GP_OK && e != cudaSuccess) {
            set_error("gp_solve_poisson: building the kernel spectrum: %s", cudaGetErrorString(e));
            rc = GP_ERR_CUDA;
        }
    }
    if (rc != GP_OK) {
        cufftDestroy(c->plan_fwd);
        cufftDestroy(c->plan_inv);
        return rc;
    }
    c->fft_ready = true;
    return GP_OK;
}

void poisson_teardown(gp_ctx* c) {
    if (c->fft_ready) {
        cufftDestroy(c->plan_fwd);
        cufftDestroy(c->plan_inv);
        c->fft_ready = false;
    }
}

int poisson_solve(gp_ctx* c) {
    int rc = poisson_setup(c);
    if (rc != GP_OK) return rc;
    const int nx = c->g.nx, ny = c->g.ny, nz = c->g.nz;
    const double* rho = (c->g.components & GP_GAS) ? c->U[GP_RHO] : nullptr;
    const double* n = (c->g.components & GP_STARS) ? c->U[GP_N] : nullptr;
    const double pi = 3.14159265358979323846;
    if (c->g.poisson == GP_POISSON_PERIODIC) {
        const size_t half = ((size_t)nx / 2 + 1) * ny * nz;
        // source rho + n in c->src (the densities are paired in the state, cuFFT wants a plain
        // array): already written by the fused step unless the state was set since, or stars only
        const double* s = c->src;
        if (!c->src_cached) {
            tic(c, K_SOURCE);
            k_source<<<blocks_for(c->N), 256, 0, c->stream>>>(c->N, rho, n, c->src);
            toc(c);
            c->n_own += 1;
        }
        tic(c, K_FFT_FWD);
        GP_CUFFT(cufftExecD2Z(c->plan_fwd, const_cast<double*>(s), c->spec));
        toc(c);
        const double coef = -4.0 * pi * c->g.G * c->g.h * c->g.h / (double)c->N;
        if (c->zfused) {
            tic(c, K_ZPASS);
            rc = launch_zpass(c, coef / 6.0);
            toc(c);
            if (rc != GP_OK) return rc;
        } else {
            tic(c, K_GREEN);
            k_green_periodic<<<blocks_for(half), 256, 0, c->stream>>>(nx / 2 + 1, ny, nz, c->tabx, c->taby, c->tabz, coef, c->spec);
            toc(c);
        }
        tic(c, K_FFT_INV);
        GP_CUFFT(cufftExecZ2D(c->plan_inv, c->spec, phi_interior(c)));
        toc(c);
        c->n_own += 1; c->n_fft += 2;
        GP_CUDA(cudaGetLastError());
        return launch_phi_ghost_bc(c, GP_BC_PERIODIC, GP_BC_PERIODIC, GP_BC_PERIODIC);
    }
    if (c->isofast) return iso_pruned_solve(c);
    const size_t total = 8 * c->N, half = ((size_t)nx + 1) * (2 * (size_t)ny) * (2 * (size_t)nz);
    tic(c, K_PAD_SOURCE);
    k_pad_source<<<blocks_for(total), 256, 0, c->stream>>>(nx, ny, nz, rho, n, c->g.h * c->g.h * c->g.h, c->padded);
    toc(c);
    tic(c, K_FFT_FWD);
    GP_CUFFT(cufftExecD2Z(c->plan_fwd, c->padded, c->spec));
    toc(c);
    tic(c, K_MUL_KERNEL);
    k_mul_real<<<blocks_for(half), 256, 0, c->stream>>>(half, c->kspec, -c->g.G / (double)total, c->spec);
    toc(c);
    tic(c, K_FFT_INV);
    GP_CUFFT(cufftExecZ2D(c->plan_inv, c->spec, c->padded));
    toc(c);
    tic(c, K_EXTRACT);
    k_extract<<<blocks_for(c->N), 256, 0, c->stream>>>(nx, ny, nz, c->padded, phi_interior(c), phi_pitch(nx), ny + 4);
    toc(c);
    c->n_own += 3; c->n_fft += 2;
    GP_CUDA(cudaGetLastError());
    // layer 2, edges and corners: never used by a result (outflow hydro boundaries), kept finite
    return launch_phi_ghost_bc(c, GP_BC_OUTFLOW, GP_BC_OUTFLOW, GP_BC_OUTFLOW, true);
}

}  // namespace gp
