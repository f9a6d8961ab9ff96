// Pruned transforms of the isolated Poisson solve (reading G3: cyclic
// convolution with -G/r on the zero-padded (2N)^3 grid).  Only the x lines, y columns and z columns
// that hold data are transformed, the implicit zeros are never read, and only the planes, rows and
// samples Phi and its six ghost faces need are written back:
//   x : cuFFT batched 1-D D2Z / Z2D over the ny*nz (resp. (ny+2)(nz+2)) lines that matter
//   y : k_colfft forward (ny rows in, 2ny out, left in digit-reversed order) and inverse
//   z : k_colfft forward * kernel spectrum * inverse in ONE pass over the spectrum
// The kernel spectrum is produced once by the same forward pipeline, so it is in the same
// (digit-reversed in y and z) layout and no reordering is ever needed.
#include <cmath>
#include <vector>

#include "fftcol.cuh"

namespace gp {

struct ColArgs {
    const double2* in;
    double2* out;
    const double* table;                       // MUL: real factor at [position * tab_rs + column]
    long long in_rs, in_ss, out_rs, out_ss;    // row and slab strides, in complex elements
    long long tab_rs;
    int tiles;                                 // column tiles (of C columns) per slab
    int nin;                                   // rows >= nin of the input are implicit zeros (FWD)
    int nkeep;                                 // INV: rows 0..nkeep are written, and row 2^P-1 as row nkeep+1; < 0: all
    double scale;                              // MUL: multiplies the table
};

// forward stages s..S-1 (FWD), factor (MUL), inverse stages S-1..s (INV)
template <int P, int C, int s, bool FWD, bool INV, bool MUL>
struct CPipe {
    __device__ static __forceinline__ void run(double2* v, double2* sm, const double2* __restrict__ tw, int t, int col,
                                               const double* __restrict__ tab, long long tab_rs, double scale) {
        constexpr int S = ZStages<P>::S;
        if (FWD) zstage<P, s, false>(v, tw, t);
        if constexpr (s + 1 < S) {
            if (FWD) ZExchange<P, C, s>::template run<s + 1>(v, sm, t, col);
            CPipe<P, C, s + 1, FWD, INV, MUL>::run(v, sm, tw, t, col, tab, tab_rs, scale);
            if (INV) ZExchange<P, C, s + 1>::template run<s>(v, sm, t, col);
        } else if (MUL) {
            constexpr int R = ZStages<P>::radix(s), L = ZStages<P>::len(s);
#pragma unroll
            for (int b = 0; b < 8 / R; ++b)
#pragma unroll
                for (int m = 0; m < R; ++m) {
                    const double f = scale * tab[(long long)zidx<P, R, L>(t, b, m) * tab_rs];
                    v[b * R + m].x *= f; v[b * R + m].y *= f;
                }
        }
        if (INV) zstage<P, s, true>(v, tw, t);
    }
};

template <int P, int C, int MINB, bool FWD, bool INV, bool MUL>
__global__ void __launch_bounds__((1 << P) / 8 * C, MINB)
k_colfft(ColArgs a, const double2* __restrict__ tw) {
    extern __shared__ double2 csm[];
    constexpr int S = ZStages<P>::S;
    constexpr int LS = FWD ? 0 : S - 1, SS = INV ? 0 : S - 1;     // register layouts of the load and of the store
    constexpr int RL = ZStages<P>::radix(LS), LL = ZStages<P>::len(LS);
    constexpr int RS = ZStages<P>::radix(SS), LSn = ZStages<P>::len(SS);
    const int col = threadIdx.x % C, t = threadIdx.x / C;
    const long long slab = blockIdx.x / a.tiles, q = (long long)(blockIdx.x % a.tiles) * C + col;
    const double2* in = a.in + slab * a.in_ss + q;
    double2 v[8];
#pragma unroll
    for (int b = 0; b < 8 / RL; ++b)
#pragma unroll
        for (int m = 0; m < RL; ++m) {
            const int r = zidx<P, RL, LL>(t, b, m);
            v[b * RL + m] = r < a.nin ? in[(long long)r * a.in_rs] : make_double2(0.0, 0.0);
        }
    CPipe<P, C, 0, FWD, INV, MUL>::run(v, csm, tw, t, col, MUL ? a.table + q : nullptr, a.tab_rs, a.scale);
    double2* out = a.out + slab * a.out_ss + q;
#pragma unroll
    for (int b = 0; b < 8 / RS; ++b)
#pragma unroll
        for (int m = 0; m < RS; ++m) {
            const int r = zidx<P, RS, LSn>(t, b, m);
            if (a.nkeep < 0 || r <= a.nkeep) out[(long long)r * a.out_rs] = v[b * RS + m];
            else if (r == (1 << P) - 1) out[(long long)(a.nkeep + 1) * a.out_rs] = v[b * RS + m];
        }
}

enum ColMode { COL_FWD = 0, COL_INV = 1, COL_FUSED = 2 };

template <int P, int C, int MINB, bool FWD, bool INV, bool MUL>
static int launch_col_k(gp_ctx* c, const ColArgs& a, long long slabs, const double2* tw) {
    const int threads = (1 << P) / 8 * C;
    const size_t smem = (size_t)(1 << P) * C * sizeof(double2);
    // the opt-in is per device and cheap: set it on every launch (a context may live on any device)
    GP_CUDA(cudaFuncSetAttribute(k_colfft<P, C, MINB, FWD, INV, MUL>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    k_colfft<P, C, MINB, FWD, INV, MUL><<<(unsigned)(slabs * a.tiles), threads, smem, c->stream>>>(a, tw);
    GP_CUDA(cudaGetLastError());
    return GP_OK;
}

template <int P, int C, int MINB>
static int launch_col_p(gp_ctx* c, int mode, ColArgs a, long long slabs, long long ncols, const double2* tw) {
    a.tiles = (int)(ncols / C);
    if (mode == COL_FWD) return launch_col_k<P, C, MINB, true, false, false>(c, a, slabs, tw);
    if (mode == COL_INV) return launch_col_k<P, C, MINB, false, true, false>(c, a, slabs, tw);
    return launch_col_k<P, C, MINB, true, true, true>(c, a, slabs, tw);
}

// n = transform length (power of two in [8, 1024]); ncols must be a multiple of 8
static int launch_col(gp_ctx* c, int n, int mode, const ColArgs& a, long long slabs, long long ncols, const double2* tw) {
    switch (n) {
        case 8: return launch_col_p<3, 8, 1>(c, mode, a, slabs, ncols, tw);
        case 16: return launch_col_p<4, 8, 1>(c, mode, a, slabs, ncols, tw);
        case 32: return launch_col_p<5, 8, 1>(c, mode, a, slabs, ncols, tw);
        case 64: return launch_col_p<6, 8, 1>(c, mode, a, slabs, ncols, tw);
        case 128: return launch_col_p<7, 8, 1>(c, mode, a, slabs, ncols, tw);
        case 256: return launch_col_p<8, 8, 1>(c, mode, a, slabs, ncols, tw);
        case 512: return launch_col_p<9, 4, 2>(c, mode, a, slabs, ncols, tw);
        case 1024: return launch_col_p<10, 4, 1>(c, mode, a, slabs, ncols, tw);   // <10, 2, 2> measured 30 % slower
    }
    set_error("isolated solve: transform length %d is not a supported power of two", n);
    return GP_ERR_UNSUPPORTED;
}

static inline size_t al256(size_t b) { return (b + 255) & ~(size_t)255; }
static inline bool pow2(int n) { return n > 0 && (n & (n - 1)) == 0; }

// the pruned path needs power-of-two ny, nz with 2n <= 1024; x goes through cuFFT and is free
bool iso_pruned_supported(const gp_grid* g) { return pow2(g->ny) && pow2(g->nz) && g->ny <= 512 && g->nz <= 512; }

static inline size_t iso_nxp(const gp_grid* g) { return ((size_t)g->nx + 1 + 7) & ~(size_t)7; }

// R real (nz+2)(ny+2)(2nx) | A complex (nz+2)(ny+2)nxp | B complex (nz+2)(2ny)nxp | K real (2nz)(2ny)nxp | twiddles
size_t iso_pruned_storage_bytes(const gp_grid* g) {
    const size_t nx = g->nx, ny = g->ny, nz = g->nz, nxp = iso_nxp(g);
    return al256((nz + 2) * (ny + 2) * 2 * nx * sizeof(double)) + al256((nz + 2) * (ny + 2) * nxp * sizeof(double2)) +
           al256((nz + 2) * 2 * ny * nxp * sizeof(double2)) + al256(2 * nz * 2 * ny * nxp * sizeof(double)) +
           al256(2 * ny * sizeof(double2)) + al256(2 * nz * sizeof(double2));
}

// ---- elementwise kernels ------------------------------------------------------------------------
// x lines of the source, zero padded to 2nx: m = (rho + n) h^3 (mass per cell)
__global__ void __launch_bounds__(256)
k_iso_pad_x(int nx, size_t lines, const double* __restrict__ rho, const double* __restrict__ n, double h3,
            double* __restrict__ R) {
    const size_t total = lines * 2 * (size_t)nx;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < total; q += (size_t)gridDim.x * blockDim.x) {
        const size_t line = q / (2 * (size_t)nx), i = q % (2 * (size_t)nx);
        double v = 0.0;
        if (i < (size_t)nx) {
            const size_t c = line * nx + i;
            if (rho) v += rho[BSTR * c];
            if (n) v += n[BSTR * c];
            v *= h3;
        }
        R[q] = v;
    }
}

// R[(nz+2)][(ny+2)][2nx] -> Phi and its six ghost faces; plane / row n holds padded index n, plane /
// row n+1 holds padded index 2n-1 (where the cyclic convolution is still exact, G3)
// phi points at cell (0,0,0) of the ghost-padded Phi array (row pitch `pitch`, py rows per plane); the
// ghost faces are its cells -1 and n.
__global__ void __launch_bounds__(256)
k_iso_extract(int nx, int ny, int nz, const double* __restrict__ R, double* __restrict__ phi, int pitch, int py) {
    const size_t mx = 2 * (size_t)nx, rows = (size_t)ny + 2;
    const size_t N = (size_t)nx * ny * nz;
    auto P = [&](size_t i, size_t j, size_t k) { return R[i + mx * (j + rows * k)]; };
    auto F = [&](long long i, long long j, long long k) -> double& { return phi[i + (long long)pitch * (j + (long long)py * k)]; };
    for (size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x; c < N; c += (size_t)gridDim.x * blockDim.x) {
        const size_t i = c % nx, r = c / nx, j = r % ny, k = r / ny;
        F(i, j, k) = P(i, j, k);
        if (i == 0) { F(-1, j, k) = P(2 * (size_t)nx - 1, j, k); F(nx, j, k) = P(nx, j, k); }
        if (j == 0) { F(i, -1, k) = P(i, ny + 1, k); F(i, ny, k) = P(i, ny, k); }
        if (k == 0) { F(i, j, -1) = P(i, j, nz + 1); F(i, j, nz) = P(i, j, nz); }
    }
}

// K(r) = 1/|r| on the padded grid stored cyclically, K(0) = kself / h (G3)
__global__ void __launch_bounds__(256)
k_iso_kernel_fill(int nx, int ny, int nz, double h, double kself, double* __restrict__ K) {
    const size_t mx = 2 * (size_t)nx, my = 2 * (size_t)ny, mz = 2 * (size_t)nz;
    const size_t total = mx * my * mz;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < total; q += (size_t)gridDim.x * blockDim.x) {
        const long long i = q % mx, r = q / mx, j = r % my, k = r / my;
        const double dx = (double)(i < nx ? i : i - (long long)mx);
        const double dy = (double)(j < ny ? j : j - (long long)my);
        const double dz = (double)(k < nz ? k : k - (long long)mz);
        const double r2 = dx * dx + dy * dy + dz * dz;
        K[q] = r2 == 0.0 ? kself / h : 1.0 / (h * sqrt(r2));
    }
}

__global__ void __launch_bounds__(256)
k_iso_take_real(size_t total, const double2* __restrict__ spec, double* __restrict__ out) {
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < total; q += (size_t)gridDim.x * blockDim.x)
        out[q] = spec[q].x;
}

static unsigned grid_for(size_t n) {
    size_t b = (n + 255) / 256;
    const size_t cap = 148 * 32;
    return (unsigned)(b > cap ? cap : (b ? b : 1));
}

static void fill_twiddles(std::vector<double>& w, int n) {
    w.resize(2 * (size_t)n);
    for (int k = 0; k < n; ++k) {
        const long double a = 2.0L * 3.14159265358979323846264338327950288L * (long double)k / (long double)n;
        w[2 * k] = (double)cosl(a);
        w[2 * k + 1] = (double)-sinl(a);
    }
}

int iso_pruned_setup(gp_ctx* c) {
    const int nx = c->g.nx, ny = c->g.ny, nz = c->g.nz;
    const int nxp = (int)iso_nxp(&c->g);
    const long long rowsB = 2LL * ny * nxp;
    std::vector<double> w;
    fill_twiddles(w, 2 * ny);
    GP_CUDA(cudaMemcpyAsync(c->itwy, w.data(), w.size() * sizeof(double), cudaMemcpyHostToDevice, c->stream));
    GP_CUDA(cudaStreamSynchronize(c->stream));
    fill_twiddles(w, 2 * nz);
    GP_CUDA(cudaMemcpyAsync(c->itwz, w.data(), w.size() * sizeof(double), cudaMemcpyHostToDevice, c->stream));
    GP_CUDA(cudaStreamSynchronize(c->stream));

    int n[1] = {2 * nx}, rembed[1] = {2 * nx}, cembed[1] = {nxp};
    // the pad columns nx+1 .. nxp-1 of A are never written by cuFFT: keep them finite
    GP_CUDA(cudaMemsetAsync(c->isoA, 0, (size_t)(nz + 2) * (ny + 2) * nxp * sizeof(double2), c->stream));
    GP_CUFFT(cufftPlanMany(&c->plan_fwd, 1, n, rembed, 1, 2 * nx, cembed, 1, nxp, CUFFT_D2Z, nz * ny));
    if (cufftPlanMany(&c->plan_inv, 1, n, cembed, 1, nxp, rembed, 1, 2 * nx, CUFFT_Z2D, (nz + 2) * (ny + 2)) != CUFFT_SUCCESS) {
        cufftDestroy(c->plan_fwd);
        set_error("isolated solve: cufftPlanMany (inverse x lines) failed");
        return GP_ERR_CUFFT;
    }
    // From here on every failure destroys both plans, and fft_ready is set only once the kernel spectrum
    // exists: a retry after a failed set-up repeats it instead of convolving with a zero spectrum.
    auto fail = [&](int code) { cufftDestroy(c->plan_fwd); cufftDestroy(c->plan_inv); return code; };
    if (cufftSetStream(c->plan_fwd, c->stream) != CUFFT_SUCCESS || cufftSetStream(c->plan_inv, c->stream) != CUFFT_SUCCESS) {
        set_error("isolated solve: cufftSetStream failed");
        return fail(GP_ERR_CUFFT);
    }

    // kernel spectrum, once, through the same forward pipeline (unpruned: the kernel fills the padded grid)
    const size_t full = 8 * c->N, spec = (size_t)(2 * nz) * rowsB;
    double* Kfull = nullptr;
    double2* T = nullptr;
    cudaError_t e = cudaMalloc(&Kfull, full * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc(&T, spec * sizeof(double2));
    if (e != cudaSuccess) {
        cudaFree(Kfull);
        set_error("isolated solve: %zu bytes of set-up scratch: %s", full * sizeof(double) + spec * sizeof(double2), cudaGetErrorString(e));
        return fail(GP_ERR_ALLOC);
    }
    cufftHandle plan_k;
    int rc = GP_OK;
    do {
        if (cufftPlanMany(&plan_k, 1, n, rembed, 1, 2 * nx, cembed, 1, nxp, CUFFT_D2Z, 4 * nz * ny) != CUFFT_SUCCESS) {
            set_error("isolated solve: cufftPlanMany for the kernel spectrum failed");
            rc = GP_ERR_CUFFT;
            break;
        }
        cufftSetStream(plan_k, c->stream);
        const double s3 = std::sqrt(3.0), pi = 3.14159265358979323846;
        const double kself = 3.0 * std::log((s3 + 1.0) / (s3 - 1.0)) - pi / 2.0;
        cudaMemsetAsync(T, 0, spec * sizeof(double2), c->stream);
        k_iso_kernel_fill<<<grid_for(full), 256, 0, c->stream>>>(nx, ny, nz, c->g.h, kself, Kfull);
        if (cufftExecD2Z(plan_k, Kfull, (cufftDoubleComplex*)T) != CUFFT_SUCCESS) { set_error("isolated solve: kernel D2Z failed"); rc = GP_ERR_CUFFT; }
        ColArgs a{};
        a.in = T; a.out = T; a.nkeep = -1; a.scale = 1.0;
        a.in_rs = a.out_rs = nxp; a.in_ss = a.out_ss = rowsB; a.nin = 2 * ny;
        if (rc == GP_OK) rc = launch_col(c, 2 * ny, COL_FWD, a, 2 * nz, nxp, (const double2*)c->itwy);
        a.in_rs = a.out_rs = rowsB; a.in_ss = a.out_ss = 0; a.nin = 2 * nz;
        if (rc == GP_OK) rc = launch_col(c, 2 * nz, COL_FWD, a, 1, rowsB, (const double2*)c->itwz);
        k_iso_take_real<<<grid_for(spec), 256, 0, c->stream>>>(spec, T, c->kspec);
        c->n_own += 4; c->n_fft += 1;
        const cudaError_t es = cudaStreamSynchronize(c->stream);
        if (rc == GP_OK && es != cudaSuccess) { set_error("isolated solve: building the kernel spectrum: %s", cudaGetErrorString(es)); rc = GP_ERR_CUDA; }
        cufftDestroy(plan_k);
    } while (0);
    cudaFree(Kfull);
    cudaFree(T);
    if (rc != GP_OK) return fail(rc);
    c->fft_ready = true;
    return GP_OK;
}

int iso_pruned_solve(gp_ctx* c) {
    const int nx = c->g.nx, ny = c->g.ny, nz = c->g.nz;
    const int nxp = (int)iso_nxp(&c->g);
    const long long rowsB = 2LL * ny * nxp;
    const double* rho = (c->g.components & GP_GAS) ? c->U[GP_RHO] : nullptr;
    const double* n = (c->g.components & GP_STARS) ? c->U[GP_N] : nullptr;
    double2* A = (double2*)c->isoA;
    double2* B = (double2*)c->spec;
    int rc;
    tic(c, K_PAD_SOURCE);
    k_iso_pad_x<<<grid_for((size_t)2 * c->N), 256, 0, c->stream>>>(nx, (size_t)ny * nz, rho, n, c->g.h * c->g.h * c->g.h, c->padded);
    toc(c);
    tic(c, K_FFT_FWD);
    GP_CUFFT(cufftExecD2Z(c->plan_fwd, c->padded, (cufftDoubleComplex*)A));
    toc(c);
    ColArgs a{};
    a.nkeep = -1; a.scale = 1.0;
    a.in = A; a.in_rs = nxp; a.in_ss = (long long)ny * nxp; a.nin = ny;
    a.out = B; a.out_rs = nxp; a.out_ss = rowsB;
    tic(c, K_ISO_YFWD);
    rc = launch_col(c, 2 * ny, COL_FWD, a, nz, nxp, (const double2*)c->itwy);
    toc(c);
    if (rc != GP_OK) return rc;
    a.in = B; a.out = B; a.in_rs = a.out_rs = rowsB; a.in_ss = a.out_ss = 0; a.nin = nz; a.nkeep = nz;
    a.table = c->kspec; a.tab_rs = rowsB; a.scale = -c->g.G / (8.0 * (double)c->N);
    tic(c, K_ISO_ZFUSED);
    rc = launch_col(c, 2 * nz, COL_FUSED, a, 1, rowsB, (const double2*)c->itwz);
    toc(c);
    if (rc != GP_OK) return rc;
    a.table = nullptr; a.scale = 1.0;
    a.in = B; a.in_rs = nxp; a.in_ss = rowsB; a.nin = 2 * ny;
    a.out = A; a.out_rs = nxp; a.out_ss = (long long)(ny + 2) * nxp; a.nkeep = ny;
    tic(c, K_ISO_YINV);
    rc = launch_col(c, 2 * ny, COL_INV, a, nz + 2, nxp, (const double2*)c->itwy);
    toc(c);
    if (rc != GP_OK) return rc;
    tic(c, K_FFT_INV);
    GP_CUFFT(cufftExecZ2D(c->plan_inv, (cufftDoubleComplex*)A, c->padded));
    toc(c);
    tic(c, K_EXTRACT);
    k_iso_extract<<<grid_for(c->N), 256, 0, c->stream>>>(nx, ny, nz, c->padded, phi_interior(c), phi_pitch(nx), ny + 4);
    toc(c);
    c->n_own += 5; c->n_fft += 2;
    GP_CUDA(cudaGetLastError());
    // layer 2, edges and corners: never used by a result (outflow hydro boundaries), kept finite
    return launch_phi_ghost_bc(c, GP_BC_OUTFLOW, GP_BC_OUTFLOW, GP_BC_OUTFLOW, true);
}

}  // namespace gp
