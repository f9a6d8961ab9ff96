// gp_kappa_noalloc (include/gpupegas.h): the correctness check kappa of PAPER.md:198-200 for callers who cannot
// let this library take device memory.
//
// Who that is.  A solver that has sized its grids to fill the card, or a PyTorch program whose caching allocator
// has been handed (nearly) all of HBM, has nothing left for a cudaMalloc issued from inside a library: the call
// fails, or succeeds only by pushing the owner of the memory into an out-of-memory error later.  A time loop that
// keeps several streams busy cannot afford one either, since cudaMalloc and cudaFree make the whole device wait.
// And a tool that only holds field arrays of its own (a snapshot some other code left on the device) should not
// have to build a gp_ctx, whose storage is about twice the state, just to evaluate two sums.  gp_kappa needs such
// a context; this entry point needs none: it reads the caller's arrays where they are and writes two doubles.
//
// How.  The reduction is the two-level, fixed-order sum of od.cu (one partial pair per block, then one block adds
// the partials), on plain unit-stride fields.  The partial sums are the only memory the kernels touch beyond their
// inputs and outputs, and they live in the file-scope __device__ array below instead of in allocated storage.  The
// array belongs to the loaded library: every GPU that loads libgpupegas.so carries its 512 KiB until the process
// exits, and every call on that GPU uses the same 512 KiB.
//
// In host code the name of a __device__ array is only a handle for the runtime, not an address a kernel can use,
// so the host asks the runtime for the device address (cudaGetSymbolAddress) once per device, with that device
// current, and hands that pointer to the kernels.
#include <mutex>

#include "gp_internal.h"

namespace gp {
namespace {

constexpr int NA_THREADS = 256;
constexpr int NA_CELLS_PER_BLOCK = 4096;                  // 16 cells per thread: one partial pair per 4096 cells
constexpr size_t NA_MAX_BLOCKS = (size_t)GP_KAPPA_NOALLOC_MAX_CELLS / NA_CELLS_PER_BLOCK;   // 32768
static_assert((size_t)GP_KAPPA_NOALLOC_MAX_CELLS % NA_CELLS_PER_BLOCK == 0, "the limit is a whole number of blocks");

// [2 b] = gas partial of block b, [2 b + 1] = collisionless partial of block b.  512 KiB.
static __device__ __align__(256) double g_na_partials[2 * NA_MAX_BLOCKS];

constexpr int NA_MAX_DEVICES = 64;
std::mutex g_na_mutex;
double* g_na_ptr[NA_MAX_DEVICES] = {};                    // device address of g_na_partials, per device ordinal

struct NaFields {
    const double* g[6];     // rho, rho v (3), rho E, rho eps                       (g[0] null: no gas)
    const double* b[16];    // n, n u (3), n E_ij (6), Pi_ij (6), xx xy xz yy yz zz (b[0] null: no collisionless part)
};

__device__ __forceinline__ constexpr int na_sym(int i, int j) {
    return i == 0 ? j : (j == 0 ? i : (i == 1 ? (j == 1 ? 3 : 4) : (j == 1 ? 4 : 5)));
}

// Block b owns cells [4096 b, 4096 (b + 1)); a thread adds its cells in ascending order, the block adds its
// threads by a fixed tree: the partial does not depend on the scheduling.  Every block writes its slot, also when
// its sums are zero, so nothing of an earlier call is left in the slots the second kernel reads.
__global__ void __launch_bounds__(NA_THREADS) k_kappa_na_partial(size_t N, NaFields F, double* __restrict__ part) {
    double kg = 0.0, kb = 0.0;
    const size_t c0 = (size_t)blockIdx.x * NA_CELLS_PER_BLOCK;
    const size_t c1 = c0 + NA_CELLS_PER_BLOCK < N ? c0 + NA_CELLS_PER_BLOCK : N;
    for (size_t c = c0 + threadIdx.x; c < c1; c += NA_THREADS) {
        if (F.g[0]) {
            const double rho = F.g[0][c];
            double v2 = 0.0;
#pragma unroll
            for (int d = 0; d < 3; ++d) { const double v = F.g[1 + d][c] / rho; v2 += v * v; }
            kg += fabs(F.g[4][c] - F.g[5][c] - 0.5 * rho * v2);
        }
        if (F.b[0]) {
            const double n = F.b[0][c];
            double u[3];
#pragma unroll
            for (int d = 0; d < 3; ++d) u[d] = F.b[1 + d][c] / n;
#pragma unroll
            for (int i = 0; i < 3; ++i)
#pragma unroll
                for (int j = i; j < 3; ++j)
                    kb += fabs(F.b[4 + na_sym(i, j)][c] - F.b[10 + na_sym(i, j)][c] - n * u[i] * u[j]);
        }
    }
    __shared__ double sg[NA_THREADS], sb[NA_THREADS];
    sg[threadIdx.x] = kg; sb[threadIdx.x] = kb;
    __syncthreads();
    for (int o = NA_THREADS / 2; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) { sg[threadIdx.x] += sg[threadIdx.x + o]; sb[threadIdx.x] += sb[threadIdx.x + o]; }
        __syncthreads();
    }
    if (threadIdx.x == 0) { part[2 * (size_t)blockIdx.x] = sg[0]; part[2 * (size_t)blockIdx.x + 1] = sb[0]; }
}

// One block adds the nb partial pairs of this call (and only those) in a fixed order.
__global__ void __launch_bounds__(NA_THREADS) k_kappa_na_final(int nb, const double* __restrict__ part, double h3,
                                                               double* __restrict__ out) {
    __shared__ double sg[NA_THREADS], sb[NA_THREADS];
    double kg = 0.0, kb = 0.0;
    for (int i = threadIdx.x; i < nb; i += NA_THREADS) { kg += part[2 * i]; kb += part[2 * i + 1]; }
    sg[threadIdx.x] = kg; sb[threadIdx.x] = kb;
    __syncthreads();
    for (int o = NA_THREADS / 2; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) { sg[threadIdx.x] += sg[threadIdx.x + o]; sb[threadIdx.x] += sb[threadIdx.x + o]; }
        __syncthreads();
    }
    if (threadIdx.x == 0) { out[0] = sg[0] * h3; out[1] = sb[0] * h3; }
}

// Device address of the partial-sum array on the current device; looked up at the first call on that device.
int na_scratch(double** out) {
    int dev = -1;
    GP_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= NA_MAX_DEVICES) {
        set_error("gp_kappa_noalloc: device ordinal %d outside [0, %d)", dev, NA_MAX_DEVICES);
        return GP_ERR_UNSUPPORTED;
    }
    std::lock_guard<std::mutex> lock(g_na_mutex);
    if (!g_na_ptr[dev]) {
        double* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void**)&p, g_na_partials);
        if (e != cudaSuccess || !p) {
            set_error("gp_kappa_noalloc: cudaGetSymbolAddress of the partial-sum array failed on device %d: %s", dev,
                      cudaGetErrorString(e));
            return GP_ERR_CUDA;
        }
        g_na_ptr[dev] = p;
    }
    *out = g_na_ptr[dev];
    return GP_OK;
}

}  // namespace
}  // namespace gp

extern "C" int gp_kappa_noalloc(size_t n_cells, double h, const double* const* gas, const double* const* stars,
                                double* out_device, void* cuda_stream) {
    using namespace gp;
    if (n_cells == 0) { set_error("gp_kappa_noalloc: n_cells is 0"); return GP_ERR_ARG; }
    if (n_cells > (size_t)GP_KAPPA_NOALLOC_MAX_CELLS) {
        set_error("gp_kappa_noalloc: %zu cells exceed the limit of %zu cells (GP_KAPPA_NOALLOC_MAX_CELLS) that the "
                  "library's fixed partial-sum array is sized for; use gp_kappa on a context, or call per slab and add",
                  n_cells, (size_t)GP_KAPPA_NOALLOC_MAX_CELLS);
        return GP_ERR_ARG;
    }
    if (!out_device || (!gas && !stars)) { set_error("gp_kappa_noalloc: NULL output, or neither component given"); return GP_ERR_ARG; }
    if (!(h > 0.0)) { set_error("gp_kappa_noalloc: h must be positive"); return GP_ERR_ARG; }
    NaFields F;
    for (int f = 0; f < 6; ++f) {
        F.g[f] = gas ? gas[f] : nullptr;
        if (gas && !gas[f]) { set_error("gp_kappa_noalloc: gas[%d] is NULL", f); return GP_ERR_ARG; }
    }
    for (int f = 0; f < 16; ++f) {
        F.b[f] = stars ? stars[f] : nullptr;
        if (stars && !stars[f]) { set_error("gp_kappa_noalloc: stars[%d] is NULL", f); return GP_ERR_ARG; }
    }
    double* part = nullptr;
    const int rc = na_scratch(&part);
    if (rc != GP_OK) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const unsigned nb = (unsigned)((n_cells + NA_CELLS_PER_BLOCK - 1) / NA_CELLS_PER_BLOCK);
    k_kappa_na_partial<<<nb, NA_THREADS, 0, st>>>(n_cells, F, part);
    k_kappa_na_final<<<1, NA_THREADS, 0, st>>>((int)nb, part, h * h * h, out_device);
    GP_CUDA(cudaGetLastError());
    return GP_OK;
}
