// C ABI of libgpupegas.so (include/gpupegas.h): context, storage, field copies, and the
// sequencing of the kernels of one timestep.  No torch types, no CPU fallback.
#include <cstdarg>
#include <cstring>
#include <new>

#include "gp_internal.h"

namespace gp {

static thread_local char g_err[512] = "";

void set_error(const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}

static inline size_t align256(size_t b) { return (b + 255) & ~(size_t)255; }

static const char* const kKernelNames[K_NUM] = {
    "cfl", "poisson_source", "cufft_forward",
    "poisson_green", "cufft_inverse", "phi_ghost", "poisson_pad_source", "poisson_mul_kernel", "poisson_extract",
    "hydro_gas_fused", "hydro_bme_fused", "poisson_zpass_green", "poisson_iso_yfwd", "poisson_iso_zfused",
    "poisson_iso_yinv", "od_cell_local"};

void tic(gp_ctx* c, int kid) {
    Timing* t = c->tim;
    if (!t || !t->on) return;
    if (t->used == t->cap) {
        const size_t ncap = t->cap ? 2 * t->cap : 256;
        cudaEvent_t* ev = new cudaEvent_t[2 * ncap];
        int* kd = new int[ncap];
        for (size_t i = 0; i < 2 * t->cap; ++i) ev[i] = t->ev[i];
        for (size_t i = 0; i < t->cap; ++i) kd[i] = t->kid[i];
        for (size_t i = 2 * t->cap; i < 2 * ncap; ++i) cudaEventCreate(&ev[i]);
        delete[] t->ev; delete[] t->kid;
        t->ev = ev; t->kid = kd; t->cap = ncap;
    }
    t->kid[t->used] = kid;
    cudaEventRecord(t->ev[2 * t->used], c->stream);
}

void toc(gp_ctx* c) {
    Timing* t = c->tim;
    if (!t || !t->on) return;
    cudaEventRecord(t->ev[2 * t->used + 1], c->stream);
    t->used++;
}

static void timing_collect(gp_ctx* c) {
    Timing* t = c->tim;
    if (!t) return;
    cudaStreamSynchronize(c->stream);
    for (size_t i = 0; i < t->used; ++i) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, t->ev[2 * i], t->ev[2 * i + 1]) == cudaSuccess) {
            t->ms[t->kid[i]] += ms;
            t->cnt[t->kid[i]]++;
        }
    }
    t->used = 0;
}

static bool field_enabled(const gp_grid& g, int f) {
    if (f == GP_PHI) return true;
    if (f < 0 || f >= GP_NFIELDS_OD) return false;
    if (f >= GP_EPS) {
        if (!(g.components & GP_OD)) return false;
        return f == GP_EPS ? (g.components & GP_GAS) != 0 : (g.components & GP_STARS) != 0;
    }
    return f < NGAS ? (g.components & GP_GAS) != 0 : (g.components & GP_STARS) != 0;
}

// Carried fields of a GP_OD context that do not follow the conserved ones (bit f - F_EPS per internal field f).
// A carried field goes stale when a conserved field of its component is written through gp_set_state, and is fresh
// again once gp_od_derive has run or the field itself has been set.  While any bit is set, gp_step / gp_od_step,
// gp_max_dt and gp_od_balance refuse (GP_ERR_STATE): a step would otherwise run on the pressure of another state
// (or on p = 0 of fresh storage) and the balance would then overwrite the evidence.
static unsigned od_all_stale(const gp_grid& g) {
    if (!(g.components & GP_OD)) return 0u;
    unsigned m = 0u;
    if (g.components & GP_GAS) m |= 1u;                      // rho*eps
    if (g.components & GP_STARS) m |= 0x3fu << 1;            // Pi_xx ... Pi_zz
    return m;
}
static int od_check_fresh(const gp_ctx* c, const char* who) {
    if (!c->od_stale) return GP_OK;
    set_error("%s: the carried fields (rho*eps / Pi_ij) of this GP_OD context do not follow the conserved fields that were "
              "set since (stale mask 0x%x): call gp_od_derive, or set them with gp_set_state(GP_EPS ... GP_PZZ)", who, c->od_stale);
    return GP_ERR_STATE;
}

static size_t storage_bytes(const gp_grid& g) {
    const size_t N = (size_t)g.nx * g.ny * g.nz;
    const size_t fb = align256(N * sizeof(double));
    size_t nf = 0;
    const bool od = (g.components & GP_OD) != 0;
    if (g.components & GP_GAS) nf += NGAS + (od ? NODG : 0);
    if (g.components & GP_STARS) nf += NBME + (od ? NODB : 0);
    size_t b = 2 * nf * fb + 64 * 256;                // U and the step's target (pairs are aligned one by one)
    b += align256(phi_pad_elems(g.nx, g.ny, g.nz) * sizeof(double));   // Phi with two ghost layers
    b += 512;                                         // dt, smax, flag; kappa
    b += poisson_storage_bytes(&g);
    return b;
}

// Carve the bound (or freshly allocated) region.
static int ensure_storage(gp_ctx* c) {
    if (c->ready) return GP_OK;
    const gp_grid& g = c->g;
    const size_t need = storage_bytes(g);
    if (!c->base) {
        void* p = nullptr;
        cudaError_t e = cudaMalloc(&p, need);
        if (e != cudaSuccess) {
            set_error("cudaMalloc of %zu bytes failed: %s", need, cudaGetErrorString(e));
            return GP_ERR_ALLOC;
        }
        c->base = (char*)p;
        c->bytes = need;
        c->owns = true;
    } else if (c->bytes < need) {
        set_error("bound storage too small: %zu < %zu", c->bytes, need);
        return GP_ERR_ARG;
    }
    char* p = c->base;
    auto take = [&](size_t bytes) { char* r = p; p += align256(bytes); return r; };
    const size_t N = c->N;
    for (int f = 0; f < NALL; ++f) c->U[f] = c->Us[f] = nullptr;
    c->od = (g.components & GP_OD) != 0;
    c->estr = c->od ? BSTR : 1;
    auto take_pair = [&](int f0, int f1) {            // one double2 per cell (gp_internal.h, BSTR)
        double* u = (double*)take(2 * N * sizeof(double));
        double* us = (double*)take(2 * N * sizeof(double));
        c->U[f0] = u; c->U[f1] = u + 1;
        c->Us[f0] = us; c->Us[f1] = us + 1;
    };
    if (c->od) {
        if (g.components & GP_GAS) take_pair(NGAS - 1, F_EPS);                      // (rho E, rho eps)
        if (g.components & GP_STARS) for (int P = 0; P < NODB / 2; ++P) take_pair(F_PI + 2 * P, F_PI + 2 * P + 1);
    }
    if (g.components & GP_GAS) {
        for (int P = 0; P < NGASP / 2; ++P) {     // (rho,m_x) (m_y,m_z): one double2 per cell (gp_internal.h, BSTR)
            double* u = (double*)take(2 * N * sizeof(double));
            double* us = (double*)take(2 * N * sizeof(double));
            c->U[2 * P] = u; c->U[2 * P + 1] = u + 1;
            c->Us[2 * P] = us; c->Us[2 * P + 1] = us + 1;
        }
        if (!c->od) {
            c->U[GP_E] = (double*)take(N * sizeof(double));
            c->Us[GP_E] = (double*)take(N * sizeof(double));
        }
    }
    if (g.components & GP_STARS)
        for (int P = 0; P < NBME / 2; ++P) {      // pairs of fields, one double2 per cell (gp_internal.h, BSTR)
            double* u = (double*)take(2 * N * sizeof(double));
            double* us = (double*)take(2 * N * sizeof(double));
            c->U[NGAS + 2 * P] = u; c->U[NGAS + 2 * P + 1] = u + 1;
            c->Us[NGAS + 2 * P] = us; c->Us[NGAS + 2 * P + 1] = us + 1;
        }
    c->phip = (double*)take(phi_pad_elems(g.nx, g.ny, g.nz) * sizeof(double)) + (PHI_XOFF - 2);   // interior rows 128-byte aligned
    c->d_kappa = (double*)take(256);
    c->kappa_cached = false;
    c->od_stale = od_all_stale(c->g);
    char* small = take(256);
    c->d_dt = (double*)small;
    c->d_smax = (unsigned long long*)(small + 64);
    c->d_flag = (int*)(small + 128);
    c->d_smax_next = (unsigned long long*)(small + 160);
    c->d_flag_next = (int*)(small + 192);
    c->cfl_cached = false;
    c->spec = nullptr; c->padded = nullptr; c->kspec = nullptr; c->tabx = c->taby = c->tabz = nullptr;
    c->ztw = nullptr; c->src = nullptr; c->src_cached = false;
    c->isofast = false; c->isoA = c->itwy = c->itwz = nullptr;
    if (g.poisson == GP_POISSON_PERIODIC) {
        c->spec = (cufftDoubleComplex*)take(((size_t)g.nx / 2 + 1) * g.ny * g.nz * sizeof(cufftDoubleComplex));
        c->tabx = (double*)take(((size_t)g.nx + g.ny + g.nz) * sizeof(double));
        c->taby = c->tabx + g.nx;
        c->tabz = c->taby + g.ny;
        c->ztw = (double*)take(2 * (size_t)g.nz * sizeof(double));
        c->src = (double*)take(N * sizeof(double));   // rho + n (the densities are paired in the state)
    } else if (g.poisson == GP_POISSON_ISOLATED && iso_pruned_supported(&g)) {
        const size_t nxp = ((size_t)g.nx + 1 + 7) & ~(size_t)7, ny = g.ny, nz = g.nz;
        c->isofast = true;
        c->padded = (double*)take((nz + 2) * (ny + 2) * 2 * (size_t)g.nx * sizeof(double));
        c->isoA = (double*)take((nz + 2) * (ny + 2) * nxp * 2 * sizeof(double));
        c->spec = (cufftDoubleComplex*)take((nz + 2) * 2 * ny * nxp * sizeof(cufftDoubleComplex));
        c->kspec = (double*)take(2 * nz * 2 * ny * nxp * sizeof(double));
        c->itwy = (double*)take(2 * ny * 2 * sizeof(double));
        c->itwz = (double*)take(2 * nz * 2 * sizeof(double));
    } else if (g.poisson == GP_POISSON_ISOLATED) {
        const size_t half = ((size_t)g.nx + 1) * (2 * (size_t)g.ny) * (2 * (size_t)g.nz);
        c->spec = (cufftDoubleComplex*)take(half * sizeof(cufftDoubleComplex));
        c->kspec = (double*)take(half * sizeof(double));
        c->padded = (double*)take(8 * N * sizeof(double));
    }
    if ((size_t)(p - c->base) > c->bytes) {
        set_error("internal: storage layout (%zu) exceeds the region (%zu)", (size_t)(p - c->base), c->bytes);
        return GP_ERR_ALLOC;
    }
    // zero state, Phi and its ghost faces (GP_POISSON_NONE with Phi never set means no gravity)
    GP_CUDA(cudaMemsetAsync(c->base, 0, (size_t)(p - c->base), c->stream));
    c->ready = true;
    return GP_OK;
}

// Copy Phi between a plain nx*ny*nz array (host or device) and the interior of the padded array.
static int copy_phi(gp_ctx* c, double* plain, bool on_device, bool to_ctx) {
    const gp_grid& g = c->g;
    cudaMemcpy3DParms p = {};
    const cudaPitchedPtr pad = make_cudaPitchedPtr(c->phip, (size_t)phi_pitch(g.nx) * sizeof(double), (size_t)phi_pitch(g.nx), (size_t)g.ny + 4);
    const cudaPitchedPtr lin = make_cudaPitchedPtr(plain, (size_t)g.nx * sizeof(double), (size_t)g.nx, (size_t)g.ny);
    const cudaPos in = make_cudaPos(2 * sizeof(double), 2, 2), zero = make_cudaPos(0, 0, 0);
    p.srcPtr = to_ctx ? lin : pad; p.srcPos = to_ctx ? zero : in;
    p.dstPtr = to_ctx ? pad : lin; p.dstPos = to_ctx ? in : zero;
    p.extent = make_cudaExtent((size_t)g.nx * sizeof(double), (size_t)g.ny, (size_t)g.nz);
    p.kind = on_device ? cudaMemcpyDeviceToDevice : (to_ctx ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToHost);
    GP_CUDA(cudaMemcpy3DAsync(&p, c->stream));
    if (!on_device) GP_CUDA(cudaStreamSynchronize(c->stream));
    return GP_OK;
}

}  // namespace gp

using namespace gp;

extern "C" {

const char* gp_last_error(void) { return g_err; }

gp_ctx* gp_create(const gp_grid* grid, double gamma, const gp_bc* bc) {
    if (!grid || !bc) { set_error("gp_create: NULL argument"); return nullptr; }
    if (grid->nx < 4 || grid->ny < 4 || grid->nz < 4 || !(grid->h > 0.0)) {
        set_error("gp_create: need nx, ny, nz >= 4 and h > 0");
        return nullptr;
    }
    if (!(grid->components & (GP_GAS | GP_STARS)) || (grid->components & ~(GP_GAS | GP_STARS | GP_OD))) {
        set_error("gp_create: components must be GP_GAS, GP_STARS or both, optionally with GP_OD");
        return nullptr;
    }
    if (grid->poisson < GP_POISSON_NONE || grid->poisson > GP_POISSON_ISOLATED) { set_error("gp_create: bad poisson mode"); return nullptr; }
    if (grid->poisson != GP_POISSON_NONE && ((grid->nx | grid->ny | grid->nz) & 1)) {
        set_error("gp_create: Poisson modes need even nx, ny, nz");
        return nullptr;
    }
    const int b[3] = {bc->x, bc->y, bc->z};
    for (int d = 0; d < 3; ++d)
        if (b[d] != GP_BC_PERIODIC && b[d] != GP_BC_OUTFLOW) { set_error("gp_create: bad boundary code"); return nullptr; }
    if (grid->poisson == GP_POISSON_ISOLATED && (b[0] != GP_BC_OUTFLOW || b[1] != GP_BC_OUTFLOW || b[2] != GP_BC_OUTFLOW)) {
        set_error("gp_create: the isolated Poisson mode needs outflow hydro boundaries on every axis");
        return nullptr;
    }
    if (!(gamma > 1.0)) { set_error("gp_create: gamma must exceed 1"); return nullptr; }
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev < 1) {
        set_error("gp_create: no CUDA device (%s); this library has no CPU path", cudaGetErrorString(e));
        return nullptr;
    }
    gp_ctx* c = new (std::nothrow) gp_ctx;
    if (!c) { set_error("gp_create: out of host memory"); return nullptr; }
    std::memset((void*)c, 0, sizeof(*c));
    c->g = *grid;
    c->gamma = gamma;
    c->bc = *bc;
    c->N = (size_t)grid->nx * grid->ny * grid->nz;
    c->stream = nullptr;
    return c;
}

void gp_destroy(gp_ctx* c) {
    if (!c) return;
    if (c->ready || c->fft_ready) cudaStreamSynchronize(c->stream);
    poisson_teardown(c);
    if (c->owns && c->base) cudaFree(c->base);
    delete c->tmc[0]; delete c->tmc[1];
    if (c->tim) {
        for (size_t i = 0; i < 2 * c->tim->cap; ++i) cudaEventDestroy(c->tim->ev[i]);
        delete[] c->tim->ev; delete[] c->tim->kid;
        delete c->tim;
    }
    delete c;
}

int gp_set_stream(gp_ctx* c, void* stream) {
    if (!c) { set_error("gp_set_stream: NULL context"); return GP_ERR_ARG; }
    if (c->ready) GP_CUDA(cudaStreamSynchronize(c->stream));
    c->stream = (cudaStream_t)stream;
    if (c->fft_ready) {
        GP_CUFFT(cufftSetStream(c->plan_fwd, c->stream));
        GP_CUFFT(cufftSetStream(c->plan_inv, c->stream));
    }
    return GP_OK;
}

size_t gp_storage_bytes(const gp_grid* grid) {
    if (!grid) return 0;
    return storage_bytes(*grid);
}

int gp_bind_storage(gp_ctx* c, void* device_ptr, size_t bytes) {
    if (!c || !device_ptr) { set_error("gp_bind_storage: NULL argument"); return GP_ERR_ARG; }
    if (c->ready || c->base) { set_error("gp_bind_storage: storage already in use"); return GP_ERR_ARG; }
    if (((size_t)device_ptr & 255) != 0) { set_error("gp_bind_storage: pointer must be 256-byte aligned"); return GP_ERR_ARG; }
    if (bytes < storage_bytes(c->g)) { set_error("gp_bind_storage: %zu bytes given, %zu needed", bytes, storage_bytes(c->g)); return GP_ERR_ARG; }
    c->base = (char*)device_ptr;
    c->bytes = bytes;
    c->owns = false;
    return GP_OK;
}

int gp_synchronize(gp_ctx* c) {
    if (!c) { set_error("gp_synchronize: NULL context"); return GP_ERR_ARG; }
    GP_CUDA(cudaStreamSynchronize(c->stream));
    return GP_OK;
}

int gp_launch_counts(gp_ctx* c, long long* own, long long* fft) {
    if (!c) { set_error("gp_launch_counts: NULL context"); return GP_ERR_ARG; }
    if (own) *own = c->n_own;
    if (fft) *fft = c->n_fft;
    return GP_OK;
}

int gp_timing_enable(gp_ctx* c, int on) {
    if (!c) { set_error("gp_timing_enable: NULL context"); return GP_ERR_ARG; }
    if (!c->tim) c->tim = new (std::nothrow) Timing;
    if (!c->tim) { set_error("gp_timing_enable: out of host memory"); return GP_ERR_ALLOC; }
    timing_collect(c);
    if (on && !c->tim->on) {
        for (int k = 0; k < K_NUM; ++k) { c->tim->ms[k] = 0.0; c->tim->cnt[k] = 0; }
    }
    c->tim->on = on != 0;
    return GP_OK;
}

int gp_timing_read(gp_ctx* c, int max_entries, int* n_entries, const char** names, double* total_ms, long long* launches) {
    if (!c || !n_entries) { set_error("gp_timing_read: NULL argument"); return GP_ERR_ARG; }
    *n_entries = 0;
    if (!c->tim) return GP_OK;
    timing_collect(c);
    int n = 0;
    for (int k = 0; k < K_NUM && n < max_entries; ++k) {
        if (!c->tim->cnt[k]) continue;
        if (names) names[n] = kKernelNames[k];
        if (total_ms) total_ms[n] = c->tim->ms[k];
        if (launches) launches[n] = c->tim->cnt[k];
        ++n;
    }
    *n_entries = n;
    return GP_OK;
}

int gp_set_state(gp_ctx* c, int field, const double* src, int on_device) {
    if (!c || !src) { set_error("gp_set_state: NULL argument"); return GP_ERR_ARG; }
    if (!field_enabled(c->g, field)) { set_error("gp_set_state: field %d is not enabled", field); return GP_ERR_ARG; }
    int rc = ensure_storage(c);
    if (rc != GP_OK) return rc;
    if (field == GP_PHI) {
        if ((rc = copy_phi(c, const_cast<double*>(src), on_device != 0, true)) != GP_OK) return rc;
        return launch_phi_ghost_bc(c, c->bc.x, c->bc.y, c->bc.z);
    }
    const int fi = field_index(field);
    double* dst = c->U[fi];
    if (field_paired(fi, c->od)) {
        // paired layout: a host array lands contiguously in the pair's step target (free between steps),
        // then one kernel interleaves it; a device array is interleaved directly
        const double* from = src;
        if (!on_device) {
            double* scratch = c->Us[pair_base(fi)];
            GP_CUDA(cudaMemcpyAsync(scratch, src, c->N * sizeof(double), cudaMemcpyHostToDevice, c->stream));
            GP_CUDA(cudaStreamSynchronize(c->stream));
            from = scratch;
        }
        if ((rc = launch_strided_copy(c, dst, BSTR, from, 1, c->N)) != GP_OK) return rc;
    } else {
        GP_CUDA(cudaMemcpyAsync(dst, src, c->N * sizeof(double), on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, c->stream));
        if (!on_device) GP_CUDA(cudaStreamSynchronize(c->stream));   // the host buffer may be reused on return
    }
    c->cfl_cached = false;
    c->src_cached = false;
    c->kappa_cached = false;
    if (c->od) {
        if (fi >= F_EPS) c->od_stale &= ~(1u << (fi - F_EPS));                  // this carried field is the caller's now
        else c->od_stale |= od_all_stale(c->g) & (fi < NGAS ? 1u : 0x3fu << 1); // its component's carried fields lag
    }
    return GP_OK;
}

int gp_get_state(gp_ctx* c, int field, double* dst, int on_device) {
    if (!c || !dst) { set_error("gp_get_state: NULL argument"); return GP_ERR_ARG; }
    if (!field_enabled(c->g, field)) { set_error("gp_get_state: field %d is not enabled", field); return GP_ERR_ARG; }
    int rc = ensure_storage(c);
    if (rc != GP_OK) return rc;
    if (field == GP_PHI) return copy_phi(c, dst, on_device != 0, false);
    const int fi = field_index(field);
    const double* src = c->U[fi];
    if (field_paired(fi, c->od)) {
        double* scratch = c->Us[pair_base(fi)];
        if ((rc = launch_strided_copy(c, on_device ? dst : scratch, 1, src, BSTR, c->N)) != GP_OK) return rc;
        if (!on_device) {
            GP_CUDA(cudaMemcpyAsync(dst, scratch, c->N * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
            GP_CUDA(cudaStreamSynchronize(c->stream));
        }
        return GP_OK;
    }
    GP_CUDA(cudaMemcpyAsync(dst, src, c->N * sizeof(double), on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, c->stream));
    if (!on_device) GP_CUDA(cudaStreamSynchronize(c->stream));
    return GP_OK;
}

int gp_solve_poisson(gp_ctx* c) {
    if (!c) { set_error("gp_solve_poisson: NULL context"); return GP_ERR_ARG; }
    if (c->g.poisson == GP_POISSON_NONE) { set_error("gp_solve_poisson: context was created with GP_POISSON_NONE"); return GP_ERR_UNSUPPORTED; }
    int rc = ensure_storage(c);
    if (rc != GP_OK) return rc;
    return poisson_solve(c);
}

int gp_max_dt(gp_ctx* c, double cfl, double* dt) {
    if (!c || !(cfl > 0.0)) { set_error("gp_max_dt: bad argument"); return GP_ERR_ARG; }
    int rc = ensure_storage(c);
    if (rc != GP_OK) return rc;
    if (c->od && (rc = od_check_fresh(c, "gp_max_dt")) != GP_OK) return rc;    // reads the carried fields (G16)
    // after a step the fused kernels have already folded the max signal speed of the new state
    rc = c->cfl_cached ? launch_cfl_from_cache(c, cfl) : launch_cfl(c, cfl);
    if (rc != GP_OK) return rc;
    if (dt) {
        double h_dt = 0.0;
        int h_flag = 0;
        GP_CUDA(cudaMemcpyAsync(&h_dt, c->d_dt, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
        GP_CUDA(cudaMemcpyAsync(&h_flag, c->d_flag, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
        GP_CUDA(cudaStreamSynchronize(c->stream));
        *dt = h_dt;
        if (h_flag) { set_error("gp_max_dt: state holds NaN/Inf or a non-positive rho, n, p or Pi_dd"); return GP_ERR_STATE; }
    }
    return GP_OK;
}

// One timestep; od_balance: -1 = plain scheme, 0 / 1 = overdetermined system without / with the energy balance.
static int step_impl(gp_ctx* c, double dt, int od_balance) {
    int rc = ensure_storage(c);
    if (rc != GP_OK) return rc;
    const bool od = od_balance >= 0;
    if (od && (rc = od_check_fresh(c, "gp_step")) != GP_OK) return rc;
    const double* d_dt = dt > 0.0 ? nullptr : c->d_dt;
    if ((rc = launch_cfl_reset_next(c)) != GP_OK) return rc;
    if (od) GP_CUDA(cudaMemsetAsync(c->d_kappa, 0, 2 * sizeof(double), c->stream));
    auto swap = [&](int f) { double* t = c->U[f]; c->U[f] = c->Us[f]; c->Us[f] = t; };
    // With both components and the periodic solve, the source rho + n of the next solve rides in
    // the epilogue of the gas kernel, which therefore runs second (n is then already new).
    c->src_cached = false;
    if (c->g.components & GP_STARS) {
        if ((rc = od ? launch_fused_bme_od(c, dt, d_dt, od_balance) : launch_fused_bme(c, dt, d_dt)) != GP_OK) return rc;
        for (int f = NGAS; f < NHYD; ++f) swap(f);
        if (od) for (int f = F_PI; f < NALL; ++f) swap(f);
    }
    if (c->g.components & GP_GAS) {
        double* src_out = c->src;          // non-null only with the periodic solve
        const double* n_new = (c->g.components & GP_STARS) ? c->U[GP_N] : nullptr;
        if ((rc = od ? launch_fused_gas_od(c, dt, d_dt, src_out ? n_new : nullptr, src_out, od_balance)
                     : launch_fused_gas(c, dt, d_dt, src_out ? n_new : nullptr, src_out)) != GP_OK) return rc;
        for (int f = 0; f < NGAS; ++f) swap(f);
        if (od) swap(F_EPS);
        c->src_cached = src_out != nullptr;
    }
    c->cfl_cached = true;
    c->kappa_cached = od;
    return GP_OK;
}

int gp_step(gp_ctx* c, double dt) {
    if (!c) { set_error("gp_step: NULL context"); return GP_ERR_ARG; }
    if (dt != dt) { set_error("gp_step: dt is NaN"); return GP_ERR_ARG; }
    return step_impl(c, dt, (c->g.components & GP_OD) ? 1 : -1);
}

#define GP_NEED_OD(name)                                                                                  \
    do {                                                                                                  \
        if (!c) { set_error(name ": NULL context"); return GP_ERR_ARG; }                                  \
        if (!(c->g.components & GP_OD)) { set_error(name ": context was created without GP_OD"); return GP_ERR_UNSUPPORTED; } \
    } while (0)

int gp_od_step(gp_ctx* c, double dt, int balance) {
    GP_NEED_OD("gp_od_step");
    if (dt != dt) { set_error("gp_od_step: dt is NaN"); return GP_ERR_ARG; }
    return step_impl(c, dt, balance ? 1 : 0);
}

int gp_od_derive(gp_ctx* c) {
    GP_NEED_OD("gp_od_derive");
    int rc = ensure_storage(c);
    if (rc != GP_OK) return rc;
    c->kappa_cached = false;
    c->od_stale = 0u;
    return launch_od_derive(c);
}

int gp_od_balance(gp_ctx* c) {
    GP_NEED_OD("gp_od_balance");
    int rc = ensure_storage(c);
    if (rc != GP_OK) return rc;
    if ((rc = od_check_fresh(c, "gp_od_balance")) != GP_OK) return rc;
    c->cfl_cached = false;       // the balance may change momenta and energies
    c->kappa_cached = false;
    return launch_od_balance(c);
}

int gp_kappa(gp_ctx* c, double* out) {
    GP_NEED_OD("gp_kappa");
    if (!out) { set_error("gp_kappa: NULL argument"); return GP_ERR_ARG; }
    int rc = ensure_storage(c);
    if (rc != GP_OK) return rc;
    if ((rc = launch_od_kappa(c, c->d_kappa + 2)) != GP_OK) return rc;
    GP_CUDA(cudaMemcpyAsync(out, c->d_kappa + 2, 2 * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    GP_CUDA(cudaStreamSynchronize(c->stream));
    return GP_OK;
}

int gp_od_last_kappa(gp_ctx* c, double* out) {
    GP_NEED_OD("gp_od_last_kappa");
    if (!out) { set_error("gp_od_last_kappa: NULL argument"); return GP_ERR_ARG; }
    if (!c->ready || !c->kappa_cached) { set_error("gp_od_last_kappa: no step has run since the state was last set"); return GP_ERR_STATE; }
    GP_CUDA(cudaMemcpyAsync(out, c->d_kappa, 2 * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    GP_CUDA(cudaStreamSynchronize(c->stream));
    const double h3 = c->g.h * c->g.h * c->g.h;
    out[0] *= h3; out[1] *= h3;
    return GP_OK;
}

int gp_fp64_rate_selftest(double* thread_inst_per_s, double* ms) {
    if (!thread_inst_per_s) { set_error("gp_fp64_rate_selftest: NULL argument"); return GP_ERR_ARG; }
    return fp64_rate_selftest(thread_inst_per_s, ms);
}

int gp_math_selftest(int n, const double* x, double* rcp, double* rsqrt_out) {
    if (n < 1 || !x || !rcp || !rsqrt_out) { set_error("gp_math_selftest: bad argument"); return GP_ERR_ARG; }
    return math_selftest(n, x, rcp, rsqrt_out);
}

}  // extern "C"
