// Fused z pass of the periodic Poisson solve: for every (k_x, k_y) column of the
// half spectrum left by the batched 2-D real transforms, ONE kernel does the forward transform
// along z, the multiplication by the Green factor of the 27-point Laplacian (PAPER.md:190 with
// the sign and k = 0 readings of DESIGN.md G3) and the inverse transform along z, so the spectrum
// crosses HBM once (read + write) instead of three times (cuFFT z pass, multiply, cuFFT z pass).
//
// The transform is a decimation-in-frequency pass (radix 8, with one closing radix 4 or 2 stage
// when log2(nz) is not a multiple of 3) whose output is left in digit-reversed order in
// registers; the inverse is the exact mirror image (conjugate twiddle, conjugate butterfly, in the
// reverse stage order), so no reordering is ever needed: the last forward stage and the first
// inverse stage work on the same register values.  Between stages the columns are exchanged
// through shared memory.  ZC adjacent columns (ZC * 16 B contiguous in HBM) share a block.
#include "fftcol.cuh"

// columns per block and blocks per SM of the 512-point pass (the headline size)
#ifndef GP_ZP9_C
#define GP_ZP9_C 4
#define GP_ZP9_MINB 2
#endif

namespace gp {

// forward stages s..S-1, Green multiply, inverse stages S-1..s (compile-time recursion)
template <int P, int C, int s>
struct ZPipe {
    __device__ static __forceinline__ void run(double2* v, double2* sm, const double2* __restrict__ tw, int t, int col,
                                               double txy, double coef6, const double* __restrict__ tz, bool origin) {
        constexpr int S = ZStages<P>::S;
        zstage<P, s, false>(v, tw, t);
        if constexpr (s + 1 < S) {
            ZExchange<P, C, s>::template run<s + 1>(v, sm, t, col);
            ZPipe<P, C, s + 1>::run(v, sm, tw, t, col, txy, coef6, tz, origin);
            ZExchange<P, C, s + 1>::template run<s>(v, sm, t, col);
        } else {
            // register r = b*R + m holds frequency k_z = sum_s m_s prod_{t<s} R_t of position idx
            constexpr int R = ZStages<P>::radix(s), L = ZStages<P>::len(s);
#pragma unroll
            for (int b = 0; b < 8 / R; ++b)
#pragma unroll
                for (int m = 0; m < R; ++m) {
                    const int pos = zidx<P, R, L>(t, b, m);
                    int kz = 0, w = 1;
#pragma unroll
                    for (int q = 0; q < S; ++q) {
                        const int Rq = ZStages<P>::radix(q), Qq = ZStages<P>::len(q) / Rq;
                        kz += ((pos / Qq) % Rq) * w;
                        w *= Rq;
                    }
                    // coef / (6 (1 - tx ty tz)), zero for the mean mode
                    const double den = fma(-txy, tz[kz], 1.0);
                    const double f = (origin && kz == 0) ? 0.0 : coef6 * zrcp(den);
                    v[b * R + m].x *= f; v[b * R + m].y *= f;
                }
        }
        zstage<P, s, true>(v, tw, t);
    }
};

template <int P, int ZC, int MINB>
__global__ void __launch_bounds__((1 << P) / 8 * ZC, MINB)
k_zpass_green(size_t plane, int nxh, const double* __restrict__ tx, const double* __restrict__ ty,
              const double* __restrict__ tz, const double2* __restrict__ tw, double coef6, double2* __restrict__ spec) {
    extern __shared__ double2 zsm[];
    const int col = threadIdx.x % ZC, t = threadIdx.x / ZC;
    const size_t q = (size_t)blockIdx.x * ZC + col;
    const bool valid = q < plane;
    const size_t qc = valid ? q : plane - 1;
    const int i = (int)(qc % nxh), j = (int)(qc / nxh);
    const double txy = tx[i] * ty[j];
    constexpr int R0 = ZStages<P>::radix(0), L0 = 1 << P;
    double2 v[8];
#pragma unroll
    for (int b = 0; b < 8 / R0; ++b)
#pragma unroll
        for (int m = 0; m < R0; ++m) v[b * R0 + m] = spec[(size_t)zidx<P, R0, L0>(t, b, m) * plane + qc];
    ZPipe<P, ZC, 0>::run(v, zsm, tw, t, col, txy, coef6, tz, qc == 0);
    if (valid) {
#pragma unroll
        for (int b = 0; b < 8 / R0; ++b)
#pragma unroll
            for (int m = 0; m < R0; ++m) spec[(size_t)zidx<P, R0, L0>(t, b, m) * plane + q] = v[b * R0 + m];
    }
}

template <int P, int ZC, int MINB>
static int launch_zpass_t(gp_ctx* c, double coef6) {
    const size_t plane = ((size_t)c->g.nx / 2 + 1) * c->g.ny;
    const int threads = (1 << P) / 8 * ZC;
    const size_t smem = (size_t)(1 << P) * ZC * sizeof(double2);
    // the opt-in is per device and cheap: set it on every launch (a context may live on any device)
    GP_CUDA(cudaFuncSetAttribute(k_zpass_green<P, ZC, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    k_zpass_green<P, ZC, MINB><<<(unsigned)((plane + ZC - 1) / ZC), threads, smem, c->stream>>>(
        plane, c->g.nx / 2 + 1, c->tabx, c->taby, c->tabz, (const double2*)c->ztw, coef6, (double2*)c->spec);
    GP_CUDA(cudaGetLastError());
    return GP_OK;
}

bool zpass_supported(int nz) { return nz >= 8 && nz <= 1024 && (nz & (nz - 1)) == 0; }

// coef6 = -4 pi G h^2 / (6 N): the Green factor is coef6 / (1 - tx ty tz)
int launch_zpass(gp_ctx* c, double coef6) {
    switch (c->g.nz) {
        case 8: return launch_zpass_t<3, 8, 1>(c, coef6);
        case 16: return launch_zpass_t<4, 8, 1>(c, coef6);
        case 32: return launch_zpass_t<5, 8, 1>(c, coef6);
        case 64: return launch_zpass_t<6, 8, 1>(c, coef6);
        case 128: return launch_zpass_t<7, 8, 1>(c, coef6);
        case 256: return launch_zpass_t<8, 8, 1>(c, coef6);
        case 512: return launch_zpass_t<9, GP_ZP9_C, GP_ZP9_MINB>(c, coef6);   // two 256-thread blocks per SM beat one of 512
        case 1024: return launch_zpass_t<10, 4, 1>(c, coef6);
    }
    set_error("launch_zpass: nz = %d is not a supported power of two", c->g.nz);
    return GP_ERR_UNSUPPORTED;
}

}  // namespace gp
