// In-register radix-8/4/2 column FFT building blocks shared by zpass.cu (periodic solve) and
// isofft.cu (isolated solve): decimation in frequency, digit-reversed output left in place, and
// the mirrored inverse; columns are exchanged between stages through shared memory.
#pragma once

#include "gp_internal.h"

namespace gp {

// C = columns per block: 8 * 16 B = one 128-byte line per z plane

__device__ __forceinline__ double2 cadd(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ double2 csub(double2 a, double2 b) { return make_double2(a.x - b.x, a.y - b.y); }
// a * w (INV: a * conj(w))
template <bool INV>
__device__ __forceinline__ double2 cmul(double2 a, double2 w) {
    return INV ? make_double2(fma(a.x, w.x, a.y * w.y), fma(a.y, w.x, -a.x * w.y))
               : make_double2(fma(a.x, w.x, -a.y * w.y), fma(a.y, w.x, a.x * w.y));
}
// 1/x: hardware seed (relative error <= 2^-20) and one cubically convergent step, ~1 ulp
__device__ __forceinline__ double zrcp(double x) {
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double r = fma(-x, y, 1.0);
    return fma(y, fma(r, r, r), y);
}
// multiply by -i (forward) or +i (inverse)
template <bool INV>
__device__ __forceinline__ double2 mul_i(double2 a) { return INV ? make_double2(-a.y, a.x) : make_double2(a.y, -a.x); }

// in-register DFTs, natural order in and out; forward kernel exp(-2 pi i m n / R), INV: conjugate
template <bool INV>
__device__ __forceinline__ void dft2(double2& a, double2& b) {
    const double2 t = a;
    a = cadd(t, b); b = csub(t, b);
}
template <bool INV>
__device__ __forceinline__ void dft4(double2& x0, double2& x1, double2& x2, double2& x3) {
    const double2 t0 = cadd(x0, x2), t1 = csub(x0, x2), t2 = cadd(x1, x3), t3 = mul_i<INV>(csub(x1, x3));
    x0 = cadd(t0, t2); x2 = csub(t0, t2); x1 = cadd(t1, t3); x3 = csub(t1, t3);
}
template <bool INV>
__device__ __forceinline__ void dft8(double2* v) {
    dft4<INV>(v[0], v[2], v[4], v[6]);      // E_k in v[2k]
    dft4<INV>(v[1], v[3], v[5], v[7]);      // O_k in v[2k+1]
    const double r = 0.70710678118654752440;
    const double2 o0 = v[1], o1 = v[3], o2 = v[5], o3 = v[7];
    // w^k O_k with w = exp(-+ 2 pi i / 8)
    const double2 w1 = INV ? make_double2(r * (o1.x - o1.y), r * (o1.x + o1.y)) : make_double2(r * (o1.x + o1.y), r * (o1.y - o1.x));
    const double2 w2 = mul_i<INV>(o2);
    const double2 w3 = INV ? make_double2(-r * (o3.x + o3.y), r * (o3.x - o3.y)) : make_double2(r * (o3.y - o3.x), -r * (o3.x + o3.y));
    const double2 e0 = v[0], e1 = v[2], e2 = v[4], e3 = v[6];
    v[0] = cadd(e0, o0); v[4] = csub(e0, o0);
    v[1] = cadd(e1, w1); v[5] = csub(e1, w1);
    v[2] = cadd(e2, w2); v[6] = csub(e2, w2);
    v[3] = cadd(e3, w3); v[7] = csub(e3, w3);
}
template <int R, bool INV>
__device__ __forceinline__ void dft(double2* v) {
    if (R == 8) dft8<INV>(v);
    else if (R == 4) dft4<INV>(v[0], v[1], v[2], v[3]);
    else dft2<INV>(v[0], v[1]);
}

// stage s of a 2^P point transform: radix and length of the sub-transforms it splits
template <int P> struct ZStages {
    static constexpr int N8 = P / 3, REM = P % 3, S = N8 + (REM ? 1 : 0);
    __host__ __device__ static constexpr int radix(int s) { return s < N8 ? 8 : (1 << REM); }
    __host__ __device__ static constexpr int len(int s) { return (1 << P) >> (3 * s); }
};

// element index of member m of butterfly b (of 8/R per thread) of thread t in a stage (R, L)
template <int P, int R, int L>
__device__ __forceinline__ int zidx(int t, int b, int m) {
    constexpr int T = (1 << P) / 8, Q = L / R;
    const int u = t + T * b;
    return (u / Q) * L + (u % Q) + m * Q;
}

// Shared-memory slot of element idx of a column.  The closing stages address elements 8 apart from consecutive threads
// (Q = 1: idx = 8 t + m), which would put the eight t values of a warp on the same banks (C * 16 B * 8 = a multiple of
// 128 B): XOR the low three bits with the next three.  Within an aligned group of eight elements this is a permutation,
// so the stages whose threads walk consecutive elements stay conflict-free.
__device__ __forceinline__ int zslot(int idx) { return idx ^ ((idx >> 3) & 7); }

template <int P, int C, int s>
struct ZExchange {
    // registers (stage s layout) -> shared -> registers (stage s2 layout)
    template <int s2>
    __device__ static __forceinline__ void run(double2* v, double2* sm, int t, int col) {
        constexpr int R = ZStages<P>::radix(s), L = ZStages<P>::len(s);
        constexpr int R2 = ZStages<P>::radix(s2), L2 = ZStages<P>::len(s2);
#pragma unroll
        for (int b = 0; b < 8 / R; ++b)
#pragma unroll
            for (int m = 0; m < R; ++m) sm[zslot(zidx<P, R, L>(t, b, m)) * C + col] = v[b * R + m];
        __syncthreads();
#pragma unroll
        for (int b = 0; b < 8 / R2; ++b)
#pragma unroll
            for (int m = 0; m < R2; ++m) v[b * R2 + m] = sm[zslot(zidx<P, R2, L2>(t, b, m)) * C + col];
    }
};

// A radix-8 stage loads the twiddles w, w^2, w^4 of its butterfly and forms w^3, w^5, w^6, w^7 by
// complex products (4 loads less and 16 fp64 operations more per butterfly; the products of unit-modulus numbers lose
// 2-3 ulp, far inside the 1e-11 bar of the potential)

template <int P, int s, bool INV>
__device__ __forceinline__ void zstage(double2* v, const double2* __restrict__ tw, int t) {
    constexpr int R = ZStages<P>::radix(s), L = ZStages<P>::len(s), Q = L / R, T = (1 << P) / 8;
    constexpr int st = (1 << P) / L;
#pragma unroll
    for (int b = 0; b < 8 / R; ++b) {
        const int o = (t + T * b) % Q;
        double2 w[8];
        if (Q > 1) {
            if (R == 8) {
                w[1] = tw[o * st];
                w[2] = tw[o * 2 * st]; w[4] = tw[o * 4 * st];
                w[3] = cmul<false>(w[1], w[2]); w[5] = cmul<false>(w[1], w[4]); w[6] = cmul<false>(w[2], w[4]);
                w[7] = cmul<false>(w[3], w[4]);
            } else {
#pragma unroll
                for (int m = 1; m < R; ++m) w[m] = tw[o * m * st];
            }
        }
#define GP_TWIDDLE(m) w[m]
        if (INV && Q > 1) {
#pragma unroll
            for (int m = 1; m < R; ++m) v[b * R + m] = cmul<true>(v[b * R + m], GP_TWIDDLE(m));
        }
        dft<R, INV>(v + b * R);
        if (!INV && Q > 1) {
#pragma unroll
            for (int m = 1; m < R; ++m) v[b * R + m] = cmul<false>(v[b * R + m], GP_TWIDDLE(m));
        }
#undef GP_TWIDDLE
    }
}

}  // namespace gp
