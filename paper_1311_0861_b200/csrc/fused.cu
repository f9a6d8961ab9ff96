// Fused hydro step of libgpupegas.so: Eulerian stage and
// Lagrangian stage of one component in ONE pass over HBM, with the CFL
// reduction of the new state (reading G4) in the epilogue.
//
// 2.5-D streaming.  A block of FX x FY = 32 x 16 threads owns an xy footprint (28 x 12 output
// cells plus a two-cell halo) and marches along z.  Per plane it
//   A  loads U^n (register prefetch one plane ahead), recovers primitives, publishes them in
//      shared memory for the x/y neighbours;
//   B  computes each x-, y- and z-face ONCE (hi face per thread; the lo face comes from the lane
//      to the left by warp shuffle, from the row below through shared memory, from the previous
//      plane in registers) and assembles U* of the footprint's inner ring;
//   C  writes U* (density, velocity w* = momentum*/density, remaining fields) into a three-plane
//      ring in shared memory -- U* never goes to HBM;
//   D  advects plane k-1 of the ring: 4-vertex face velocities as separable (1/4,1/2,1/4)
//      averages, upwind donor-cell fluxes in coefficient form, writes U^{n+1}, and folds the
//      max signal speed of U^{n+1} into a block maximum.
// Ghost cells are index maps (wrap / clamp of the load address); for outflow the U* ghosts are
// copies of the nearest interior U* (H6), restored in shared memory after step C.
#include "gp_internal.h"

namespace gp {

constexpr int FX = 32, FY = 16, PL = FX * FY;
constexpr int TXO = FX - 4, TYO = FY - 4;

// ---- fp64 reciprocal and reciprocal square root: MUFU seed + one cubically convergent step ----
// seed relative error <= 2^-20  ->  after the step <= ~2^-59; final rounding ~1 ulp.
__device__ __forceinline__ double frcp(double x) {
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double r = fma(-x, y, 1.0);
    const double t = fma(r, r, r);
    return fma(y, t, y);
}
__device__ __forceinline__ double frsqrt(double x) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double xy = x * y;
    const double r = fma(-xy, y, 1.0);
    const double p = fma(0.375, r, 0.5);
    const double yr = y * r;
    return fma(yr, p, y);
}

__device__ __forceinline__ int map_safe(int i, int n, int bc) {
    if (bc == GP_BC_PERIODIC) {
        if (i < 0) i += n;
        else if (i >= n) i -= n;
    }
    return i < 0 ? 0 : (i >= n ? n - 1 : i);
}

// Phi of one footprint column (fixed virtual x, y), plane by plane.  A position with exactly one
// coordinate outside the grid by one reads the ghost-face array of that side (periodic solve:
// the wrapped value; isolated solve: the padded convolution; user-set Phi: the hydro rule);
// anything further out is only ever used by U* of periodic ghost cells and reads the mapped cell.
struct PhiCol {
    const double* p; size_t stride;      // planes inside the grid
    const double* zlo; const double* zhi;   // planes -1 and nz when x and y are inside, else null
    const double* cm; size_t nxny;       // mapped cell column
};

__device__ __forceinline__ PhiCol phi_col(const Geo& g, const Phi& P, int xv, int yv, int xm, int ym) {
    PhiCol c;
    const bool xin = xv >= 0 && xv < g.nx, yin = yv >= 0 && yv < g.ny;
    c.nxny = (size_t)g.nx * g.ny;
    c.cm = P.c + (size_t)xm + (size_t)g.nx * ym;
    c.p = c.cm; c.stride = c.nxny; c.zlo = c.zhi = nullptr;
    if (xin && yin) {
        c.zlo = P.gz0 + (size_t)xm + (size_t)g.nx * ym;
        c.zhi = P.gz1 + (size_t)xm + (size_t)g.nx * ym;
    } else if (yin && (xv == -1 || xv == g.nx)) {
        c.p = (xv < 0 ? P.gx0 : P.gx1) + ym; c.stride = g.ny;
    } else if (xin && (yv == -1 || yv == g.ny)) {
        c.p = (yv < 0 ? P.gy0 : P.gy1) + xm; c.stride = g.nx;
    }
    return c;
}

__device__ __forceinline__ double phi_load(const PhiCol& c, int kv, int zm, int nz) {
    if (kv >= 0 && kv < nz) return c.p[(size_t)zm * c.stride];
    if (c.zlo && kv == -1) return *c.zlo;
    if (c.zlo && kv == nz) return *c.zhi;
    return c.cm[(size_t)zm * c.nxny];
}

// ---- face solvers ------------------------------------------------------------------------------
// PAPER.md:112, 114 with Z = sqrt(rl rr gamma (pl+pr)/(rl+rr)) = num*r, 1/Z = den*r, r = rsqrt(num*den).
__device__ __forceinline__ void gas_face(double gamma, double rl, double vl, double pl, double rr, double vr, double pr,
                                         double& P, double& PV) {
    const double ps = pl + pr;
    const double num = rl * rr * (gamma * ps), den = rl + rr;
    const double r = frsqrt(num * den);
    const double Z = num * r, iZ = den * r;
    const double V = fma(0.5 * (pl - pr), iZ, 0.5 * (vl + vr));
    P = fma(0.5 * (vl - vr), Z, 0.5 * ps);
    PV = P * V;
}

// PAPER.md:170-178 for a face normal to axis D, bracketed parameters averaged (PAPER.md:180,
// reading G7).  In: n, u[3], Pd[3] = Pi_{xD}, Pi_{yD}, Pi_{zD} of both sides.
// Out: Ps[3] = Pi*_{.D} (momentum flux) and EF[6] = Pi*_{jD} u*_i + Pi*_{iD} u*_j for
// (i,j) = xx xy xz yy yz zz (flux of nE_ij).
// With q = 2 nl nr, s = nl+nr, a = (Pl+Pr)/2:  [rho] = q/s, Z1 = sqrt([rho] a) = q a r,
// 1/Z1 = s r, 1/a = q s r^2, where r = rsqrt(q a s).
template <int D>
__device__ __forceinline__ void bme_face(double nl, const double ul[3], const double Pl[3],
                                         double nr, const double ur[3], const double Pr[3],
                                         double Ps[3], double EF[6]) {
    const double s3 = 1.7320508075688772935, is3 = 0.57735026918962576451;
    const double q = (nl + nl) * nr, s = nl + nr;
    const double a = 0.5 * (Pl[D] + Pr[D]);
    const double qa = q * a;
    const double r = frsqrt(qa * s);
    const double Z1 = qa * r, iZ1 = s * r;
    const double ia = (q * s) * (r * r);
    const double Z3 = s3 * Z1, iZ3 = is3 * iZ1;
    const double dPdd = 0.5 * (Pl[D] - Pr[D]);
    const double dud = 0.5 * (ul[D] - ur[D]);
    double us[3];
    us[D] = fma(dPdd, iZ3, 0.5 * (ul[D] + ur[D]));
    Ps[D] = fma(dud, Z3, a);
    const double ku = (1.0 - s3) * (ia * iZ3) * dPdd;      // dPdd (1-sqrt3) / (a Z3)
    const double kp = (s3 - 1.0) * (Z1 * ia) * dud;        // dud [rho] (sqrt3-1) / Z1 = dud (sqrt3-1) Z1 / a
#pragma unroll
    for (int w = 1; w <= 2; ++w) {
        const int t = (D + w) % 3;
        const double b = 0.5 * (Pl[t] + Pr[t]);
        us[t] = fma(b, ku, fma(0.5 * (Pl[t] - Pr[t]), iZ1, 0.5 * (ul[t] + ur[t])));
        Ps[t] = fma(b, kp, fma(0.5 * (ul[t] - ur[t]), Z1, b));
    }
    EF[0] = 2.0 * Ps[0] * us[0];
    EF[1] = fma(Ps[1], us[0], Ps[0] * us[1]);
    EF[2] = fma(Ps[2], us[0], Ps[0] * us[2]);
    EF[3] = 2.0 * Ps[1] * us[1];
    EF[4] = fma(Ps[2], us[1], Ps[1] * us[2]);
    EF[5] = 2.0 * Ps[2] * us[2];
}

// ---- Lagrangian stage of one output cell from the U* ring ---------------------------------------
// Ring slot layout: [field][PL], field 0 = density, 1..3 = w*, 4.. = the NO remaining fields.
// Upwind flux form in coefficient form:
//   F+ = max(w+,0) f0 + min(w+,0) f+,  F- = max(w-,0) f- + min(w-,0) f0
//   f' = f0 - th (sum_d F+ - F-) = c0 f0 + sum_q c_q f_q
// Momentum = density * w*, so its update is sum_q (c_q dens_q) w_q.
template <int NO>
__device__ __forceinline__ void lagrange_cell(const double* __restrict__ rm, const double* __restrict__ r0,
                                              const double* __restrict__ rp, int t, double th,
                                              double wxm, double wxp, double wym, double wyp, double wzm, double wzp,
                                              double out[4 + NO]) {
    const double cxm = th * fmax(wxm, 0.0), cxp = -th * fmin(wxp, 0.0);
    const double cym = th * fmax(wym, 0.0), cyp = -th * fmin(wyp, 0.0);
    const double czm = th * fmax(wzm, 0.0), czp = -th * fmin(wzp, 0.0);
    const double sum = (fmax(wxp, 0.0) - fmin(wxm, 0.0)) + (fmax(wyp, 0.0) - fmin(wym, 0.0)) +
                       (fmax(wzp, 0.0) - fmin(wzm, 0.0));
    const double c0 = fma(-th, sum, 1.0);
    // density-weighted coefficients
    const double d0 = c0 * r0[t], dxm = cxm * r0[t - 1], dxp = cxp * r0[t + 1];
    const double dym = cym * r0[t - FX], dyp = cyp * r0[t + FX];
    const double dzm = czm * rm[t], dzp = czp * rp[t];
    out[0] = ((d0 + dxm) + (dxp + dym)) + ((dyp + dzm) + dzp);
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const double* w0 = r0 + (1 + d) * PL;
        double v = d0 * w0[t];
        v = fma(dxm, w0[t - 1], v);
        v = fma(dxp, w0[t + 1], v);
        v = fma(dym, w0[t - FX], v);
        v = fma(dyp, w0[t + FX], v);
        v = fma(dzm, rm[(1 + d) * PL + t], v);
        v = fma(dzp, rp[(1 + d) * PL + t], v);
        out[1 + d] = v;
    }
#pragma unroll
    for (int f = 0; f < NO; ++f) {
        const double* e0 = r0 + (4 + f) * PL;
        double v = c0 * e0[t];
        v = fma(cxm, e0[t - 1], v);
        v = fma(cxp, e0[t + 1], v);
        v = fma(cym, e0[t - FX], v);
        v = fma(cyp, e0[t + FX], v);
        v = fma(czm, rm[(4 + f) * PL + t], v);
        v = fma(czp, rp[(4 + f) * PL + t], v);
        out[4 + f] = v;
    }
}

// (1/4,1/2,1/4) average of three values
__device__ __forceinline__ double avg3(double a, double b, double c) { return fma(0.25, a + c, 0.5 * b); }

// 3x3 (omega x omega) average around t in a plane
__device__ __forceinline__ double avg9(const double* __restrict__ s, int t) {
    const double lo = avg3(s[t - FX - 1], s[t - FX], s[t - FX + 1]);
    const double mi = avg3(s[t - 1], s[t], s[t + 1]);
    const double hi = avg3(s[t + FX - 1], s[t + FX], s[t + FX + 1]);
    return avg3(lo, mi, hi);
}

template <int NF>
struct FusedArgs {
    Geo g;
    const double* U[NF];
    double* Un[NF];
    Phi phi;
    double h, gamma, dt_val;
    const double* dt_ptr;
    int zchunk;
    unsigned long long* smax_bits;
    int* flag;
};

struct Foot {
    int tx, ty, t, xv, yv, xm, ym, z0, z1;
    size_t base, nxny;
    bool star_row, out_row, is_out, fix, block_fix;
    int fix_src;
};

__device__ __forceinline__ Foot make_foot(const Geo& g, int zchunk) {
    Foot f;
    f.tx = threadIdx.x; f.ty = threadIdx.y; f.t = f.ty * FX + f.tx;
    const int x0 = blockIdx.x * TXO, y0 = blockIdx.y * TYO;
    f.z0 = blockIdx.z * zchunk;
    f.z1 = min(g.nz, f.z0 + zchunk);
    f.xv = x0 - 2 + f.tx; f.yv = y0 - 2 + f.ty;
    f.xm = map_safe(f.xv, g.nx, g.bcx); f.ym = map_safe(f.yv, g.ny, g.bcy);
    f.nxny = (size_t)g.nx * g.ny;
    f.base = (size_t)f.xm + (size_t)g.nx * f.ym;
    f.star_row = f.ty >= 1 && f.ty <= FY - 2;
    f.out_row = f.ty >= 2 && f.ty <= FY - 3;
    f.is_out = f.out_row && f.tx >= 2 && f.tx <= FX - 3 && f.xv < g.nx && f.yv < g.ny;
    // outflow: U* ghost (one layer round the grid) := nearest interior U*
    f.fix = false; f.fix_src = f.t;
    if (g.bcx == GP_BC_OUTFLOW) {
        if (f.xv == -1) { f.fix_src += 1; f.fix = true; }
        else if (f.xv == g.nx) { f.fix_src -= 1; f.fix = true; }
    }
    if (g.bcy == GP_BC_OUTFLOW) {
        if (f.yv == -1) { f.fix_src += FX; f.fix = true; }
        else if (f.yv == g.ny) { f.fix_src -= FX; f.fix = true; }
    }
    f.fix = f.fix && f.star_row && f.tx >= 1 && f.tx <= FX - 2;
    f.block_fix = (g.bcx == GP_BC_OUTFLOW && (x0 == 0 || x0 + TXO >= g.nx)) ||
                  (g.bcy == GP_BC_OUTFLOW && (y0 == 0 || y0 + TYO >= g.ny));
    return f;
}

__device__ __forceinline__ int ring_slot(int k) { return (k + 3) % 3; }

// block maximum of the signal speed -> one atomicMax of the bit pattern (speeds are >= 0)
__device__ __forceinline__ void block_max_commit(double smax, int bad, unsigned long long* smax_bits, int* flag,
                                                 double* scratch) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        smax = fmax(smax, __shfl_xor_sync(0xffffffffu, smax, o));
        bad |= __shfl_xor_sync(0xffffffffu, bad, o);
    }
    __syncthreads();
    int* sbad = (int*)(scratch + FY);
    if (threadIdx.x == 0) { scratch[threadIdx.y] = smax; sbad[threadIdx.y] = bad; }
    __syncthreads();
    if (threadIdx.y == 0) {
        smax = threadIdx.x < FY ? scratch[threadIdx.x] : 0.0;
        bad = threadIdx.x < FY ? sbad[threadIdx.x] : 0;
#pragma unroll
        for (int o = 8; o > 0; o >>= 1) {
            smax = fmax(smax, __shfl_xor_sync(0xffffffffu, smax, o));
            bad |= __shfl_xor_sync(0xffffffffu, bad, o);
        }
        if (threadIdx.x == 0) {
            atomicMax(smax_bits, (unsigned long long)__double_as_longlong(smax));
            if (bad) atomicOr(flag, 1);
        }
    }
}

// =================================================================================================
// Gas: fields rho, mx, my, mz, E.   Shared planes: 5 prims (rho, vx, vy, p, Phi), 2 y-flux,
// 3 x 5 ring (rho, wx, wy, wz, E), 2 smoothing = 24 planes = 96 KB.
// =================================================================================================
constexpr int GAS_NR = 5;
constexpr int GAS_PLANES = 5 + 2 + 3 * GAS_NR + 2;

__global__ void __launch_bounds__(PL, 1)
k_fused_gas(FusedArgs<NGAS> a) {
    extern __shared__ double sm[];
    double* s_rho = sm; double* s_vx = sm + PL; double* s_vy = sm + 2 * PL; double* s_p = sm + 3 * PL;
    double* s_phi = sm + 4 * PL; double* s_fP = sm + 5 * PL; double* s_fPV = sm + 6 * PL;
    double* ring = sm + 7 * PL;
    double* s_tx = ring + 3 * GAS_NR * PL; double* s_ty = s_tx + PL;

    const Geo g = a.g;
    const Foot f = make_foot(g, a.zchunk);
    const int t = f.t;
    const double tau = a.dt_ptr ? *a.dt_ptr : a.dt_val;
    const double th = tau / a.h, inv2h = 0.5 / a.h, gamma = a.gamma, gm1 = a.gamma - 1.0;
    const PhiCol pc = phi_col(g, a.phi, f.xv, f.yv, f.xm, f.ym);
    const bool zout = g.bcz == GP_BC_OUTFLOW;

    double nx_[NGAS], nphi;
    {
        const int zm = map_safe(f.z0 - 2, g.nz, g.bcz);
        const size_t off = f.base + (size_t)zm * f.nxny;
#pragma unroll
        for (int q = 0; q < NGAS; ++q) nx_[q] = a.U[q][off];
        nphi = phi_load(pc, f.z0 - 2, zm, g.nz);
    }
    double pr_rho = 1.0, pr_ir = 1.0, pr_vz = 0.0, pr_mz = 0.0, pr_p = 1.0;
    double acc_mx = 0.0, acc_my = 0.0, acc_mz = 0.0, acc_E = 0.0;
    double phi_m1 = 0.0, phi_m2 = 0.0;
    double Sz_prev = 0.0, wzp_prev = 0.0, smax = 0.0;
    int bad = 0;

    for (int kv = f.z0 - 2; kv <= f.z1 + 1; ++kv) {
        const double rho = nx_[0], mx = nx_[1], my = nx_[2], mz = nx_[3], E = nx_[4], phi = nphi;
        if (kv <= f.z1) {
            const int zm = map_safe(kv + 1, g.nz, g.bcz);
            const size_t off = f.base + (size_t)zm * f.nxny;
#pragma unroll
            for (int q = 0; q < NGAS; ++q) nx_[q] = a.U[q][off];
            nphi = phi_load(pc, kv + 1, zm, g.nz);
        }
        // A: primitives (S0)
        const double ir = frcp(rho);
        const double vx = mx * ir, vy = my * ir, vz = mz * ir;
        const double p = gm1 * (E - 0.5 * fma(mx, vx, fma(my, vy, mz * vz)));
        s_rho[t] = rho; s_vx[t] = vx; s_vy[t] = vy; s_p[t] = p; s_phi[t] = phi;
        __syncthreads();

        // B: faces
        const bool xy_stage = kv >= f.z0 - 1 && kv <= f.z1;
        const bool z_stage = kv >= f.z0 - 1;
        double Pyh = 0.0, PVyh = 0.0, Pxh = 0.0, PVxh = 0.0, Pxl = 0.0, PVxl = 0.0, Pz = 0.0, PVz = 0.0;
        if (xy_stage && f.ty <= FY - 2) {
            gas_face(gamma, rho, vy, p, s_rho[t + FX], s_vy[t + FX], s_p[t + FX], Pyh, PVyh);
            s_fP[t] = Pyh; s_fPV[t] = PVyh;
        }
        if (f.star_row) {
            if (xy_stage) {
                const int tr = f.tx < FX - 1 ? t + 1 : t;
                gas_face(gamma, rho, vx, p, s_rho[tr], s_vx[tr], s_p[tr], Pxh, PVxh);
                Pxl = __shfl_up_sync(0xffffffffu, Pxh, 1);
                PVxl = __shfl_up_sync(0xffffffffu, PVxh, 1);
            }
            if (z_stage) gas_face(gamma, pr_rho, pr_vz, pr_p, rho, vz, p, Pz, PVz);
        }
        __syncthreads();

        // C: finish U*(kv-1), start U*(kv)
        if (f.star_row) {
            if (kv >= f.z0) {
                double* rs = ring + ring_slot(kv - 1) * GAS_NR * PL;
                if (zout && kv - 1 == g.nz) {          // top ghost plane := U*(nz-1)
                    const double* rq = ring + ring_slot(kv - 2) * GAS_NR * PL;
#pragma unroll
                    for (int q = 0; q < GAS_NR; ++q) rs[q * PL + t] = rq[q * PL + t];
                } else {
                    const double gz = (phi - phi_m2) * inv2h;
                    const double mzs = acc_mz - th * Pz - tau * pr_rho * gz;
                    const double Es = acc_E - th * PVz - tau * (pr_mz - 0.5 * tau * pr_rho * gz) * gz;
                    const double wx = acc_mx * pr_ir, wy = acc_my * pr_ir, wz = mzs * pr_ir;
                    rs[t] = pr_rho; rs[PL + t] = wx; rs[2 * PL + t] = wy; rs[3 * PL + t] = wz; rs[4 * PL + t] = Es;
                    if (zout && kv - 1 == 0) {         // bottom ghost plane := U*(0)
                        double* rg = ring + ring_slot(-1) * GAS_NR * PL;
                        rg[t] = pr_rho; rg[PL + t] = wx; rg[2 * PL + t] = wy; rg[3 * PL + t] = wz; rg[4 * PL + t] = Es;
                    }
                }
            }
            if (xy_stage) {
                const double Pyl = s_fP[t - FX], PVyl = s_fPV[t - FX];
                const double gx = (s_phi[t + 1] - s_phi[t - 1]) * inv2h;
                const double gy = (s_phi[t + FX] - s_phi[t - FX]) * inv2h;
                acc_mx = mx - th * (Pxh - Pxl) - tau * rho * gx;
                acc_my = my - th * (Pyh - Pyl) - tau * rho * gy;
                acc_mz = fma(th, Pz, mz);
                acc_E = E - th * ((PVxh - PVxl) + (PVyh - PVyl)) + th * PVz -
                        tau * ((mx - 0.5 * tau * rho * gx) * gx + (my - 0.5 * tau * rho * gy) * gy);
            }
        }
        pr_rho = rho; pr_ir = ir; pr_vz = vz; pr_mz = mz; pr_p = p;
        phi_m2 = phi_m1; phi_m1 = phi;
        __syncthreads();

        if (kv < f.z0) continue;
        if (f.block_fix) {
            if (f.fix) {
                double* rs = ring + ring_slot(kv - 1) * GAS_NR * PL;
#pragma unroll
                for (int q = 0; q < GAS_NR; ++q) rs[q * PL + t] = rs[q * PL + f.fix_src];
                if (zout && kv - 1 == 0) {
                    double* rg = ring + ring_slot(-1) * GAS_NR * PL;
#pragma unroll
                    for (int q = 0; q < GAS_NR; ++q) rg[q * PL + t] = rg[q * PL + f.fix_src];
                }
            }
            __syncthreads();
        }

        // D: Lagrangian stage of plane k = kv-2 (ring planes kv-3, kv-2, kv-1)
        const double* rp = ring + ring_slot(kv - 1) * GAS_NR * PL;
        const double* r0 = ring + ring_slot(kv - 2) * GAS_NR * PL;
        const double* rm = ring + ring_slot(kv - 3) * GAS_NR * PL;
        const bool do_out = kv >= f.z0 + 2;
        if (do_out && f.star_row) {
            s_tx[t] = avg3(rm[PL + t], r0[PL + t], rp[PL + t]);
            s_ty[t] = avg3(rm[2 * PL + t], r0[2 * PL + t], rp[2 * PL + t]);
        }
        if (do_out) __syncthreads();
        if (f.out_row) {
            const double Sz_new = avg9(rp + 3 * PL, t);
            if (zout && kv - 1 == 0) Sz_prev = Sz_new;
            if (kv >= f.z0 + 1) {
                const double wzp = 0.5 * (Sz_prev + Sz_new);
                if (do_out) {
                    const double a_m = avg3(s_tx[t - FX - 1], s_tx[t - 1], s_tx[t + FX - 1]);
                    const double a_0 = avg3(s_tx[t - FX], s_tx[t], s_tx[t + FX]);
                    const double a_p = avg3(s_tx[t - FX + 1], s_tx[t + 1], s_tx[t + FX + 1]);
                    const double b_m = avg3(s_ty[t - FX - 1], s_ty[t - FX], s_ty[t - FX + 1]);
                    const double b_0 = avg3(s_ty[t - 1], s_ty[t], s_ty[t + 1]);
                    const double b_p = avg3(s_ty[t + FX - 1], s_ty[t + FX], s_ty[t + FX + 1]);
                    double out[NGAS];
                    lagrange_cell<1>(rm, r0, rp, t, th, 0.5 * (a_m + a_0), 0.5 * (a_0 + a_p), 0.5 * (b_m + b_0),
                                     0.5 * (b_0 + b_p), wzp_prev, wzp, out);
                    if (f.is_out) {
                        const size_t off = f.base + (size_t)(kv - 2) * f.nxny;
#pragma unroll
                        for (int q = 0; q < NGAS; ++q) a.Un[q][off] = out[q];
                        // CFL of the new state (reading G4)
                        const double irn = frcp(out[0]);
                        const double ux = out[1] * irn, uy = out[2] * irn, uz = out[3] * irn;
                        const double pn = gm1 * (out[4] - 0.5 * fma(out[1], ux, fma(out[2], uy, out[3] * uz)));
                        const double c2 = gamma * pn * irn;
                        const double cs = c2 * frsqrt(c2);
                        const double s = fmax(fmax(fabs(ux), fabs(uy)), fabs(uz)) + cs;
                        if (!(out[0] > 0.0) || !(pn > 0.0) || !(s <= 1.7976931348623157e308)) bad = 1;
                        smax = fmax(smax, s);
                    }
                }
                wzp_prev = wzp;
            }
            Sz_prev = Sz_new;
        }
    }
    block_max_commit(smax, bad, a.smax_bits, a.flag, s_rho);
}

// =================================================================================================
// Collisionless component: fields n, nu (3), nE_ij (6).  Shared planes: 10 prims (n, u3, Pixx,
// Pixy, Pixz, Piyy, Piyz, Phi), 9 y-flux, 3 x 10 ring (n, w3, E6), 2 smoothing = 51 planes = 204 KB.
// =================================================================================================
constexpr int BME_NR = 10;
constexpr int BME_PLANES = 10 + 9 + 3 * BME_NR + 2;

__global__ void __launch_bounds__(PL, 1)
k_fused_bme(FusedArgs<NBME> a) {
    extern __shared__ double sm[];
    double* s_n = sm;                 // prims: n, ux, uy, uz, Pxx, Pxy, Pxz, Pyy, Pyz, Phi
    double* s_phi = sm + 9 * PL;
    double* s_fl = sm + 10 * PL;      // y-flux: Ps[3], EF[6]
    double* ring = sm + 19 * PL;
    double* s_tx = ring + 3 * BME_NR * PL; double* s_ty = s_tx + PL;

    const Geo g = a.g;
    const Foot f = make_foot(g, a.zchunk);
    const int t = f.t;
    const double tau = a.dt_ptr ? *a.dt_ptr : a.dt_val;
    const double th = tau / a.h, inv2h = 0.5 / a.h;
    const PhiCol pc = phi_col(g, a.phi, f.xv, f.yv, f.xm, f.ym);
    const bool zout = g.bcz == GP_BC_OUTFLOW;

    double nx_[NBME], nphi;
    {
        const int zm = map_safe(f.z0 - 2, g.nz, g.bcz);
        const size_t off = f.base + (size_t)zm * f.nxny;
#pragma unroll
        for (int q = 0; q < NBME; ++q) nx_[q] = a.U[q][off];
        nphi = phi_load(pc, f.z0 - 2, zm, g.nz);
    }
    // previous plane (for the z-face and for finishing U*(kv-1))
    double pr_n = 1.0, pr_in = 1.0, pr_u[3] = {0.0, 0.0, 0.0}, pr_Pz[3] = {0.0, 0.0, 1.0};
    double pr_gx = 0.0, pr_gy = 0.0;
    double acc[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};     // nu (3), nE (6) of U*(kv-1) so far
    double phi_m1 = 0.0, phi_m2 = 0.0;
    double Sz_prev = 0.0, wzp_prev = 0.0, smax = 0.0;
    int bad = 0;

    for (int kv = f.z0 - 2; kv <= f.z1 + 1; ++kv) {
        double Uc[NBME];
#pragma unroll
        for (int q = 0; q < NBME; ++q) Uc[q] = nx_[q];
        const double phi = nphi;
        if (kv <= f.z1) {
            const int zm = map_safe(kv + 1, g.nz, g.bcz);
            const size_t off = f.base + (size_t)zm * f.nxny;
#pragma unroll
            for (int q = 0; q < NBME; ++q) nx_[q] = a.U[q][off];
            nphi = phi_load(pc, kv + 1, zm, g.nz);
        }
        // A: primitives (S0): u = nu/n, Pi_ij = nE_ij - n u_i u_j
        const double n = Uc[0];
        const double in = frcp(n);
        double u[3] = {Uc[1] * in, Uc[2] * in, Uc[3] * in};
        double Pi[6];
        Pi[0] = fma(-Uc[1], u[0], Uc[4]); Pi[1] = fma(-Uc[1], u[1], Uc[5]); Pi[2] = fma(-Uc[1], u[2], Uc[6]);
        Pi[3] = fma(-Uc[2], u[1], Uc[7]); Pi[4] = fma(-Uc[2], u[2], Uc[8]); Pi[5] = fma(-Uc[3], u[2], Uc[9]);
        s_n[t] = n; s_n[PL + t] = u[0]; s_n[2 * PL + t] = u[1]; s_n[3 * PL + t] = u[2];
        s_n[4 * PL + t] = Pi[0]; s_n[5 * PL + t] = Pi[1]; s_n[6 * PL + t] = Pi[2];
        s_n[7 * PL + t] = Pi[3]; s_n[8 * PL + t] = Pi[4]; s_phi[t] = phi;
        __syncthreads();

        // B: faces
        const bool xy_stage = kv >= f.z0 - 1 && kv <= f.z1;
        const bool z_stage = kv >= f.z0 - 1;
        double Py[3], EFy[6], Px[3], EFx[6], Pxl[3], EFxl[6], Pz[3], EFz[6];
#pragma unroll
        for (int q = 0; q < 3; ++q) { Py[q] = Px[q] = Pxl[q] = Pz[q] = 0.0; }
#pragma unroll
        for (int q = 0; q < 6; ++q) { EFy[q] = EFx[q] = EFxl[q] = EFz[q] = 0.0; }
        if (xy_stage && f.ty <= FY - 2) {
            const int tr = t + FX;
            const double ur[3] = {s_n[PL + tr], s_n[2 * PL + tr], s_n[3 * PL + tr]};
            const double Pl[3] = {Pi[1], Pi[3], Pi[4]};
            const double Pr[3] = {s_n[5 * PL + tr], s_n[7 * PL + tr], s_n[8 * PL + tr]};
            bme_face<1>(n, u, Pl, s_n[tr], ur, Pr, Py, EFy);
#pragma unroll
            for (int q = 0; q < 3; ++q) s_fl[q * PL + t] = Py[q];
#pragma unroll
            for (int q = 0; q < 6; ++q) s_fl[(3 + q) * PL + t] = EFy[q];
        }
        if (f.star_row) {
            if (xy_stage) {
                const int tr = f.tx < FX - 1 ? t + 1 : t;
                const double ur[3] = {s_n[PL + tr], s_n[2 * PL + tr], s_n[3 * PL + tr]};
                const double Pl[3] = {Pi[0], Pi[1], Pi[2]};
                const double Pr[3] = {s_n[4 * PL + tr], s_n[5 * PL + tr], s_n[6 * PL + tr]};
                bme_face<0>(n, u, Pl, s_n[tr], ur, Pr, Px, EFx);
#pragma unroll
                for (int q = 0; q < 3; ++q) Pxl[q] = __shfl_up_sync(0xffffffffu, Px[q], 1);
#pragma unroll
                for (int q = 0; q < 6; ++q) EFxl[q] = __shfl_up_sync(0xffffffffu, EFx[q], 1);
            }
            if (z_stage) {
                const double Pr[3] = {Pi[2], Pi[4], Pi[5]};
                bme_face<2>(pr_n, pr_u, pr_Pz, n, u, Pr, Pz, EFz);
            }
        }
        __syncthreads();

        // C: finish U*(kv-1), start U*(kv)
        if (f.star_row) {
            if (kv >= f.z0) {
                double* rs = ring + ring_slot(kv - 1) * BME_NR * PL;
                if (zout && kv - 1 == g.nz) {
                    const double* rq = ring + ring_slot(kv - 2) * BME_NR * PL;
#pragma unroll
                    for (int q = 0; q < BME_NR; ++q) rs[q * PL + t] = rq[q * PL + t];
                } else {
                    const double gr[3] = {pr_gx, pr_gy, (phi - phi_m2) * inv2h};
                    double uc[3];       // time-centred velocity u - tau g / 2 (reading G5)
#pragma unroll
                    for (int d = 0; d < 3; ++d) uc[d] = fma(-0.5 * tau, gr[d], pr_u[d]);
                    const double tn = tau * pr_n;
                    double o[BME_NR];
                    o[0] = pr_n;
#pragma unroll
                    for (int d = 0; d < 3; ++d) o[1 + d] = (acc[d] - th * Pz[d] - tn * gr[d]) * pr_in;
                    o[4] = acc[3] - th * EFz[0] - tn * (2.0 * uc[0] * gr[0]);
                    o[5] = acc[4] - th * EFz[1] - tn * fma(uc[0], gr[1], uc[1] * gr[0]);
                    o[6] = acc[5] - th * EFz[2] - tn * fma(uc[0], gr[2], uc[2] * gr[0]);
                    o[7] = acc[6] - th * EFz[3] - tn * (2.0 * uc[1] * gr[1]);
                    o[8] = acc[7] - th * EFz[4] - tn * fma(uc[1], gr[2], uc[2] * gr[1]);
                    o[9] = acc[8] - th * EFz[5] - tn * (2.0 * uc[2] * gr[2]);
#pragma unroll
                    for (int q = 0; q < BME_NR; ++q) rs[q * PL + t] = o[q];
                    if (zout && kv - 1 == 0) {
                        double* rg = ring + ring_slot(-1) * BME_NR * PL;
#pragma unroll
                        for (int q = 0; q < BME_NR; ++q) rg[q * PL + t] = o[q];
                    }
                }
            }
            if (xy_stage) {
                acc[0] = Uc[1] - th * ((Px[0] - Pxl[0]) + (Py[0] - s_fl[0 * PL + t - FX])) + th * Pz[0];
                acc[1] = Uc[2] - th * ((Px[1] - Pxl[1]) + (Py[1] - s_fl[1 * PL + t - FX])) + th * Pz[1];
                acc[2] = Uc[3] - th * ((Px[2] - Pxl[2]) + (Py[2] - s_fl[2 * PL + t - FX])) + th * Pz[2];
#pragma unroll
                for (int q = 0; q < 6; ++q)
                    acc[3 + q] = Uc[4 + q] - th * ((EFx[q] - EFxl[q]) + (EFy[q] - s_fl[(3 + q) * PL + t - FX])) + th * EFz[q];
                pr_gx = (s_phi[t + 1] - s_phi[t - 1]) * inv2h;
                pr_gy = (s_phi[t + FX] - s_phi[t - FX]) * inv2h;
            }
        }
        pr_n = n; pr_in = in;
#pragma unroll
        for (int d = 0; d < 3; ++d) pr_u[d] = u[d];
        pr_Pz[0] = Pi[2]; pr_Pz[1] = Pi[4]; pr_Pz[2] = Pi[5];
        phi_m2 = phi_m1; phi_m1 = phi;
        __syncthreads();

        if (kv < f.z0) continue;
        if (f.block_fix) {
            if (f.fix) {
                double* rs = ring + ring_slot(kv - 1) * BME_NR * PL;
#pragma unroll
                for (int q = 0; q < BME_NR; ++q) rs[q * PL + t] = rs[q * PL + f.fix_src];
                if (zout && kv - 1 == 0) {
                    double* rg = ring + ring_slot(-1) * BME_NR * PL;
#pragma unroll
                    for (int q = 0; q < BME_NR; ++q) rg[q * PL + t] = rg[q * PL + f.fix_src];
                }
            }
            __syncthreads();
        }

        // D: Lagrangian stage of plane k = kv-2
        const double* rp = ring + ring_slot(kv - 1) * BME_NR * PL;
        const double* r0 = ring + ring_slot(kv - 2) * BME_NR * PL;
        const double* rm = ring + ring_slot(kv - 3) * BME_NR * PL;
        const bool do_out = kv >= f.z0 + 2;
        if (do_out && f.star_row) {
            s_tx[t] = avg3(rm[PL + t], r0[PL + t], rp[PL + t]);
            s_ty[t] = avg3(rm[2 * PL + t], r0[2 * PL + t], rp[2 * PL + t]);
        }
        if (do_out) __syncthreads();
        if (f.out_row) {
            const double Sz_new = avg9(rp + 3 * PL, t);
            if (zout && kv - 1 == 0) Sz_prev = Sz_new;
            if (kv >= f.z0 + 1) {
                const double wzp = 0.5 * (Sz_prev + Sz_new);
                if (do_out) {
                    const double a_m = avg3(s_tx[t - FX - 1], s_tx[t - 1], s_tx[t + FX - 1]);
                    const double a_0 = avg3(s_tx[t - FX], s_tx[t], s_tx[t + FX]);
                    const double a_p = avg3(s_tx[t - FX + 1], s_tx[t + 1], s_tx[t + FX + 1]);
                    const double b_m = avg3(s_ty[t - FX - 1], s_ty[t - FX], s_ty[t - FX + 1]);
                    const double b_0 = avg3(s_ty[t - 1], s_ty[t], s_ty[t + 1]);
                    const double b_p = avg3(s_ty[t + FX - 1], s_ty[t + FX], s_ty[t + FX + 1]);
                    double out[NBME];
                    lagrange_cell<6>(rm, r0, rp, t, th, 0.5 * (a_m + a_0), 0.5 * (a_0 + a_p), 0.5 * (b_m + b_0),
                                     0.5 * (b_0 + b_p), wzp_prev, wzp, out);
                    if (f.is_out) {
                        const size_t off = f.base + (size_t)(kv - 2) * f.nxny;
#pragma unroll
                        for (int q = 0; q < NBME; ++q) a.Un[q][off] = out[q];
                        // CFL of the new state (reading G4): |u_d| + sqrt(3 Pi_dd / n)
                        const double inn = frcp(out[0]);
                        const int dd[3] = {4, 7, 9};
                        if (!(out[0] > 0.0)) bad = 1;
#pragma unroll
                        for (int d = 0; d < 3; ++d) {
                            const double ud = out[1 + d] * inn;
                            const double Pdd = fma(-out[1 + d], ud, out[dd[d]]);
                            const double c2 = 3.0 * Pdd * inn;
                            const double s = fabs(ud) + c2 * frsqrt(c2);
                            if (!(Pdd > 0.0) || !(s <= 1.7976931348623157e308)) bad = 1;
                            smax = fmax(smax, s);
                        }
                    }
                }
                wzp_prev = wzp;
            }
            Sz_prev = Sz_new;
        }
    }
    block_max_commit(smax, bad, a.smax_bits, a.flag, s_n);
}

// -------------------------------------------------------------------------------------------------
// launches
// -------------------------------------------------------------------------------------------------
static int pick_zchunk(const gp_ctx* c, int tiles_xy) {
    // enough blocks for >= 8 waves of 148 one-block SMs, chunks no shorter than 16 planes
    const int nz = c->g.nz;
    int chunks = (8 * 148 + tiles_xy - 1) / tiles_xy;
    if (chunks < 1) chunks = 1;
    int zc = (nz + chunks - 1) / chunks;
    if (zc < 16) zc = 16;
    if (zc > nz) zc = nz;
    return zc;
}

template <int NF, class K>
static int launch_fused_t(gp_ctx* c, K kernel, int f0, int planes, int kid, double dt, const double* d_dt) {
    FusedArgs<NF> a;
    a.g = Geo{c->g.nx, c->g.ny, c->g.nz, c->bc.x, c->bc.y, c->bc.z};
    for (int f = 0; f < NF; ++f) { a.U[f] = c->U[f0 + f]; a.Un[f] = c->Us[f0 + f]; }
    a.phi = Phi{c->phi, c->phig[0], c->phig[1], c->phig[2], c->phig[3], c->phig[4], c->phig[5]};
    a.h = c->g.h; a.gamma = c->gamma; a.dt_val = dt; a.dt_ptr = d_dt;
    a.smax_bits = c->d_smax_next; a.flag = c->d_flag_next;
    const int tx = (c->g.nx + TXO - 1) / TXO, ty = (c->g.ny + TYO - 1) / TYO;
    a.zchunk = pick_zchunk(c, tx * ty);
    const int tz = (c->g.nz + a.zchunk - 1) / a.zchunk;
    const size_t smem = (size_t)planes * PL * sizeof(double);
    static bool attr_done[2] = {false, false};
    if (!attr_done[NF == NGAS ? 0 : 1]) {
        GP_CUDA(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        attr_done[NF == NGAS ? 0 : 1] = true;
    }
    tic(c, kid);
    kernel<<<dim3(tx, ty, tz), dim3(FX, FY, 1), smem, c->stream>>>(a);
    toc(c);
    c->n_own++;
    GP_CUDA(cudaGetLastError());
    return GP_OK;
}

int launch_fused_gas(gp_ctx* c, double dt, const double* d_dt) {
    return launch_fused_t<NGAS>(c, k_fused_gas, 0, GAS_PLANES, K_FUSED_GAS, dt, d_dt);
}

int launch_fused_bme(gp_ctx* c, double dt, const double* d_dt) {
    return launch_fused_t<NBME>(c, k_fused_bme, NGAS, BME_PLANES, K_FUSED_BME, dt, d_dt);
}

// evaluate the device reciprocal / reciprocal square root on n host-supplied values (self test)
__global__ void k_math_selftest(int n, const double* __restrict__ x, double* __restrict__ rcp, double* __restrict__ rsq) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) { rcp[i] = frcp(x[i]); rsq[i] = frsqrt(x[i]); }
}

int math_selftest(int n, const double* x, double* rcp, double* rsq) {
    double *dx = nullptr;
    GP_CUDA(cudaMalloc(&dx, 3 * (size_t)n * sizeof(double)));
    cudaError_t e = cudaMemcpy(dx, x, (size_t)n * sizeof(double), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
        k_math_selftest<<<(n + 255) / 256, 256>>>(n, dx, dx + n, dx + 2 * (size_t)n);
        e = cudaMemcpy(rcp, dx + n, (size_t)n * sizeof(double), cudaMemcpyDeviceToHost);
    }
    if (e == cudaSuccess) e = cudaMemcpy(rsq, dx + 2 * (size_t)n, (size_t)n * sizeof(double), cudaMemcpyDeviceToHost);
    cudaFree(dx);
    GP_CUDA(e);
    return GP_OK;
}

}  // namespace gp
