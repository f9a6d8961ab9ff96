// Fused hydro step of libgpupegas.so: Eulerian stage and
// Lagrangian stage of one component in ONE pass over HBM, with the CFL
// reduction of the new state (reading G4) in the epilogue.
//
// 2.5-D streaming.  A block of FX x FY = 32 x 16 threads owns an xy footprint (28 x 12 output
// cells plus a two-cell halo) and marches along z.  Per plane it
//   B  computes the x and y faces of plane j ONCE each (hi face per thread; the lo face comes
//      from the lane to the left by warp shuffle and from the row below through shared memory);
//   C  adds the flux differences and the gravity source to U*(j) held in registers;
//   E  takes plane j+1 (staged asynchronously, cp.async, into the ring slot that is about to be
//      rewritten), recovers its primitives, computes the z face (j, j+1), completes U*(j) and
//      writes it (density, w* = momentum*/density, remaining fields) into a three-plane ring in
//      shared memory -- U* never goes to HBM -- and publishes the primitives of plane j+1;
//   D  advects plane j-1 of the ring: 4-vertex face velocities as separable (1/4,1/2,1/4)
//      averages, upwind donor-cell fluxes in coefficient form, writes U^{n+1}, and folds the
//      max signal speed of U^{n+1} into a block maximum.
// Two block barriers per plane (after B, after E).
// Ghost cells are index maps (wrap / clamp of the load address); for outflow the U* ghosts are
// copies of the nearest interior U* (H6), restored in shared memory after step C.
#include "gp_internal.h"

namespace gp {
namespace GP_FUSED_NS {

#ifndef GP_FY
#define GP_FY 16
#endif
constexpr int FX = 32, FY = GP_FY, PL = FX * FY;
constexpr int TXO = FX - 4, TYO = FY - 4;
#define GP_KBOUNDS __launch_bounds__(PL, 1)
#ifndef GP_BME_MERGE
#define GP_BME_MERGE 0
#endif
// x neighbours of the Lagrangian stage: 1 = 128-bit shared-memory loads of the cells t-1, t+1; 0 = warp
// shuffles of the centre value (two SHFL plus register moves per double).  With the register budget
// of the present footprints the loads are faster (21.99 against 22.43 ms per 512^3 step).
#ifndef GP_X_LDS
#define GP_X_LDS 1
#endif

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

__device__ __forceinline__ const double* phi_ptr(const PhiCol& c, int kv, int zm, int nz) {
    if (kv >= 0 && kv < nz) return c.p + (size_t)zm * c.stride;
    if (c.zlo && kv == -1) return c.zlo;
    if (c.zlo && kv == nz) return c.zhi;
    return c.cm + (size_t)zm * c.nxny;
}
__device__ __forceinline__ double phi_load(const PhiCol& c, int kv, int zm, int nz) { return *phi_ptr(c, kv, zm, nz); }

// ---- face solvers ------------------------------------------------------------------------------
// The solvers return DOUBLED face values (2P, 4PV ...) so that the factors 1/2 of the paper's
// formulas fold into the flux coefficients tau/(2h), tau/(4h) (exact power-of-two scalings).
//
// PAPER.md:112, 114 with Z = sqrt(rl rr gamma (pl+pr)/(rl+rr)) = num*r, 1/Z = den*r, r = rsqrt(num*den).
// Out: P2 = 2P, PV4 = 4 P V.
__device__ __forceinline__ void gas_face(double gamma, double rl, double vl, double pl, double rr, double vr, double pr,
                                         double& P2, double& PV4) {
    const double ps = pl + pr;
    const double num = rl * rr * (gamma * ps), den = rl + rr;
    const double r = frsqrt(num * den);
    const double Z = num * r, iZ = den * r;
    const double V2 = fma(pl - pr, iZ, vl + vr);
    P2 = fma(vl - vr, Z, ps);
    PV4 = P2 * V2;
}

// PAPER.md:170-178 for a face normal to axis D, bracketed parameters averaged (PAPER.md:180,
// reading G7).  In: n, u[3], Pd[3] = Pi_{xD}, Pi_{yD}, Pi_{zD} of both sides.
// Out: Ps2[3] = 2 Pi*_{.D} (momentum flux) and EF4[6] = 4 (Pi*_{jD} u*_i + Pi*_{iD} u*_j) for
// (i,j) = xx xy xz yy yz zz (flux of nE_ij).
// With q = nl nr, s = nl+nr, A = Pl+Pr (= 2a):  [rho] a = q A / s,  Z1 = sqrt([rho] a) = q A r,
// 1/Z1 = s r, 1/a = 2 q s r^2, where r = rsqrt(q A s).
template <int D>
__device__ __forceinline__ void bme_face(double nl, const double ul[3], const double Pl[3],
                                         double nr, const double ur[3], const double Pr[3],
                                         double Ps2[3], double EF4[6]) {
    const double s3 = 1.7320508075688772935, is3 = 0.57735026918962576451;
    const double q = nl * nr, s = nl + nr;
    const double A = Pl[D] + Pr[D];
    const double qA = q * A;
    const double r = frsqrt(qA * s);
    const double Z1 = qA * r, iZ1 = s * r;
    const double ia = (q * s) * (2.0 * r * r);
    const double Z3 = s3 * Z1, iZ3 = is3 * iZ1;
    const double DP = Pl[D] - Pr[D], DU = ul[D] - ur[D];
    double us2[3];
    us2[D] = fma(DP, iZ3, ul[D] + ur[D]);
    Ps2[D] = fma(DU, Z3, A);
    // b ku = (B/2) (1-sqrt3) (DP/2) / (a Z3) and doubled: B * [(1-sqrt3)/2 * ia * iZ3 * DP]
    const double ku = (0.5 * (1.0 - s3)) * (ia * iZ3) * DP;
    const double kp = (0.5 * (s3 - 1.0)) * (Z1 * ia) * DU;
#pragma unroll
    for (int w = 1; w <= 2; ++w) {
        const int t = (D + w) % 3;
        const double B = Pl[t] + Pr[t];
        us2[t] = fma(B, ku, fma(Pl[t] - Pr[t], iZ1, ul[t] + ur[t]));
        Ps2[t] = fma(B, kp, fma(ul[t] - ur[t], Z1, B));
    }
    EF4[0] = 2.0 * Ps2[0] * us2[0];
    EF4[1] = fma(Ps2[1], us2[0], Ps2[0] * us2[1]);
    EF4[2] = fma(Ps2[2], us2[0], Ps2[0] * us2[2]);
    EF4[3] = 2.0 * Ps2[1] * us2[1];
    EF4[4] = fma(Ps2[2], us2[1], Ps2[1] * us2[2]);
    EF4[5] = 2.0 * Ps2[2] * us2[2];
}

// ---- shared-memory helpers ---------------------------------------------------------------------
__device__ __forceinline__ double2 lds2(const double* p) { return *reinterpret_cast<const double2*>(p); }
__device__ __forceinline__ void sts2(double* p, double a, double b) { *reinterpret_cast<double2*>(p) = make_double2(a, b); }

// 8-byte asynchronous global -> shared copy (LDGSTS): the next plane is staged without holding
// registers while the current plane is computed.
__device__ __forceinline__ void cp_async8(double* smem, const double* gmem) {
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(s), "l"(gmem) : "memory");
}
// 16-byte variant for the paired collisionless fields (gp_internal.h, BSTR); .cg: no L1 allocation
__device__ __forceinline__ void cp_async16(double* smem, const double* gmem) {
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gmem) : "memory");
}
__device__ __forceinline__ void prefetch_l2(const double* gmem) { asm volatile("prefetch.global.L2 [%0];" ::"l"(gmem)); }
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// 4 x the (1/4,1/2,1/4) average of three values; the power-of-two normalisations of the face
// velocity (reading G2: 1/4 * 1/4 * 1/2 = 1/32) fold into the flux coefficient (lag_coef).
__device__ __forceinline__ double sum3(double a, double b, double c) { return fma(2.0, b, a + c); }

// Ring slot layout (doubles): pair plane P at offset P*2*PL, cell t at 2*t, two fields per cell:
//   P0 = (density, w*_z)   P1 = (w*_x, w*_y)   P2.. = the remaining fields in pairs
// so that every neighbour access is one 128-bit load.
constexpr int PP = 2 * PL;   // doubles per pair plane

// Values of the x neighbours come from the adjacent lanes (a footprint row is one warp): a
// shuffle costs about a quarter of the shared-memory wavefronts of the load it replaces.  Lanes
// 0 and 31 get their own value back; they are halo columns whose results are never used.
constexpr unsigned FULL = 0xffffffffu;
__device__ __forceinline__ double from_left(double v) { return __shfl_up_sync(FULL, v, 1); }
__device__ __forceinline__ double from_right(double v) { return __shfl_down_sync(FULL, v, 1); }
__device__ __forceinline__ double2 from_left(double2 v) { return make_double2(from_left(v.x), from_left(v.y)); }
__device__ __forceinline__ double2 from_right(double2 v) { return make_double2(from_right(v.x), from_right(v.y)); }
// 4 x the (1/4,1/2,1/4) average along x of a per-thread value
__device__ __forceinline__ double sum3_x(double v) { return sum3(from_left(v), v, from_right(v)); }

// 16 x the 3x3 (omega x omega) average of the second member of pair plane P0 (w*_z) around cell t.
// Must be called by whole warps.
__device__ __forceinline__ double sum9_wz(const double* __restrict__ r, int t) {
    const double2 lo = lds2(r + 2 * (t - FX)), mi = lds2(r + 2 * t), hi = lds2(r + 2 * (t + FX));
    return sum3(sum3_x(lo.y), sum3_x(mi.y), sum3_x(hi.y));
}

// Upwind flux form of one cell in coefficient form:
//   F+ = max(w+,0) f0 + min(w+,0) f+,  F- = max(w-,0) f- + min(w-,0) f0,
//   f' = f0 - th (sum_d F+ - F-) = c0 f0 + sum_q c_q f_q,   max(w,0) = (w+|w|)/2, min(w,0) = (w-|w|)/2.
// The face velocities come in as W = 32 w (unnormalised sums), so the coefficient is th/64.
struct LagCoef { double c0, xm, xp, ym, yp, zm, zp; };

__device__ __forceinline__ LagCoef lag_coef(double th64, double wxm, double wxp, double wym, double wyp, double wzm, double wzp) {
    LagCoef c;
    c.xm = th64 * (wxm + fabs(wxm)); c.xp = th64 * (fabs(wxp) - wxp);
    c.ym = th64 * (wym + fabs(wym)); c.yp = th64 * (fabs(wyp) - wyp);
    c.zm = th64 * (wzm + fabs(wzm)); c.zp = th64 * (fabs(wzp) - wzp);
    const double sum = ((wxp + fabs(wxp)) + (fabs(wxm) - wxm)) + ((wyp + fabs(wyp)) + (fabs(wym) - wym)) +
                       ((wzp + fabs(wzp)) + (fabs(wzm) - wzm));
    c.c0 = fma(-th64, sum, 1.0);
    return c;
}

// Lagrangian stage of one output cell from the U* ring, in two parts so that the ring slot of
// plane j-2 (read only at the thread's own column) can be handed to the asynchronous staging of
// the next plane as early as possible.  Momentum = density * w*, so its update is
// sum_q (c_q dens_q) w*_q.  out = (density, momentum x y z, NO remaining fields).
template <int NO>
__device__ __forceinline__ void lagrange_lower(const double* __restrict__ rm, int t, const LagCoef& c, double out[4 + NO]) {
    const double2 azm = lds2(rm + 2 * t), bzm = lds2(rm + PP + 2 * t);
    const double dzm = c.zm * azm.x;
    out[0] = dzm; out[3] = dzm * azm.y; out[1] = dzm * bzm.x; out[2] = dzm * bzm.y;
#pragma unroll
    for (int P = 0; P < (NO + 1) / 2; ++P) {
        const int o = (2 + P) * PP;
        if (2 * P + 1 < NO) {
            const double2 ezm = lds2(rm + o + 2 * t);
            out[4 + 2 * P] = c.zm * ezm.x; out[5 + 2 * P] = c.zm * ezm.y;
        } else {
            out[4 + 2 * P] = c.zm * rm[o + 2 * t];
        }
    }
}

template <int NO>
__device__ __forceinline__ void lagrange_rest(const double* __restrict__ r0, const double* __restrict__ rp, int t,
                                              const LagCoef& c, double out[4 + NO]) {
    // whole warps only: the x neighbours are fetched by shuffle
    const double2 a0 = lds2(r0 + 2 * t), aym = lds2(r0 + 2 * (t - FX)), ayp = lds2(r0 + 2 * (t + FX));
    const double2 azp = lds2(rp + 2 * t);
#if GP_X_LDS
    const double2 axm = lds2(r0 + 2 * (t - 1)), axp = lds2(r0 + 2 * (t + 1));
#else
    const double2 axm = from_left(a0), axp = from_right(a0);
#endif
    const double d0 = c.c0 * a0.x, dxm = c.xm * axm.x, dxp = c.xp * axp.x, dym = c.ym * aym.x, dyp = c.yp * ayp.x,
                 dzp = c.zp * azp.x;
    out[0] = ((out[0] + d0) + (dxm + dxp)) + ((dym + dyp) + dzp);
    out[3] = fma(dzp, azp.y, fma(dyp, ayp.y, fma(dym, aym.y, fma(dxp, axp.y, fma(dxm, axm.y, fma(d0, a0.y, out[3]))))));
    {
        const double2 b0 = lds2(r0 + PP + 2 * t), bym = lds2(r0 + PP + 2 * (t - FX)), byp = lds2(r0 + PP + 2 * (t + FX));
        const double2 bzp = lds2(rp + PP + 2 * t);
#if GP_X_LDS
        const double2 bxm = lds2(r0 + PP + 2 * (t - 1)), bxp = lds2(r0 + PP + 2 * (t + 1));
#else
        const double2 bxm = from_left(b0), bxp = from_right(b0);
#endif
        out[1] = fma(dzp, bzp.x, fma(dyp, byp.x, fma(dym, bym.x, fma(dxp, bxp.x, fma(dxm, bxm.x, fma(d0, b0.x, out[1]))))));
        out[2] = fma(dzp, bzp.y, fma(dyp, byp.y, fma(dym, bym.y, fma(dxp, bxp.y, fma(dxm, bxm.y, fma(d0, b0.y, out[2]))))));
    }
#pragma unroll
    for (int P = 0; P < (NO + 1) / 2; ++P) {
        const int o = (2 + P) * PP;
        if (2 * P + 1 < NO) {
            const double2 e0 = lds2(r0 + o + 2 * t), eym = lds2(r0 + o + 2 * (t - FX)), eyp = lds2(r0 + o + 2 * (t + FX));
            const double2 ezp = lds2(rp + o + 2 * t);
#if GP_X_LDS
            const double2 exm = lds2(r0 + o + 2 * (t - 1)), exp_ = lds2(r0 + o + 2 * (t + 1));
#else
            const double2 exm = from_left(e0), exp_ = from_right(e0);
#endif
            out[4 + 2 * P] = fma(c.zp, ezp.x, fma(c.yp, eyp.x, fma(c.ym, eym.x, fma(c.xp, exp_.x, fma(c.xm, exm.x, fma(c.c0, e0.x, out[4 + 2 * P]))))));
            out[5 + 2 * P] = fma(c.zp, ezp.y, fma(c.yp, eyp.y, fma(c.ym, eym.y, fma(c.xp, exp_.y, fma(c.xm, exm.y, fma(c.c0, e0.y, out[5 + 2 * P]))))));
        } else {
            const double e0 = r0[o + 2 * t], eym = r0[o + 2 * (t - FX)], eyp = r0[o + 2 * (t + FX)];
            const double ezp = rp[o + 2 * t];
            const double exm = from_left(e0), exp_ = from_right(e0);
            out[4 + 2 * P] = fma(c.zp, ezp, fma(c.yp, eyp, fma(c.ym, eym, fma(c.xp, exp_, fma(c.xm, exm, fma(c.c0, e0, out[4 + 2 * P]))))));
        }
    }
}

// 32 x the face velocities of one output cell (reading G2) from the z-summed (4 x averaged) w*_x,
// w*_y pair plane (s_tz): x faces = sum of the y-summed columns tx-1|tx and tx|tx+1, y faces likewise.
__device__ __forceinline__ void face_vel_xy(const double* __restrict__ s_tz, int t, double& wxm, double& wxp, double& wym,
                                            double& wyp) {
    // whole warps only (shuffles)
    const double2 m0 = lds2(s_tz + 2 * (t - FX)), z0 = lds2(s_tz + 2 * t), p0 = lds2(s_tz + 2 * (t + FX));
    const double a_0 = sum3(m0.x, z0.x, p0.x);
    const double a_m = from_left(a_0), a_p = from_right(a_0);
    const double b_m = sum3_x(m0.y), b_0 = sum3_x(z0.y), b_p = sum3_x(p0.y);
    wxm = a_m + a_0; wxp = a_0 + a_p;
    wym = b_m + b_0; wyp = b_0 + b_p;
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
    const double* src_in;     // gas kernel only: density n of the new collisionless state, or null
    double* src_out;          // ... and where to write the Poisson source rho + n of the new state, or null
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
        for (int o = 16; o > 0; o >>= 1) {
            smax = fmax(smax, __shfl_xor_sync(0xffffffffu, smax, o));
            bad |= __shfl_xor_sync(0xffffffffu, bad, o);
        }
        if (threadIdx.x == 0) {
            atomicMax(smax_bits, (unsigned long long)__double_as_longlong(smax));
            if (bad) atomicOr(flag, 1);
        }
    }
}

#ifdef GP_FUSED_GAS
// =================================================================================================
// Gas: fields rho, mx, my, mz, E.
// Shared planes (of PL doubles): (rho,p) pair 2, vx 1, vy 1, Phi 1, y-flux (P,PV) pair 2,
// ring 3 x 3 pair planes = 18, z-averaged (w*_x,w*_y) pair 2  ->  27 planes = 108 KB.
// The raw U of the next plane is staged (cp.async) in the ring slot that is about to be rewritten.
// =================================================================================================
constexpr int GAS_SLOT = 3 * PP;
constexpr int GAS_PLANES = 2 + 3 + 2 + 3 * 6 + 2;

struct GasCarry {
    double rho, ir, vx, vy, vz, p;        // primitives of the current plane j (own cell)
    double amx, amy, amz, aE;             // U*(j) under construction
    double phi0, phim;                    // Phi(j), Phi(j-1) of the own column
    double Sz_prev, wzp_prev, smax;
    int bad;
};

struct GasShared {
    double *rp, *vx, *vy, *phi, *fy, *ring, *tz;
};

template <bool ST>
__device__ __forceinline__ void gas_iter(const FusedArgs<NGAS>& a, const Foot& f, const PhiCol& pc, const GasShared& S,
                                         GasCarry& c, int j, double tau, double th, double inv2h) {
    const Geo& g = a.g;
    const int t = f.t;
    const double gamma = a.gamma, gm1 = a.gamma - 1.0;
    const double th2 = 0.5 * th, th4 = 0.25 * th;
    const bool zout = g.bcz == GP_BC_OUTFLOW;
    const bool top_copy = !ST && zout && j == g.nz;
    const bool bot_dup = !ST && zout && j == 0;
    const bool do_out = ST || j - 1 >= f.z0;
    const bool do_wzp = ST || j >= f.z0;
    const bool stage_next = ST || j + 1 <= f.z1;

    // B: x and y faces of plane j, each computed once (hi face per thread), in one basic block so
    // that the two solvers interleave.  Row FY-1 has no row above it; its faces are never used.
    double Pyh = 0.0, PVyh = 0.0, gy = 0.0;
    if (f.ty <= FY - 2) {
        const int tr = f.tx < FX - 1 ? t + 1 : t;
        const double2 ry = lds2(S.rp + 2 * (t + FX)), rx = lds2(S.rp + 2 * tr);
        const double vyr = S.vy[t + FX], vxr = S.vx[tr];
        const double phe = S.phi[tr], phn = S.phi[t + FX];
        const double phw = S.phi[f.tx > 0 ? t - 1 : t], phs = S.phi[f.ty > 0 ? t - FX : t];
        double Pxh, PVxh;
        gas_face(gamma, c.rho, c.vy, c.p, ry.x, vyr, ry.y, Pyh, PVyh);
        gas_face(gamma, c.rho, c.vx, c.p, rx.x, vxr, rx.y, Pxh, PVxh);
        sts2(S.fy + 2 * t, Pyh, PVyh);
        const double Pxl = __shfl_up_sync(0xffffffffu, Pxh, 1);
        const double PVxl = __shfl_up_sync(0xffffffffu, PVxh, 1);
        const double gx = (phe - phw) * inv2h;
        gy = (phn - phs) * inv2h;
        const double trg = tau * c.rho * gx;
        const double mx = c.rho * c.vx;
        c.amx = c.amx - th2 * (Pxh - Pxl) - trg;
        c.aE = c.aE - th4 * (PVxh - PVxl) - fma(-0.5 * tau, trg, tau * mx) * gx;
    }
    __syncthreads();

    // C: y-flux difference
    if (f.star_row) {
        const double2 lo = lds2(S.fy + 2 * (t - FX));
        const double trg = tau * c.rho * gy;
        const double my = c.rho * c.vy;
        c.amy = c.amy - th2 * (Pyh - lo.x) - trg;
        c.aE = c.aE - th4 * (PVyh - lo.y) - fma(-0.5 * tau, trg, tau * my) * gy;
    }

    // E: plane j+1 arrives; z face (j, j+1); U*(j) complete -> ring slot j; publish primitives(j+1)
    double* rs = S.ring + ring_slot(j) * GAS_SLOT;
    cp_async_wait_all();
    const double2 s0 = lds2(rs + 2 * t), s1 = lds2(rs + PP + 2 * t), s2 = lds2(rs + 2 * PP + 2 * t);
    const double rho_n = s0.x, mx_n = s0.y, my_n = s1.x, mz_n = s1.y, E_n = s2.x, phi_n = s2.y;
    const double ir_n = frcp(rho_n);
    const double vx_n = mx_n * ir_n, vy_n = my_n * ir_n, vz_n = mz_n * ir_n;
    const double p_n = gm1 * (E_n - 0.5 * fma(mx_n, vx_n, fma(my_n, vy_n, mz_n * vz_n)));
    double Pz = 0.0, PVz = 0.0;
    if (f.star_row) {
        gas_face(gamma, c.rho, c.vz, c.p, rho_n, vz_n, p_n, Pz, PVz);
        double wx, wy, wz, Es, dens;
        if (top_copy) {                       // outflow: U*(nz) := U*(nz-1)
            const double* rq = S.ring + ring_slot(j - 1) * GAS_SLOT;
            const double2 q0 = lds2(rq + 2 * t), q1 = lds2(rq + PP + 2 * t);
            dens = q0.x; wz = q0.y; wx = q1.x; wy = q1.y; Es = rq[2 * PP + 2 * t];
        } else {
            const double gz = (phi_n - c.phim) * inv2h;
            const double trg = tau * c.rho * gz;
            const double mz = c.rho * c.vz;
            const double mzs = c.amz - th2 * Pz - trg;
            Es = c.aE - th4 * PVz - fma(-0.5 * tau, trg, tau * mz) * gz;
            dens = c.rho; wx = c.amx * c.ir; wy = c.amy * c.ir; wz = mzs * c.ir;
        }
        sts2(rs + 2 * t, dens, wz); sts2(rs + PP + 2 * t, wx, wy); rs[2 * PP + 2 * t] = Es;
        if (bot_dup) {                        // outflow: U*(-1) := U*(0)
            double* rg = S.ring + ring_slot(-1) * GAS_SLOT;
            sts2(rg + 2 * t, dens, wz); sts2(rg + PP + 2 * t, wx, wy); rg[2 * PP + 2 * t] = Es;
        }
        if (do_out) {                         // 4 x z-average of w*_x, w*_y for plane j-1
            const double2 wm = lds2(S.ring + ring_slot(j - 2) * GAS_SLOT + PP + 2 * t);
            const double2 w0 = lds2(S.ring + ring_slot(j - 1) * GAS_SLOT + PP + 2 * t);
            sts2(S.tz + 2 * t, sum3(wm.x, w0.x, wx), sum3(wm.y, w0.y, wy));
        }
    }
    sts2(S.rp + 2 * t, rho_n, p_n); S.vx[t] = vx_n; S.vy[t] = vy_n; S.phi[t] = phi_n;
    c.amx = mx_n; c.amy = my_n; c.amz = fma(th2, Pz, mz_n); c.aE = fma(th4, PVz, E_n);
    c.rho = rho_n; c.ir = ir_n; c.vx = vx_n; c.vy = vy_n; c.vz = vz_n; c.p = p_n;
    c.phim = c.phi0; c.phi0 = phi_n;
    __syncthreads();

    if (f.block_fix) {
        if (f.fix) {
#pragma unroll
            for (int P = 0; P < 3; ++P) {
                const double2 v = lds2(rs + P * PP + 2 * f.fix_src);
                sts2(rs + P * PP + 2 * t, v.x, v.y);
                if (bot_dup) sts2(S.ring + ring_slot(-1) * GAS_SLOT + P * PP + 2 * t, v.x, v.y);
            }
            const double2 v = lds2(S.tz + 2 * f.fix_src);
            sts2(S.tz + 2 * t, v.x, v.y);
        }
        __syncthreads();
    }

    // D: Lagrangian stage of plane j-1 (ring planes j-2, j-1, j).  The slot of plane j-2 is read
    // first (own column only) and then handed to the staging of plane j+2.
    double out[NGAS];
    LagCoef lc;
    double n_other = 0.0;
    bool emit = false;
    if (f.out_row) {
        const double Sz_new = sum9_wz(rs, t);             // 16 x
        if (bot_dup) c.Sz_prev = Sz_new;
        if (do_wzp) {
            const double wzp = c.Sz_prev + Sz_new;        // 32 x face velocity between planes j-1 and j
            if (do_out) {
                double wxm, wxp, wym, wyp;
                face_vel_xy(S.tz, t, wxm, wxp, wym, wyp);
                lc = lag_coef(th * 0.015625, wxm, wxp, wym, wyp, c.wzp_prev, wzp);
                // density of the other component for the Poisson source: asked for early, used last
                if (a.src_in && f.is_out) n_other = a.src_in[BSTR * (f.base + (size_t)(j - 1) * f.nxny)];
                lagrange_lower<1>(S.ring + ring_slot(j - 2) * GAS_SLOT, t, lc, out);
                emit = true;
            }
            c.wzp_prev = wzp;
        }
        c.Sz_prev = Sz_new;
    }
    if (stage_next) {
        const int zm = map_safe(j + 2, g.nz, g.bcz);
        const size_t off = f.base + (size_t)zm * f.nxny;
        double* st = S.ring + ring_slot(j + 1) * GAS_SLOT;
        cp_async16(st + 2 * t, a.U[0] + BSTR * off); cp_async16(st + PP + 2 * t, a.U[2] + BSTR * off);   // pairs
        cp_async8(st + 2 * PP + 2 * t, a.U[4] + off);
        cp_async8(st + 2 * PP + 2 * t + 1, phi_ptr(pc, j + 2, zm, g.nz));
    }
    cp_async_commit();
    if (emit) {
        lagrange_rest<1>(S.ring + ring_slot(j - 1) * GAS_SLOT, rs, t, lc, out);
        if (f.is_out) {
            const size_t off = f.base + (size_t)(j - 1) * f.nxny;
#pragma unroll
            for (int P = 0; P < NGASP / 2; ++P)
                *reinterpret_cast<double2*>(a.Un[2 * P] + BSTR * off) = make_double2(out[2 * P], out[2 * P + 1]);
            a.Un[4][off] = out[4];
            if (a.src_out) a.src_out[off] = out[0] + n_other;
            // CFL of the new state (reading G4)
            const double irn = frcp(out[0]);
            const double ux = out[1] * irn, uy = out[2] * irn, uz = out[3] * irn;
            const double pn = gm1 * (out[4] - 0.5 * fma(out[1], ux, fma(out[2], uy, out[3] * uz)));
            const double c2 = gamma * pn * irn;
            const double sp = fmax(fmax(fabs(ux), fabs(uy)), fabs(uz)) + c2 * frsqrt(c2);
            if (!(out[0] > 0.0) || !(pn > 0.0) || !(sp <= 1.7976931348623157e308)) c.bad = 1;
            c.smax = fmax(c.smax, sp);
        }
    }
}

__global__ void GP_KBOUNDS
k_fused_gas(FusedArgs<NGAS> a) {
    extern __shared__ double2 sm2[];
    double* sm = reinterpret_cast<double*>(sm2);
    GasShared S;
    S.rp = sm; S.vx = sm + 2 * PL; S.vy = sm + 3 * PL; S.phi = sm + 4 * PL; S.fy = sm + 5 * PL;
    S.ring = sm + 7 * PL; S.tz = S.ring + 3 * GAS_SLOT;

    const Geo& g = a.g;
    const Foot f = make_foot(g, a.zchunk);
    const int t = f.t;
    const double tau = a.dt_ptr ? *a.dt_ptr : a.dt_val;
    const double th = tau / a.h, inv2h = 0.5 / a.h, gm1 = a.gamma - 1.0;
    const PhiCol pc = phi_col(g, a.phi, f.xv, f.yv, f.xm, f.ym);

    GasCarry c;
    c.Sz_prev = c.wzp_prev = c.smax = 0.0; c.bad = 0;
    {   // prologue: primitives of plane z0-2, then plane z0-1 with the z face between them
        int zm = map_safe(f.z0 - 2, g.nz, g.bcz);
        size_t off = f.base + (size_t)zm * f.nxny;
        double rho = a.U[0][BSTR * off], mx = a.U[1][BSTR * off], my = a.U[2][BSTR * off], mz = a.U[3][BSTR * off], E = a.U[4][off];
        const double phi_a = phi_load(pc, f.z0 - 2, zm, g.nz);
        double ir = frcp(rho);
        const double vz_a = mz * ir;
        // same expression as the main loop, so that a 1-D problem stays bitwise 1-D across the chunk edge
        const double p_a = gm1 * (E - 0.5 * fma(mx, mx * ir, fma(my, my * ir, mz * vz_a)));
        const double rho_a = rho;
        zm = map_safe(f.z0 - 1, g.nz, g.bcz);
        off = f.base + (size_t)zm * f.nxny;
        rho = a.U[0][BSTR * off]; mx = a.U[1][BSTR * off]; my = a.U[2][BSTR * off]; mz = a.U[3][BSTR * off]; E = a.U[4][off];
        const double phi_b = phi_load(pc, f.z0 - 1, zm, g.nz);
        ir = frcp(rho);
        c.rho = rho; c.ir = ir; c.vx = mx * ir; c.vy = my * ir; c.vz = mz * ir;
        c.p = gm1 * (E - 0.5 * fma(mx, c.vx, fma(my, c.vy, mz * c.vz)));
        double Pz, PVz;
        gas_face(a.gamma, rho_a, vz_a, p_a, c.rho, c.vz, c.p, Pz, PVz);
        c.amx = mx; c.amy = my; c.amz = fma(0.5 * th, Pz, mz); c.aE = fma(0.25 * th, PVz, E);
        c.phim = phi_a; c.phi0 = phi_b;
        sts2(S.rp + 2 * t, c.rho, c.p); S.vx[t] = c.vx; S.vy[t] = c.vy; S.phi[t] = phi_b;
        // stage plane z0 where U*(z0-1) will be written
        zm = map_safe(f.z0, g.nz, g.bcz);
        off = f.base + (size_t)zm * f.nxny;
        double* st = S.ring + ring_slot(f.z0 - 1) * GAS_SLOT;
        cp_async16(st + 2 * t, a.U[0] + BSTR * off); cp_async16(st + PP + 2 * t, a.U[2] + BSTR * off);   // pairs
        cp_async8(st + 2 * PP + 2 * t, a.U[4] + off);
        cp_async8(st + 2 * PP + 2 * t + 1, phi_ptr(pc, f.z0, zm, g.nz));
        cp_async_commit();
    }
    __syncthreads();

    int j = f.z0 - 1;
    for (; j <= f.z0 && j <= f.z1; ++j) gas_iter<false>(a, f, pc, S, c, j, tau, th, inv2h);
    for (; j <= f.z1 - 1; ++j) gas_iter<true>(a, f, pc, S, c, j, tau, th, inv2h);
    for (; j <= f.z1; ++j) gas_iter<false>(a, f, pc, S, c, j, tau, th, inv2h);
    cp_async_wait_all();
    block_max_commit(c.smax, c.bad, a.smax_bits, a.flag, S.rp);
}

#endif  // GP_FUSED_GAS

#ifdef GP_FUSED_BME
// =================================================================================================
// Collisionless component: fields n, nu (3), nE_ij (6: xx xy xz yy yz zz).
// Shared planes (of PL doubles): primitives (n,ux) (uy,uz) (Pxx,Pxz) (Pyy,Pyz) pairs 8 + Pxy 1 +
// Phi 1, y-flux (Ps0,Ps1) (Ps2,EF0) (EF1,EF2) (EF3,EF4) pairs 8 + EF5 1, ring 3 x 5 pair planes = 30,
// z-averaged (w*_x,w*_y) pair 2, staged Phi 1  ->  52 planes = 208 KB.
// =================================================================================================
constexpr int BME_SLOT = 5 * PP;
constexpr int BME_PLANES = 10 + 9 + 3 * 10 + 2 + 1;

struct BmeCarry {
    double n, in, u[3], Pi[6];            // primitives of the current plane j (own cell)
    double acc[9];                        // U*(j) under construction: nu (3), nE (6)
    double phi0, phim, phin;              // Phi(j), Phi(j-1), Phi(j+1) of the own column
    double Sz_prev, wzp_prev, smax;
    int bad;
};

struct BmeShared {
    double *nu, *uu, *px, *py, *pxy, *phi, *fy, *ring, *tz, *phst;
};

template <bool ST>
__device__ __forceinline__ void bme_iter(const FusedArgs<NBME>& a, const Foot& f, const PhiCol& pc, const BmeShared& S,
                                         BmeCarry& c, int j, double tau, double th, double inv2h) {
    const Geo& g = a.g;
    const int t = f.t;
    const double th2 = 0.5 * th, th4 = 0.25 * th;
    const bool zout = g.bcz == GP_BC_OUTFLOW;
    const bool top_copy = !ST && zout && j == g.nz;
    const bool bot_dup = !ST && zout && j == 0;
    const bool do_out = ST || j - 1 >= f.z0;
    const bool do_wzp = ST || j >= f.z0;
    const bool stage_next = ST || j + 1 <= f.z1;

    // B: x and y faces of plane j (hi face per thread)
    double Py[3] = {0.0, 0.0, 0.0}, EFy[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    double gx = 0.0, gy = 0.0;
#if GP_BME_MERGE
    {   // both solvers in ONE basic block so that their dependent chains interleave; rows 0 and FY-1
        // (halo rows whose results are never used) run them on whatever they read
        const int tn = t + FX, te = f.tx < FX - 1 ? t + 1 : t;
        const double2 y0 = lds2(S.nu + 2 * tn), y1 = lds2(S.uu + 2 * tn), y2 = lds2(S.py + 2 * tn);
        const double2 x0 = lds2(S.nu + 2 * te), x1 = lds2(S.uu + 2 * te), x2 = lds2(S.px + 2 * te);
        const double pxy_n = S.pxy[tn], pxy_e = S.pxy[te];
        const double ury[3] = {y0.y, y1.x, y1.y}, urx[3] = {x0.y, x1.x, x1.y};
        const double Ply[3] = {c.Pi[1], c.Pi[3], c.Pi[4]}, Plx[3] = {c.Pi[0], c.Pi[1], c.Pi[2]};
        const double Pry[3] = {pxy_n, y2.x, y2.y}, Prx[3] = {x2.x, pxy_e, x2.y};
        double Px[3], EFx[6];
        bme_face<1>(c.n, c.u, Ply, y0.x, ury, Pry, Py, EFy);
        bme_face<0>(c.n, c.u, Plx, x0.x, urx, Prx, Px, EFx);
        double* fy = S.fy;
        sts2(fy + 2 * t, Py[0], Py[1]); sts2(fy + PP + 2 * t, Py[2], EFy[0]);
        sts2(fy + 2 * PP + 2 * t, EFy[1], EFy[2]); sts2(fy + 3 * PP + 2 * t, EFy[3], EFy[4]);
        fy[4 * PP + t] = EFy[5];
#pragma unroll
        for (int q = 0; q < 3; ++q) c.acc[q] -= th2 * (Px[q] - __shfl_up_sync(0xffffffffu, Px[q], 1));
#pragma unroll
        for (int q = 0; q < 6; ++q) c.acc[3 + q] -= th4 * (EFx[q] - __shfl_up_sync(0xffffffffu, EFx[q], 1));
        gx = (S.phi[t + 1] - S.phi[t - 1]) * inv2h;
        gy = (S.phi[t + FX] - S.phi[t - FX]) * inv2h;
    }
#else
    if (f.ty <= FY - 2) {
        const int tn = t + FX;
        const double2 y0 = lds2(S.nu + 2 * tn), y1 = lds2(S.uu + 2 * tn), y2 = lds2(S.py + 2 * tn);
        const double ur[3] = {y0.y, y1.x, y1.y};
        const double Pl[3] = {c.Pi[1], c.Pi[3], c.Pi[4]};
        const double Pr[3] = {S.pxy[tn], y2.x, y2.y};
        bme_face<1>(c.n, c.u, Pl, y0.x, ur, Pr, Py, EFy);
        double* fy = S.fy;
        sts2(fy + 2 * t, Py[0], Py[1]); sts2(fy + PP + 2 * t, Py[2], EFy[0]);
        sts2(fy + 2 * PP + 2 * t, EFy[1], EFy[2]); sts2(fy + 3 * PP + 2 * t, EFy[3], EFy[4]);
        fy[4 * PP + t] = EFy[5];
    }
    if (f.star_row) {
        const int te = f.tx < FX - 1 ? t + 1 : t;
        const double2 x0 = lds2(S.nu + 2 * te), x1 = lds2(S.uu + 2 * te), x2 = lds2(S.px + 2 * te);
        const double ur[3] = {x0.y, x1.x, x1.y};
        const double Pl[3] = {c.Pi[0], c.Pi[1], c.Pi[2]};
        const double Pr[3] = {x2.x, S.pxy[te], x2.y};
        double Px[3], EFx[6];
        bme_face<0>(c.n, c.u, Pl, x0.x, ur, Pr, Px, EFx);
#pragma unroll
        for (int q = 0; q < 3; ++q) c.acc[q] -= th2 * (Px[q] - __shfl_up_sync(0xffffffffu, Px[q], 1));
#pragma unroll
        for (int q = 0; q < 6; ++q) c.acc[3 + q] -= th4 * (EFx[q] - __shfl_up_sync(0xffffffffu, EFx[q], 1));
        gx = (S.phi[t + 1] - S.phi[t - 1]) * inv2h;
        gy = (S.phi[t + FX] - S.phi[t - FX]) * inv2h;
    }
#endif
    __syncthreads();

    // C: y-flux difference, then everything of U*(j) but the upper z face
    if (f.star_row) {
        const double* fy = S.fy + 2 * (t - FX);
        const double2 l0 = lds2(fy), l1 = lds2(fy + PP), l2 = lds2(fy + 2 * PP), l3 = lds2(fy + 3 * PP);
        const double l4 = S.fy[4 * PP + t - FX];
        c.acc[0] -= th2 * (Py[0] - l0.x); c.acc[1] -= th2 * (Py[1] - l0.y); c.acc[2] -= th2 * (Py[2] - l1.x);
        c.acc[3] -= th4 * (EFy[0] - l1.y); c.acc[4] -= th4 * (EFy[1] - l2.x); c.acc[5] -= th4 * (EFy[2] - l2.y);
        c.acc[6] -= th4 * (EFy[3] - l3.x); c.acc[7] -= th4 * (EFy[4] - l3.y); c.acc[8] -= th4 * (EFy[5] - l4);
        // gravity (reading G5): -tau n g_i and -tau n [(u_i - tau g_i/2) g_j + (u_j - tau g_j/2) g_i]
        const double gr[3] = {gx, gy, (c.phin - c.phim) * inv2h};
        double uc[3];
#pragma unroll
        for (int d = 0; d < 3; ++d) uc[d] = fma(-0.5 * tau, gr[d], c.u[d]);
        const double tn = tau * c.n;
#pragma unroll
        for (int d = 0; d < 3; ++d) c.acc[d] = fma(-tn, gr[d], c.acc[d]);
        c.acc[3] = fma(-tn, 2.0 * uc[0] * gr[0], c.acc[3]);
        c.acc[4] = fma(-tn, fma(uc[0], gr[1], uc[1] * gr[0]), c.acc[4]);
        c.acc[5] = fma(-tn, fma(uc[0], gr[2], uc[2] * gr[0]), c.acc[5]);
        c.acc[6] = fma(-tn, 2.0 * uc[1] * gr[1], c.acc[6]);
        c.acc[7] = fma(-tn, fma(uc[1], gr[2], uc[2] * gr[1]), c.acc[7]);
        c.acc[8] = fma(-tn, 2.0 * uc[2] * gr[2], c.acc[8]);
    }

    // E: plane j+1 arrives; z face (j, j+1); U*(j) complete -> ring slot j; publish primitives(j+1)
    double* rs = S.ring + ring_slot(j) * BME_SLOT;
    cp_async_wait_all();
    double Un[NBME];
    {
        const double2 s0 = lds2(rs + 2 * t), s1 = lds2(rs + PP + 2 * t), s2 = lds2(rs + 2 * PP + 2 * t),
                      s3 = lds2(rs + 3 * PP + 2 * t), s4 = lds2(rs + 4 * PP + 2 * t);
        Un[0] = s0.x; Un[1] = s0.y; Un[2] = s1.x; Un[3] = s1.y; Un[4] = s2.x; Un[5] = s2.y;
        Un[6] = s3.x; Un[7] = s3.y; Un[8] = s4.x; Un[9] = s4.y;
    }
    const double phi_n2 = S.phst[t];      // Phi(j+2), staged with plane j+1
    const double n_n = Un[0];
    const double in_n = frcp(n_n);
    const double u_n[3] = {Un[1] * in_n, Un[2] * in_n, Un[3] * in_n};
    double Pi_n[6];
    Pi_n[0] = fma(-Un[1], u_n[0], Un[4]); Pi_n[1] = fma(-Un[1], u_n[1], Un[5]); Pi_n[2] = fma(-Un[1], u_n[2], Un[6]);
    Pi_n[3] = fma(-Un[2], u_n[1], Un[7]); Pi_n[4] = fma(-Un[2], u_n[2], Un[8]); Pi_n[5] = fma(-Un[3], u_n[2], Un[9]);
    double Pz[3] = {0.0, 0.0, 0.0}, EFz[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    if (f.star_row) {
        const double Pl[3] = {c.Pi[2], c.Pi[4], c.Pi[5]};
        const double Pr[3] = {Pi_n[2], Pi_n[4], Pi_n[5]};
        bme_face<2>(c.n, c.u, Pl, n_n, u_n, Pr, Pz, EFz);
        double o[NBME];      // n, w (3), nE (6)
        if (top_copy) {                       // outflow: U*(nz) := U*(nz-1)
            const double* rq = S.ring + ring_slot(j - 1) * BME_SLOT;
            const double2 q0 = lds2(rq + 2 * t), q1 = lds2(rq + PP + 2 * t), q2 = lds2(rq + 2 * PP + 2 * t),
                          q3 = lds2(rq + 3 * PP + 2 * t), q4 = lds2(rq + 4 * PP + 2 * t);
            o[0] = q0.x; o[3] = q0.y; o[1] = q1.x; o[2] = q1.y; o[4] = q2.x; o[5] = q2.y; o[6] = q3.x; o[7] = q3.y;
            o[8] = q4.x; o[9] = q4.y;
        } else {
            o[0] = c.n;
#pragma unroll
            for (int d = 0; d < 3; ++d) o[1 + d] = fma(-th2, Pz[d], c.acc[d]) * c.in;
#pragma unroll
            for (int q = 0; q < 6; ++q) o[4 + q] = fma(-th4, EFz[q], c.acc[3 + q]);
        }
        sts2(rs + 2 * t, o[0], o[3]); sts2(rs + PP + 2 * t, o[1], o[2]); sts2(rs + 2 * PP + 2 * t, o[4], o[5]);
        sts2(rs + 3 * PP + 2 * t, o[6], o[7]); sts2(rs + 4 * PP + 2 * t, o[8], o[9]);
        if (bot_dup) {                        // outflow: U*(-1) := U*(0)
            double* rg = S.ring + ring_slot(-1) * BME_SLOT;
            sts2(rg + 2 * t, o[0], o[3]); sts2(rg + PP + 2 * t, o[1], o[2]); sts2(rg + 2 * PP + 2 * t, o[4], o[5]);
            sts2(rg + 3 * PP + 2 * t, o[6], o[7]); sts2(rg + 4 * PP + 2 * t, o[8], o[9]);
        }
        if (do_out) {                         // 4 x z-average of w*_x, w*_y for plane j-1
            const double2 wm = lds2(S.ring + ring_slot(j - 2) * BME_SLOT + PP + 2 * t);
            const double2 w0 = lds2(S.ring + ring_slot(j - 1) * BME_SLOT + PP + 2 * t);
            sts2(S.tz + 2 * t, sum3(wm.x, w0.x, o[1]), sum3(wm.y, w0.y, o[2]));
        }
    }
    sts2(S.nu + 2 * t, n_n, u_n[0]); sts2(S.uu + 2 * t, u_n[1], u_n[2]); sts2(S.px + 2 * t, Pi_n[0], Pi_n[2]);
    sts2(S.py + 2 * t, Pi_n[3], Pi_n[4]); S.pxy[t] = Pi_n[1]; S.phi[t] = c.phin;
#pragma unroll
    for (int d = 0; d < 3; ++d) c.acc[d] = fma(th2, Pz[d], Un[1 + d]);
#pragma unroll
    for (int q = 0; q < 6; ++q) c.acc[3 + q] = fma(th4, EFz[q], Un[4 + q]);
    c.n = n_n; c.in = in_n;
#pragma unroll
    for (int d = 0; d < 3; ++d) c.u[d] = u_n[d];
#pragma unroll
    for (int q = 0; q < 6; ++q) c.Pi[q] = Pi_n[q];
    c.phim = c.phi0; c.phi0 = c.phin; c.phin = phi_n2;
    __syncthreads();

    if (f.block_fix) {
        if (f.fix) {
#pragma unroll
            for (int P = 0; P < 5; ++P) {
                const double2 v = lds2(rs + P * PP + 2 * f.fix_src);
                sts2(rs + P * PP + 2 * t, v.x, v.y);
                if (bot_dup) sts2(S.ring + ring_slot(-1) * BME_SLOT + P * PP + 2 * t, v.x, v.y);
            }
            const double2 v = lds2(S.tz + 2 * f.fix_src);
            sts2(S.tz + 2 * t, v.x, v.y);
        }
        __syncthreads();
    }

    // D: Lagrangian stage of plane j-1 (ring planes j-2, j-1, j)
    if (f.out_row) {
        const double Sz_new = sum9_wz(rs, t);             // 16 x
        if (bot_dup) c.Sz_prev = Sz_new;
        if (do_wzp) {
            const double wzp = c.Sz_prev + Sz_new;        // 32 x face velocity between planes j-1 and j
            if (do_out) {
                double wxm, wxp, wym, wyp;
                face_vel_xy(S.tz, t, wxm, wxp, wym, wyp);
                const LagCoef lc = lag_coef(th * 0.015625, wxm, wxp, wym, wyp, c.wzp_prev, wzp);
                double out[NBME];
                lagrange_lower<6>(S.ring + ring_slot(j - 2) * BME_SLOT, t, lc, out);
                lagrange_rest<6>(S.ring + ring_slot(j - 1) * BME_SLOT, rs, t, lc, out);
                if (f.is_out) {
                    const size_t off = f.base + (size_t)(j - 1) * f.nxny;
#pragma unroll
                    for (int P = 0; P < NBME / 2; ++P)
                        *reinterpret_cast<double2*>(a.Un[2 * P] + BSTR * off) = make_double2(out[2 * P], out[2 * P + 1]);
                    // CFL of the new state (reading G4): |u_d| + sqrt(3 Pi_dd / n)
                    const double inn = frcp(out[0]);
                    const int dd[3] = {4, 7, 9};
                    if (!(out[0] > 0.0)) c.bad = 1;
#pragma unroll
                    for (int d = 0; d < 3; ++d) {
                        const double ud = out[1 + d] * inn;
                        const double Pdd = fma(-out[1 + d], ud, out[dd[d]]);
                        const double c2 = 3.0 * Pdd * inn;
                        const double sp = fabs(ud) + c2 * frsqrt(c2);
                        if (!(Pdd > 0.0) || !(sp <= 1.7976931348623157e308)) c.bad = 1;
                        c.smax = fmax(c.smax, sp);
                    }
                }
            }
            c.wzp_prev = wzp;
        }
        c.Sz_prev = Sz_new;
    }
    // stage plane j+2 into the slot D just finished with (own column only), and Phi(j+3)
    if (stage_next) {
        const int zm = map_safe(j + 2, g.nz, g.bcz);
        const size_t off = f.base + (size_t)zm * f.nxny;
        double* st = S.ring + ring_slot(j + 1) * BME_SLOT + 2 * t;
#pragma unroll
        for (int P = 0; P < NBME / 2; ++P) cp_async16(st + P * PP, a.U[2 * P] + BSTR * off);     // one pair per copy
        cp_async8(S.phst + t, phi_ptr(pc, j + 3, map_safe(j + 3, g.nz, g.bcz), g.nz));
        // pull plane j+3 into L2 so that the next staging is an L2 hit
        const size_t off3 = f.base + (size_t)map_safe(j + 3, g.nz, g.bcz) * f.nxny;
#pragma unroll
        for (int P = 0; P < NBME / 2; ++P) prefetch_l2(a.U[2 * P] + BSTR * off3);
    }
    cp_async_commit();
}

__global__ void GP_KBOUNDS
k_fused_bme(FusedArgs<NBME> a) {
    extern __shared__ double2 sm2[];
    double* sm = reinterpret_cast<double*>(sm2);
    BmeShared S;
    S.nu = sm; S.uu = sm + 2 * PL; S.px = sm + 4 * PL; S.py = sm + 6 * PL; S.pxy = sm + 8 * PL; S.phi = sm + 9 * PL;
    S.fy = sm + 10 * PL; S.ring = sm + 19 * PL; S.tz = S.ring + 3 * BME_SLOT; S.phst = S.tz + 2 * PL;

    const Geo& g = a.g;
    const Foot f = make_foot(g, a.zchunk);
    const int t = f.t;
    const double tau = a.dt_ptr ? *a.dt_ptr : a.dt_val;
    const double th = tau / a.h, inv2h = 0.5 / a.h;
    const PhiCol pc = phi_col(g, a.phi, f.xv, f.yv, f.xm, f.ym);

    BmeCarry c;
    c.Sz_prev = c.wzp_prev = c.smax = 0.0; c.bad = 0;
    {   // prologue: primitives of plane z0-2, then plane z0-1 with the z face between them
        int zm = map_safe(f.z0 - 2, g.nz, g.bcz);
        size_t off = f.base + (size_t)zm * f.nxny;
        double U0[NBME];
#pragma unroll
        for (int q = 0; q < NBME; ++q) U0[q] = a.U[q][BSTR * off];
        c.phim = phi_load(pc, f.z0 - 2, zm, g.nz);
        const double n_a = U0[0];
        double in = frcp(n_a);
        const double u_a[3] = {U0[1] * in, U0[2] * in, U0[3] * in};
        const double Pz_a[3] = {fma(-U0[1], u_a[2], U0[6]), fma(-U0[2], u_a[2], U0[8]), fma(-U0[3], u_a[2], U0[9])};
        zm = map_safe(f.z0 - 1, g.nz, g.bcz);
        off = f.base + (size_t)zm * f.nxny;
#pragma unroll
        for (int q = 0; q < NBME; ++q) U0[q] = a.U[q][BSTR * off];
        c.phi0 = phi_load(pc, f.z0 - 1, zm, g.nz);
        c.n = U0[0]; c.in = frcp(c.n);
#pragma unroll
        for (int d = 0; d < 3; ++d) c.u[d] = U0[1 + d] * c.in;
        c.Pi[0] = fma(-U0[1], c.u[0], U0[4]); c.Pi[1] = fma(-U0[1], c.u[1], U0[5]); c.Pi[2] = fma(-U0[1], c.u[2], U0[6]);
        c.Pi[3] = fma(-U0[2], c.u[1], U0[7]); c.Pi[4] = fma(-U0[2], c.u[2], U0[8]); c.Pi[5] = fma(-U0[3], c.u[2], U0[9]);
        const double Pr[3] = {c.Pi[2], c.Pi[4], c.Pi[5]};
        double Pz[3], EFz[6];
        bme_face<2>(n_a, u_a, Pz_a, c.n, c.u, Pr, Pz, EFz);
#pragma unroll
        for (int d = 0; d < 3; ++d) c.acc[d] = fma(0.5 * th, Pz[d], U0[1 + d]);
#pragma unroll
        for (int q = 0; q < 6; ++q) c.acc[3 + q] = fma(0.25 * th, EFz[q], U0[4 + q]);
        sts2(S.nu + 2 * t, c.n, c.u[0]); sts2(S.uu + 2 * t, c.u[1], c.u[2]); sts2(S.px + 2 * t, c.Pi[0], c.Pi[2]);
        sts2(S.py + 2 * t, c.Pi[3], c.Pi[4]); S.pxy[t] = c.Pi[1]; S.phi[t] = c.phi0;
        // stage plane z0 where U*(z0-1) will be written
        zm = map_safe(f.z0, g.nz, g.bcz);
        off = f.base + (size_t)zm * f.nxny;
        double* st = S.ring + ring_slot(f.z0 - 1) * BME_SLOT + 2 * t;
#pragma unroll
        for (int P = 0; P < NBME / 2; ++P) cp_async16(st + P * PP, a.U[2 * P] + BSTR * off);
        c.phin = phi_load(pc, f.z0, zm, g.nz);
        cp_async8(S.phst + t, phi_ptr(pc, f.z0 + 1, map_safe(f.z0 + 1, g.nz, g.bcz), g.nz));
        cp_async_commit();
    }
    __syncthreads();

    int j = f.z0 - 1;
    for (; j <= f.z0 && j <= f.z1; ++j) bme_iter<false>(a, f, pc, S, c, j, tau, th, inv2h);
    for (; j <= f.z1 - 1; ++j) bme_iter<true>(a, f, pc, S, c, j, tau, th, inv2h);
    for (; j <= f.z1; ++j) bme_iter<false>(a, f, pc, S, c, j, tau, th, inv2h);
    cp_async_wait_all();
    block_max_commit(c.smax, c.bad, a.smax_bits, a.flag, S.nu);
}

#endif  // GP_FUSED_BME

// -------------------------------------------------------------------------------------------------
// launches
// -------------------------------------------------------------------------------------------------
static int pick_zchunk(const gp_ctx* c, int tiles_xy) {
    // One block per SM: the grid runs in waves of 148 blocks, and every chunk pays about three
    // planes of pipeline fill.  Pick the chunk length that minimises waves x (planes + fill).
    const int nz = c->g.nz;
    int best = nz;
    long long best_cost = -1;
    for (int chunks = 1; chunks <= 64; ++chunks) {
        const int zc = (nz + chunks - 1) / chunks;
        if (zc < 16 && chunks > 1) break;
        const long long blocks = (long long)tiles_xy * ((nz + zc - 1) / zc);
        const long long waves = (blocks + 147) / 148;
        const long long cost = waves * (zc + 3);
        if (best_cost < 0 || cost < best_cost) { best_cost = cost; best = zc; }
    }
    return best;
}

template <int NF, class K>
static int launch_fused_t(gp_ctx* c, K kernel, int f0, int planes, int kid, double dt, const double* d_dt,
                          const double* src_in = nullptr, double* src_out = nullptr) {
    FusedArgs<NF> a;
    a.src_in = src_in; a.src_out = src_out;
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

#ifdef GP_FUSED_GAS
static int launch_gas_impl(gp_ctx* c, double dt, const double* d_dt, const double* src_in, double* src_out) {
    return launch_fused_t<NGAS>(c, k_fused_gas, 0, GAS_PLANES, K_FUSED_GAS, dt, d_dt, src_in, src_out);
}
#endif
#ifdef GP_FUSED_BME
static int launch_bme_impl(gp_ctx* c, double dt, const double* d_dt) {
    return launch_fused_t<NBME>(c, k_fused_bme, NGAS, BME_PLANES, K_FUSED_BME, dt, d_dt);
}
#endif

#ifdef GP_FUSED_GAS
// evaluate the device reciprocal / reciprocal square root on n host-supplied values (self test)
__global__ void k_math_selftest(int n, const double* __restrict__ x, double* __restrict__ rcp, double* __restrict__ rsq) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) { rcp[i] = frcp(x[i]); rsq[i] = frsqrt(x[i]); }
}

static int math_selftest_impl(int n, const double* x, double* rcp, double* rsq) {
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
#endif

}  // namespace GP_FUSED_NS

#ifdef GP_FUSED_GAS
int launch_fused_gas(gp_ctx* c, double dt, const double* d_dt, const double* src_in, double* src_out) {
    return GP_FUSED_NS::launch_gas_impl(c, dt, d_dt, src_in, src_out);
}
int math_selftest(int n, const double* x, double* rcp, double* rsq) { return GP_FUSED_NS::math_selftest_impl(n, x, rcp, rsq); }
#endif
#ifdef GP_FUSED_BME
int launch_fused_bme(gp_ctx* c, double dt, const double* d_dt) { return GP_FUSED_NS::launch_bme_impl(c, dt, d_dt); }
#endif

}  // namespace gp
