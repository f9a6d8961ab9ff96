// Fused hydro step of libgpupegas.so: Eulerian stage and
// Lagrangian stage of one component in ONE pass over HBM, with the CFL
// reduction of the new state (reading G4) in the epilogue.
//
// 2.5-D streaming, warp-specialised.  A block owns an xy footprint of FX x FY = 32 x FY cells
// (28 x (FY-4) output cells plus a two-cell halo) and marches along z.  It runs two groups of warps
// that work on different planes at the same time, so that the shared-memory-heavy Lagrangian stage
// of one plane overlaps the fp64-heavy Eulerian stage of a later one:
//
//   * Eulerian warps ("E"; GP_EROWS = 1: one per footprint row, thread = one cell column; GP_EROWS = 2, the gas
//     kernel: one per two adjacent rows, thread = two cells, the y face between them solved once in registers).
//     Per plane j:
//       B  x and y faces of plane j, each computed ONCE (hi face per thread; the lo face comes
//          from the lane to the left by warp shuffle and from the row below through shared memory);
//       C  flux differences and the gravity source into U*(j), held in registers;
//       E  plane j+1 has landed in the ring slot that U*(j) is about to take: recover its
//          primitives, z face (j, j+1), complete U*(j) and write it (density, w* = momentum*/
//          density, remaining fields) over the staged data -- U* never goes to HBM -- and publish
//          the primitives of plane j+1 for the next B.
//     Rows synchronise with their two neighbours only, through two mbarriers per row (row_arrive_at /
//     mbar_wait_at: "y fluxes written", "primitives published"); there is no block-wide barrier in the loop.
//   * NDW Lagrangian warps ("D"; each serves (FY-4)/NDW output rows, one in the shipped builds).  Per plane j
//     they wait for U*(j), advect plane j-1 from the NS-slot U* ring (4-vertex face velocities as
//     separable (1/4,1/2,1/4) averages, upwind donor-cell fluxes in coefficient form), write
//     U^{n+1}(j-1) to HBM and fold its max signal speed.  They also PRODUCE: as soon as all of them
//     are done with the oldest ring slot, plane j+NS-1 (and Phi(j+NS)) is requested into it: one thread
//     issues one TMA tensor copy (cp.async.bulk.tensor, a 32 x FY x 1 box) per field pair, completing
//     on an mbarrier with a transaction count; no compute thread issues or waits for a copy
//     instruction.  TMA cannot wrap or clamp, so blocks whose footprint reaches over the edge of
//     the grid (and grids with odd nx, whose rows are not 16-byte aligned) stage cell by cell with
//     cp.async on the same mbarrier.
//   * E -> D hand-off: one mbarrier per ring slot ("U*(j) complete"), arrived on by one lane of every
//     E warp.  D -> E: the "landed" mbarrier of the slot.  The E group runs up to NS-3 planes ahead of
//     the D group.  Registers are split between the groups with setmaxnreg.
//
// Ghost cells are index maps (wrap / clamp of the source row, plane or x segment); for outflow the U*
// ghosts are copies of the nearest interior U* (H6), restored in shared memory after E.
// Phi comes from an array padded by two ghost layers (gp_internal.h, PhiPad), filled by the rule of
// the Poisson mode, so its staging needs no case analysis.
//
// Build parameters (set per translation unit by fused_gas.cu, fused_bme.cu and their _od twins): GP_FY, GP_NDW,
// GP_NS, GP_EROWS, GP_REG_E / GP_REG_D, GP_OVERDET, GP_TZREG, GP_EARLYPUB; the measured effect of
// each is recorded in DESIGN.md section 8.
#include <cuda.h>

#include <cstddef>
#include <cstring>
#include <mutex>
#include <new>

#include "gp_internal.h"

namespace gp {
namespace GP_FUSED_NS {

#ifndef GP_FY
#define GP_FY 12
#endif
constexpr int FX = 32, FY = GP_FY, PL = FX * FY;
constexpr int TXO = FX - 4, TYO = FY - 4;
#ifndef GP_NDW
#define GP_NDW 8
#endif
// GP_EROWS: footprint rows per Eulerian warp (1, or 2 adjacent rows per thread in the gas kernel: the y face between
// the two rows stays in registers, half as many row hand-offs)
#ifndef GP_EROWS
#define GP_EROWS 1
#endif
constexpr int EROWS = GP_EROWS;
static_assert(FY % EROWS == 0 && (EROWS == 1 || EROWS == 2), "one or two footprint rows per Eulerian warp");
constexpr int NEW = FY / EROWS;           // Eulerian warps, one per EROWS footprint rows
constexpr int NDW = GP_NDW;               // Lagrangian / producer warps
// setmaxnreg works on aligned groups of four warps: when the registers are re-split the Eulerian group is padded to a
// multiple of four warps; the padding warps take part in nothing but the register split and the final reduction
#ifndef GP_REG_E
#define GP_REG_E 0
#endif
constexpr int NEWP = GP_REG_E ? (NEW + 3) / 4 * 4 : NEW;
constexpr int NTE = NEWP * 32, NTD = NDW * 32, NT = NTE + NTD;
constexpr int DROWS = TYO / NDW;          // output rows per Lagrangian warp
#ifndef GP_NS
#define GP_NS 4
#endif
// GP_OVERDET (contexts created with GP_OD): the kernels also carry the overdetermined system (PAPER.md:41 4th equation): one more gas field
// (rho*eps, paired with the energy), six more collisionless fields (Pi_ij); pressure and dispersion tensor of the
// face solvers come from the carried fields; kappa and the energy balance (G15) sit in
// the epilogue of the Lagrangian stage.
#ifndef GP_OVERDET
#define GP_OVERDET 0
#endif
constexpr bool OD = GP_OVERDET != 0;
// GP_TZREG: the Eulerian threads keep w*_x, w*_y of their own column of the last two planes in registers for the
// z-averaged face-velocity plane instead of reading them back from the ring (32 bytes of shared-memory traffic less
// per thread and plane, 8 registers more)
#ifndef GP_TZREG
#define GP_TZREG 0
#endif
constexpr bool TZREG = GP_TZREG != 0;
// GP_EARLYPUB: stage E publishes the primitives of plane j+1 (and releases the rows waiting for them) as soon as they
// are recovered, before the z face solve and the U* stores, instead of at the end of the stage
#ifndef GP_EARLYPUB
#define GP_EARLYPUB 0
#endif
constexpr bool EARLYPUB = GP_EARLYPUB != 0;
constexpr int NS = GP_NS;                 // slots of the U* ring: planes j-2, j-1, j of the Lagrangian warps and NS - 3 ahead
constexpr int NPHI = NS + 2;              // slots of the Phi ring
constexpr int NTZ = NS - 2;               // buffers of the z-averaged face-velocity plane
static_assert(NS >= 4, "the ring holds three planes for the Lagrangian stage and at least one ahead");
// ring slot / mbarrier phase parity of plane index it (>= 0, counted from the first plane of the block)
__host__ __device__ constexpr int rslot(int it) { return it % NS; }
__host__ __device__ constexpr unsigned rpar(int it) { return (unsigned)(it / NS) & 1u; }
__host__ __device__ constexpr int pslot(int k) { return k % NPHI; }
static_assert(TYO % NDW == 0, "output rows must divide among the Lagrangian warps");

// register budgets after the split (0: leave the launch allocation alone)
#ifndef GP_REG_D
#define GP_REG_D 0
#endif
static_assert(GP_REG_E == 0 || (NEWP % 4 == 0 && NDW % 4 == 0), "setmaxnreg works on warpgroups of four warps");
// the block is launched with 65536 / NT registers per thread rounded down to a multiple of 8; the split must fit in
// that pool, or setmaxnreg.inc waits for ever
static_assert(GP_REG_E == 0 || NTE * GP_REG_E + NTD * GP_REG_D <= NT * (65536 / NT / 8 * 8), "register split exceeds the block's pool");

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

// ---- face solvers ------------------------------------------------------------------------------
// The solvers return DOUBLED face values (2P, 4PV ...) so that the factors 1/2 of the paper's
// formulas fold into the flux coefficients tau/(2h), tau/(4h) (exact power-of-two scalings).
//
// PAPER.md:112, 114 with Z = sqrt(rl rr gamma (pl+pr)/(rl+rr)) = num*r, 1/Z = den*r, r = rsqrt(num*den).
// Out: P2 = 2P, PV4 = 4 P V, V2 = 2V.
__device__ __forceinline__ void gas_face(double gamma, double rl, double vl, double pl, double rr, double vr, double pr,
                                         double& P2, double& PV4, double& V2) {
    const double ps = pl + pr;
    const double num = rl * rr * (gamma * ps), den = rl + rr;
    const double r = frsqrt(num * den);
    const double Z = num * r, iZ = den * r;
    V2 = fma(pl - pr, iZ, vl + vr);
    P2 = fma(vl - vr, Z, ps);
    PV4 = P2 * V2;
}

// PAPER.md:170-178 for a face normal to axis D, bracketed parameters averaged (PAPER.md:180,
// reading G7).  In: n, u[3], Pd[3] = Pi_{xD}, Pi_{yD}, Pi_{zD} of both sides.
// Out: Ps2[3] = 2 Pi*_{.D} (momentum flux), EF4[6] = 4 (Pi*_{jD} u*_i + Pi*_{iD} u*_j) for
// (i,j) = xx xy xz yy yz zz (flux of nE_ij) and us2[3] = 2 u* (PAPER.md:170-172).
// With q = nl nr, s = nl+nr, A = Pl+Pr (= 2a):  [rho] a = q A / s,  Z1 = sqrt([rho] a) = q A r,
// 1/Z1 = s r, 1/a = 2 q s r^2, where r = rsqrt(q A s).
template <int D>
__device__ __forceinline__ void bme_face(double nl, const double ul[3], const double Pl[3],
                                         double nr, const double ur[3], const double Pr[3],
                                         double Ps2[3], double EF4[6], double us2[3]) {
    const double s3 = 1.7320508075688772935, is3 = 0.57735026918962576451;
    const double q = nl * nr, s = nl + nr;
    const double A = Pl[D] + Pr[D];
    const double qA = q * A;
    const double r = frsqrt(qA * s);
    const double Z1 = qA * r, iZ1 = s * r;
    const double ia = (q * s) * (2.0 * r * r);
    const double Z3 = s3 * Z1, iZ3 = is3 * iZ1;
    const double DP = Pl[D] - Pr[D], DU = ul[D] - ur[D];
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

// ---- shared-memory, barrier and copy helpers ---------------------------------------------------
__device__ __forceinline__ double2 lds2(const double* p) { return *reinterpret_cast<const double2*>(p); }
__device__ __forceinline__ void sts2(double* p, double a, double b) { *reinterpret_cast<double2*>(p) = make_double2(a, b); }
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(unsigned long long* b, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned long long* b) {
    asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.shared::cta.b64 st, [%0];\n\t}" ::"r"(smem_u32(b)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned long long* b, unsigned bytes) {
    asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.expect_tx.shared::cta.b64 st, [%0], %1;\n\t}" ::"r"(smem_u32(b)), "r"(bytes)
                 : "memory");
}
// Wait for the phase of given parity of the mbarrier at shared address base + OFF (bytes; an immediate, so that no
// second address register stays live across the loop).  try_wait suspends the warp for up to the hinted time, so a
// waiting warp issues a poll only now and then instead of spinning on the issue port of the working warps.
template <int OFF = 0>
__device__ __forceinline__ void mbar_wait_at(unsigned base, unsigned parity) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "W_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0+%3], %1, %2;\n\t"
        "@p bra D_%=;\n\t"
        "bra W_%=;\n\t"
        "D_%=:\n\t}" ::"r"(base), "r"(parity), "r"(0x989680), "n"(OFF)
        : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* b, unsigned parity) { mbar_wait_at<0>(smem_u32(b), parity); }
template <int OFF = 0>
__device__ __forceinline__ void mbar_arrive_at(unsigned base) {
    asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.shared::cta.b64 st, [%0+%1];\n\t}" ::"r"(base), "n"(OFF) : "memory");
}
// Neighbouring Eulerian warps (footprint rows r, r+1) hand data to each other through two mbarriers per row, one
// arrival (lane 0 of the producing row) per plane, phase parity = plane parity: yrdy[r] "the y fluxes of row r are
// written" (row r+1 waits before stage C) and prdy[r] "the primitives of the next plane of row r are published" (row
// r-1 waits before its next stage B).  Each also orders the overwrite that follows it: row r+1 publishes new primitives
// only after row r has read the old ones, row r rewrites its y fluxes only after row r+1 has read them.  No
// block-wide barrier is left in the Eulerian group.
template <int OFF>
__device__ __forceinline__ void row_arrive_at(unsigned base) {
    __syncwarp();
    if ((threadIdx.x & 31) == 0) mbar_arrive_at<OFF>(base);
}
// barrier among the warps of one group: one lane per warp arrives, everybody waits for the phase
__device__ __forceinline__ void group_sync(unsigned long long* b, unsigned parity) {
    __syncwarp();
    if ((threadIdx.x & 31) == 0) mbar_arrive(b);
    mbar_wait(b, parity);
}
// the arrival is triggered when every cp.async this thread issued before has completed
__device__ __forceinline__ void mbar_arrive_on_cp_async(unsigned long long* b) {
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(b)) : "memory");
}
// order earlier generic-proxy accesses to shared memory before later async-proxy (bulk copy) writes
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// global -> shared TMA tensor copy of one 3-D box (SASS UTMALDG); completes the box's bytes on the mbarrier's
// transaction count.  Coordinates are in elements of the map, innermost first.  smem: 128-byte aligned.
__device__ __forceinline__ void tma_load_3d(void* smem, const CUtensorMap* tm, int c0, int c1, int c2, unsigned long long* bar) {
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(
                     smem_u32(smem)),
                 "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void cp_async8(double* smem, const double* gmem) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_u32(smem)), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async16(double* smem, const double* gmem) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(smem)), "l"(gmem) : "memory");
}

template <int R>
__device__ __forceinline__ void reg_alloc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(R)); }
template <int R>
__device__ __forceinline__ void reg_dealloc() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(R)); }

// 4 x the (1/4,1/2,1/4) average of three values; the power-of-two normalisations of the face
// velocity (reading G2: 1/4 * 1/4 * 1/2 = 1/32) fold into the flux coefficient (lag_coef).
__device__ __forceinline__ double sum3(double a, double b, double c) { return fma(2.0, b, a + c); }

// Ring slot layout (doubles): pair plane P at offset P*2*PL, cell t at 2*t, two fields per cell:
//   P0 = (density, w*_z)   P1 = (w*_x, w*_y)   P2.. = the remaining fields in pairs (the gas energy: one
//   plain plane, cell t at t) so that every neighbour access is one 128-bit load.
// Before U*(j) is written there the slot holds the raw state of plane j+1 in the HBM pairing
// (density, m_x) (m_y, m_z) ..., as the copies deliver it.
constexpr int PP = 2 * PL;   // doubles per pair plane

// Values of the x neighbours come from the adjacent lanes (a footprint row is one warp).  Lanes
// 0 and 31 get their own value back; they are halo columns whose results are never used.
constexpr unsigned FULL = 0xffffffffu;
__device__ __forceinline__ double from_left(double v) { return __shfl_up_sync(FULL, v, 1); }
__device__ __forceinline__ double from_right(double v) { return __shfl_down_sync(FULL, v, 1); }
// 4 x the (1/4,1/2,1/4) average along x of a per-thread value
__device__ __forceinline__ double sum3_x(double v) { return sum3(from_left(v), v, from_right(v)); }

// 16 x the 3x3 (omega x omega) average of the second member of pair plane P0 (w*_z) around cell t.
// Must be called by whole warps.
__device__ __forceinline__ double sum9_wz(const double* __restrict__ r, int t) {
    const double2 lo = lds2(r + 2 * (t - FX)), mi = lds2(r + 2 * t), hi = lds2(r + 2 * (t + FX));
    return sum3_x(sum3(lo.y, mi.y, hi.y));       // rows first: one exchange along x instead of three
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

// Lagrangian stage of one output cell, neighbour by neighbour: out += c_q * U*_q for one neighbour cell tq of
// ring slot r (PAPER.md:124, 128 in the coefficient form above).  Momentum = density * w*, so its update is
// (c_q dens_q) w*_q.  NP2 = number of pair planes after P0, P1; LAST1: one more plain plane follows them.
// out = (density, momentum x y z, the remaining fields).  INIT: out = ... instead of out += ...
// An upwind scheme reads a neighbour only where the flow comes from it: c_q = 0 on the downwind side, and when
// that holds for every output lane of the warp the caller skips the neighbour altogether (lag_needed).
template <int NP2, bool LAST1, bool INIT>
__device__ __forceinline__ void lagrange_add(const double* __restrict__ r, int tq, double cq,
                                             double out[4 + 2 * NP2 + (LAST1 ? 1 : 0)]) {
    const double2 a = lds2(r + 2 * tq), b = lds2(r + PP + 2 * tq);
    double2 e[NP2 > 0 ? NP2 : 1];
#pragma unroll
    for (int P = 0; P < NP2; ++P) e[P] = lds2(r + (2 + P) * PP + 2 * tq);
    double el = 0.0;
    if (LAST1) el = r[(2 + NP2) * PP + tq];
    const double d = cq * a.x;
    if (INIT) {
        out[0] = d; out[3] = d * a.y; out[1] = d * b.x; out[2] = d * b.y;
#pragma unroll
        for (int P = 0; P < NP2; ++P) { out[4 + 2 * P] = cq * e[P].x; out[5 + 2 * P] = cq * e[P].y; }
        if (LAST1) out[4 + 2 * NP2] = cq * el;
    } else {
        out[0] += d; out[3] = fma(d, a.y, out[3]); out[1] = fma(d, b.x, out[1]); out[2] = fma(d, b.y, out[2]);
#pragma unroll
        for (int P = 0; P < NP2; ++P) { out[4 + 2 * P] = fma(cq, e[P].x, out[4 + 2 * P]); out[5 + 2 * P] = fma(cq, e[P].y, out[5 + 2 * P]); }
        if (LAST1) out[4 + 2 * NP2] = fma(cq, el, out[4 + 2 * NP2]);
    }
}
// does any output lane of the warp take anything from this neighbour?
__device__ __forceinline__ bool lag_needed(double cq, bool lane_out) {
    return __any_sync(FULL, lane_out && cq != 0.0) != 0;
}

// 32 x the face velocities of one output cell (reading G2) from the z-summed (4 x averaged) w*_x,
// w*_y pair plane (s_tz): x faces = sum of the y-summed columns tx-1|tx and tx|tx+1, y faces likewise.
__device__ __forceinline__ void face_vel_xy(const double* __restrict__ s_tz, int t, double& wxm, double& wxp, double& wym,
                                            double& wyp) {
    // whole warps only (shuffles)
    const double2 m0 = lds2(s_tz + 2 * (t - FX)), z0 = lds2(s_tz + 2 * t), p0 = lds2(s_tz + 2 * (t + FX));
    const double a_0 = sum3(m0.x, z0.x, p0.x);
    const double a_m = from_left(a_0), a_p = from_right(a_0);
    wxm = a_m + a_0; wxp = a_0 + a_p;
    wym = sum3_x(m0.y + z0.y); wyp = sum3_x(z0.y + p0.y);   // the two-row sums first: two exchanges along x instead of three
}

// tensor maps of a launch: the field pairs (then the gas energy) of U, and the padded Phi
template <int NF>
struct FusedArgs {
    alignas(64) CUtensorMap tm[(NF + 1) / 2 + 1];
    int use_tma;              // the maps are valid (even nx, encode succeeded)
    Geo g;
    const double* U[NF];
    double* Un[NF];
    PhiPad phi;
    double h, gamma, dt_val;
    const double* dt_ptr;
    int zchunk;
    unsigned long long* smax_bits;
    int* flag;
    const double* src_in;     // gas kernel only: density n of the new collisionless state, or null
    double* src_out;          // ... and where to write the Poisson source rho + n of the new state, or null
    int balance;              // GP_OD: apply the energy balance (G15) to the new state
    double* kappa;            // GP_OD: += sum over cells of this component's kappa integrand, before the balance
};

// Small per-block tables (shared memory, written once by thread 0).
struct alignas(128) BlockTab {
    unsigned long long landed[NS];     // staged plane (+ Phi) has arrived in ring slot s
    unsigned long long ufull[NS];      // U* of ring slot s is complete
    unsigned long long pro;            // the three Phi planes of the prologue have arrived
    unsigned long long dsync, esync;   // group barriers of the Lagrangian / the Eulerian warps
    unsigned long long yrdy[FY], prdy[FY];   // row hand-offs of the Eulerian warps (see row_arrive)
    long long rowoff[FY];              // nx * (mapped y of footprint row)
    long long phirow[FY];              // pitch * (padded y of footprint row)
    int phi_len;                       // doubles of a Phi row that exist in the padded array
    int percell;                       // 1: stage cell by cell (cp.async), 0: TMA boxes
};

struct Blk {
    int x0, y0, z0, z1;
    bool block_fix;
};

__device__ __forceinline__ Blk make_blk(const Geo& g, int zchunk) {
    Blk b;
    b.x0 = blockIdx.x * TXO; b.y0 = blockIdx.y * TYO;
    b.z0 = blockIdx.z * zchunk;
    b.z1 = min(g.nz, b.z0 + zchunk);
    b.block_fix = (g.bcx == GP_BC_OUTFLOW && (b.x0 == 0 || b.x0 + TXO >= g.nx)) ||
                  (g.bcy == GP_BC_OUTFLOW && (b.y0 == 0 || b.y0 + TYO >= g.ny));
    return b;
}

__device__ void build_tab(BlockTab* T, const Geo& g, const PhiPad& phi, const Blk& b, int use_tma) {
    for (int r = 0; r < FY; ++r) {
        T->rowoff[r] = (long long)g.nx * map_safe(b.y0 - 2 + r, g.ny, g.bcy);
        T->phirow[r] = (long long)phi.pitch * min(b.y0 + r, g.ny + 3);
    }
    T->phi_len = min(FX, phi.pitch - b.x0);
    // a TMA box neither wraps nor clamps: the footprint must lie inside the grid
    const bool inside = b.x0 - 2 >= 0 && b.x0 - 2 + FX <= g.nx && b.y0 - 2 >= 0 && b.y0 - 2 + FY <= g.ny;
    T->percell = (use_tma && inside) ? 0 : 1;
}

// Producer (Lagrangian warps): request plane kz of the state into ring slot `dst` (layout above: NPAIR pair
// planes, then one plain plane if LAST1).  TMA mode: thread 0 of the group issues one box per plane.
template <int NPAIR, bool LAST1, int NF>
__device__ __forceinline__ void stage_state(const FusedArgs<NF>& a, const BlockTab* T, const Blk& b, double* dst, int kz,
                                            unsigned long long* bar, int dtid) {
    const Geo& g = a.g;
    const int zm = map_safe(kz, g.nz, g.bcz);
    if (!T->percell) {
        if (dtid == 0) {
#pragma unroll
            for (int P = 0; P < NPAIR; ++P) tma_load_3d(dst + P * PP, &a.tm[P], 2 * (b.x0 - 2), b.y0 - 2, zm, bar);
            if (LAST1) tma_load_3d(dst + NPAIR * PP, &a.tm[NPAIR], b.x0 - 2, b.y0 - 2, zm, bar);
        }
    } else {
        const long long zoff = (long long)zm * g.nx * g.ny;
        for (int c = dtid; c < PL; c += NTD) {
            const int row = c / FX, tx = c % FX;
            const long long cell = zoff + T->rowoff[row] + map_safe(b.x0 - 2 + tx, g.nx, g.bcx);
#pragma unroll
            for (int P = 0; P < NPAIR; ++P) cp_async16(dst + P * PP + 2 * c, a.U[2 * P] + BSTR * cell);
            if (LAST1) cp_async8(dst + NPAIR * PP + c, a.U[2 * NPAIR] + cell);
        }
    }
}

// ... and plane kz of Phi into its ring slot (PL doubles).
template <int NF>
__device__ __forceinline__ void stage_phi(const FusedArgs<NF>& a, const BlockTab* T, const Blk& b, double* dst, int kz,
                                          unsigned long long* bar, int dtid) {
    const PhiPad& p = a.phi;
    if (!T->percell) {
        if (dtid == 0) tma_load_3d(dst, &a.tm[(NF + 1) / 2], b.x0, b.y0, kz + 2, bar);
    } else {
        const double* src = p.p + (long long)p.pitch * p.py * (kz + 2) + b.x0;
        for (int c = dtid; c < PL; c += NTD) {
            const int row = c / FX, tx = c % FX;
            cp_async8(dst + c, src + T->phirow[row] + min(tx, T->phi_len - 1));
        }
    }
}

// block maximum of the signal speed -> one atomicMax of the bit pattern (speeds are >= 0)
// (GP_OD: and the block's sum of the kappa integrand -> one atomicAdd)
__device__ __forceinline__ void block_max_commit(double smax, int bad, unsigned long long* smax_bits, int* flag,
                                                 double* scratch, double kap = 0.0, double* kappa = nullptr) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        smax = fmax(smax, __shfl_xor_sync(0xffffffffu, smax, o));
        bad |= __shfl_xor_sync(0xffffffffu, bad, o);
        if (OD) kap += __shfl_xor_sync(0xffffffffu, kap, o);
    }
    __syncthreads();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    constexpr int NW = NT / 32;
    int* sbad = (int*)(scratch + NW);
    double* skap = scratch + 2 * NW;
    if (lane == 0) { scratch[warp] = smax; sbad[warp] = bad; if (OD) skap[warp] = kap; }
    __syncthreads();
    if (warp == 0) {
        smax = lane < NW ? scratch[lane] : 0.0;
        bad = lane < NW ? sbad[lane] : 0;
        kap = (OD && lane < NW) ? skap[lane] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            smax = fmax(smax, __shfl_xor_sync(0xffffffffu, smax, o));
            bad |= __shfl_xor_sync(0xffffffffu, bad, o);
            if (OD) kap += __shfl_xor_sync(0xffffffffu, kap, o);
        }
        if (lane == 0) {
            atomicMax(smax_bits, (unsigned long long)__double_as_longlong(smax));
            if (bad) atomicOr(flag, 1);
            if (OD && kappa) atomicAdd(kappa, kap);
        }
    }
}

// Per-thread geometry of an Eulerian thread (one footprint cell column).
struct Foot {
    int tx, ty, t, xv, yv;
    size_t base, nxny;
    bool star_row, fix;
    int fix_src;
    unsigned tabbar;     // shared address of the block table (= of landed[0])
    unsigned rowbar;     // shared address of yrdy[ty - 1]; the row's other hand-off barriers sit at the offsets below
};
// byte offsets from Foot::rowbar: y fluxes of the row below / of this row, primitives of this row / of the row above
constexpr int OY_LO = 0, OY_OWN = 8, OY_UP = 16, OP_LO = 8 * FY, OP_OWN = 8 + 8 * FY, OP_UP = 16 + 8 * FY;
static_assert(offsetof(BlockTab, landed) == 0 && offsetof(BlockTab, ufull) == 8 * NS, "ring barriers are addressed from the table base");
static_assert(offsetof(BlockTab, prdy) == offsetof(BlockTab, yrdy) + 8 * FY, "row barriers are addressed from yrdy");

// row: footprint row of the thread (the q-th row of warp w is EROWS * w + q); the hand-off barriers are per warp
__device__ __forceinline__ Foot make_foot(const Geo& g, const Blk& b, const BlockTab* T, int row) {
    Foot f;
    f.tx = threadIdx.x & 31; f.ty = row; f.t = f.ty * FX + f.tx;
    f.xv = b.x0 - 2 + f.tx; f.yv = b.y0 - 2 + f.ty;
    f.nxny = (size_t)g.nx * g.ny;
    f.base = (size_t)map_safe(f.xv, g.nx, g.bcx) + (size_t)g.nx * map_safe(f.yv, g.ny, g.bcy);
    f.star_row = f.ty >= 1 && f.ty <= FY - 2;
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
    f.tabbar = smem_u32(T);
    f.rowbar = smem_u32(&T->yrdy[0]) + 8 * ((int)(threadIdx.x >> 5) - 1);
    return f;
}

// Per-thread state of a Lagrangian thread: DROWS output cells (rows 2 + w + NDW q of the footprint, column lane).
struct LagRows {
    double Sz_prev[DROWS], wzp_prev[DROWS], pre[DROWS];
    double smax, kap;
    int bad;
};

// The Lagrangian warps' whole loop, prologue included (see the header).  Traits TR supply the component's
// layout.  Per plane j (it = j - (z0-1)): wait for U*(j); face velocities and upwind coefficients of the warp's
// rows; the part of the update that reads ring slot it+2 (plane j-2, own column); hand that slot over: it takes
// the staged plane j+3 (consumed by E(j+2), two planes ahead of the Eulerian warps); then the rest.
template <class TR, int NF>
__device__ __forceinline__ void lag_warps(const FusedArgs<NF>& a, BlockTab* T, const Blk& b, double* ring, double* tz,
                                          double* phir, double th, LagRows& L) {
    const Geo& g = a.g;
    const int dtid = threadIdx.x - NTE, dw = dtid >> 5, lane = dtid & 31;
    const int j0 = b.z0 - 1;
    const bool bulk = !T->percell;
    constexpr unsigned UBYTES = PL * (16 * TR::NPAIR + (TR::LAST1 ? 8 : 0)), PBYTES = PL * 8;   // one staged plane: state, Phi
    const bool zout = g.bcz == GP_BC_OUTFLOW;
    const size_t nxny = (size_t)g.nx * g.ny;
    const bool lane_out = lane >= 2 && lane <= FX - 3;
    bool row_out[DROWS];         // this thread's cell of row q is an output cell of the grid, at row_off[q] in its plane
    size_t row_off[DROWS];
#pragma unroll
    for (int q = 0; q < DROWS; ++q) {
        const int xv = b.x0 - 2 + lane, yv = b.y0 + dw + NDW * q;
        row_out[q] = lane_out && xv < g.nx && yv < g.ny;
        row_off[q] = (size_t)xv + (size_t)g.nx * yv;
        L.Sz_prev[q] = L.wzp_prev[q] = L.pre[q] = 0.0;
    }
    L.smax = 0.0; L.kap = 0.0; L.bad = 0;
    // prologue: Phi(z0-2 .. z0) for the first B and C, then the bundles (U(k+1), Phi(k+2)) of the first NS - 2 planes
    // k = z0-1 ... into ring slots 0 ...; E(k) consumes bundle k
    if (bulk && dtid == 0) mbar_arrive_expect_tx(&T->pro, 3 * PBYTES);
    __syncwarp();
    for (int k = 0; k < 3; ++k) stage_phi(a, T, b, phir + k * PL, b.z0 - 2 + k, &T->pro, dtid);
    if (!bulk) mbar_arrive_on_cp_async(&T->pro);
    for (int i = 0; i < NS - 2 && j0 + i <= b.z1; ++i) {
        const bool with_phi = j0 + i + 1 <= b.z1;        // C(k+1) exists and needs Phi(k+2)
        if (bulk && dtid == 0) mbar_arrive_expect_tx(&T->landed[i], UBYTES + (with_phi ? PBYTES : 0u));
        __syncwarp();
        stage_state<TR::NPAIR, TR::LAST1>(a, T, b, ring + i * TR::SLOT, j0 + i + 1, &T->landed[i], dtid);
        if (with_phi) stage_phi(a, T, b, phir + pslot(i + 3) * PL, j0 + i + 2, &T->landed[i], dtid);
        if (!bulk) mbar_arrive_on_cp_async(&T->landed[i]);
    }

    for (int j = j0; j <= b.z1; ++j) {
        const int it = j - j0;
        const bool bot_dup = zout && j == 0;
        const bool do_out = j - 1 >= b.z0;
        const bool do_wzp = j >= b.z0;
        const double* rs = ring + rslot(it) * TR::SLOT;
        const double* r0 = ring + rslot(it + NS - 1) * TR::SLOT;
        const double* rm = ring + rslot(it + NS - 2) * TR::SLOT;
        const double* tzj = tz + (it % NTZ) * PP;
        mbar_wait(&T->ufull[rslot(it)], rpar(it));      // U*(j) complete

        const int kb = j + NS - 2;                // the plane whose bundle (U(kb+1), Phi(kb+2)) takes the freed slot
        const bool more = kb <= b.z1;             // E(kb) exists
        const bool more_phi = kb + 1 <= b.z1;     // C(kb+1) exists
#pragma unroll
        for (int q = 0; q < DROWS; ++q) {
            const int t = (2 + dw + NDW * q) * FX + lane;
            LagCoef lc;
            double out[NF];
            bool emit = false;
            const bool is_out = row_out[q];
            const size_t off = row_off[q] + (size_t)(j - 1) * nxny;
            // one plane ahead: what this row's NEXT output cell needs from global memory besides the ring
            const double pre = L.pre[q];
            L.pre[q] = TR::early(a, off + nxny, is_out && do_wzp && j + 1 <= b.z1);
            const double Sz_new = sum9_wz(rs, t);             // 16 x
            if (bot_dup) L.Sz_prev[q] = Sz_new;
            if (do_wzp) {
                const double wzp = L.Sz_prev[q] + Sz_new;      // 32 x face velocity between planes j-1 and j
                if (do_out) {
                    double wxm, wxp, wym, wyp;
                    face_vel_xy(tzj, t, wxm, wxp, wym, wyp);
                    lc = lag_coef(th * 0.015625, wxm, wxp, wym, wyp, L.wzp_prev[q], wzp);
                    // centre first (always needed), then plane j-2, whose slot is handed over below
                    lagrange_add<TR::NP2, TR::LAST1, true>(r0, t, lc.c0, out);
                    if (lag_needed(lc.zm, lane_out)) lagrange_add<TR::NP2, TR::LAST1, false>(rm, t, lc.zm, out);
                    emit = true;
                }
                L.wzp_prev[q] = wzp;
            }
            L.Sz_prev[q] = Sz_new;

            // After the last row's lower part the ring slot of plane j-2 is no longer needed by this warp; when that
            // holds for all of them it takes the bundle of plane kb = j-2+NS
            if (q == DROWS - 1 && more) {
                unsigned long long* land = &T->landed[rslot(it + NS - 2)];
                double* dst = ring + rslot(it + NS - 2) * TR::SLOT;
                double* pdst = phir + pslot(it + NS + 1) * PL;
                if (bulk) fence_proxy_async();
                group_sync(&T->dsync, it & 1);
                if (bulk) {
                    if (dtid == 0) {
                        mbar_arrive_expect_tx(land, UBYTES + (more_phi ? PBYTES : 0u));
                        stage_state<TR::NPAIR, TR::LAST1>(a, T, b, dst, kb + 1, land, dtid);
                        if (more_phi) stage_phi(a, T, b, pdst, kb + 2, land, dtid);
                    }
                } else {
                    stage_state<TR::NPAIR, TR::LAST1>(a, T, b, dst, kb + 1, land, dtid);
                    if (more_phi) stage_phi(a, T, b, pdst, kb + 2, land, dtid);
                    mbar_arrive_on_cp_async(land);
                }
            }

            if (emit) {
                if (lag_needed(lc.xm, lane_out)) lagrange_add<TR::NP2, TR::LAST1, false>(r0, t - 1, lc.xm, out);
                if (lag_needed(lc.xp, lane_out)) lagrange_add<TR::NP2, TR::LAST1, false>(r0, t + 1, lc.xp, out);
                if (lag_needed(lc.ym, lane_out)) lagrange_add<TR::NP2, TR::LAST1, false>(r0, t - FX, lc.ym, out);
                if (lag_needed(lc.yp, lane_out)) lagrange_add<TR::NP2, TR::LAST1, false>(r0, t + FX, lc.yp, out);
                if (lag_needed(lc.zp, lane_out)) lagrange_add<TR::NP2, TR::LAST1, false>(rs, t, lc.zp, out);
                if (is_out) TR::emit(a, off, out, pre, L.smax, L.bad, L.kap);
            }
        }
    }
}

#ifdef GP_FUSED_GAS
// =================================================================================================
// Gas: fields rho, mx, my, mz, E.
// Shared planes (of PL doubles): (rho,p) pair 2, vx 1, vy 1, Phi ring 8, y-flux (P,PV) pair 2,
// U* ring 4 x (2 pair planes + 1 plain) = 20, z-averaged (w*_x,w*_y) pair 2 x 2 = 4  ->  38 planes.
// =================================================================================================
// GP_OD: one more field, rho*eps, paired with the energy: (rho E, rho eps) in HBM and in the ring; the y-flux exchange
// carries 2V as a third value.
constexpr int NFG = NGAS + (OD ? NODG : 0);
constexpr int IEPS = OD ? NGAS : 0;       // rho*eps among the fields (only used under GP_OD; in range either way)
struct GasTraits {
    static constexpr int NPAIR = OD ? 3 : 2, NP2 = OD ? 1 : 0;
    static constexpr bool LAST1 = !OD;
    static constexpr int SLOT = OD ? 3 * PP : 2 * PP + PL;
    static constexpr int PLANES = 2 + 1 + 1 + NPHI + (OD ? 3 : 2) + NS * (OD ? 6 : 5) + 2 * NTZ;
    // density of the other component for the Poisson source, asked for one plane before it is used
    __device__ static __forceinline__ double early(const FusedArgs<NFG>& a, size_t off, bool is_out) {
        return (a.src_in && is_out) ? a.src_in[BSTR * off] : 0.0;
    }
    __device__ static __forceinline__ void emit(const FusedArgs<NFG>& a, size_t off, double out[NFG], double n_other, double& smax,
                                                int& bad, double& kap) {
        const double gm1 = a.gamma - 1.0;
        const double irn = frcp(out[0]);
        double ux = out[1] * irn, uy = out[2] * irn, uz = out[3] * irn;
        double kin = 0.5 * fma(out[1], ux, fma(out[2], uy, out[3] * uz));
        if (OD) {
            // correctness check of the state as the two stages left it, then the energy balance (G15)
            const double e_tot = out[4] - kin;            // rho eps as the total energy implies it
            kap += fabs(e_tot - out[IEPS]);
            if (a.balance) {
                if (e_tot > 0.0) {
                    out[IEPS] = e_tot;
                } else {                                  // gas-vacuum border: the carried internal energy wins
                    const double kin_new = out[4] - out[IEPS];
                    if (kin_new > 0.0 && kin > 0.0) {
                        const double sc = sqrt(kin_new / kin);
                        out[1] *= sc; out[2] *= sc; out[3] *= sc;
                        ux *= sc; uy *= sc; uz *= sc;
                        kin = 0.5 * fma(out[1], ux, fma(out[2], uy, out[3] * uz));
                    } else {
                        out[1] = out[2] = out[3] = 0.0; ux = uy = uz = 0.0; kin = 0.0;
                        out[4] = out[IEPS];
                    }
                }
            }
        }
#pragma unroll
        for (int P = 0; P < NPAIR; ++P)
            *reinterpret_cast<double2*>(a.Un[2 * P] + BSTR * off) = make_double2(out[2 * P], out[2 * P + 1]);
        if (LAST1) a.Un[4][off] = out[4];
        if (a.src_out) a.src_out[off] = out[0] + n_other;
        // CFL of the new state (reading G4)
        const double pn = OD ? gm1 * out[IEPS] : gm1 * (out[4] - kin);   // GP_OD: the carried pressure (reading G16)
        const double c2 = a.gamma * pn * irn;
        const double sp = fmax(fmax(fabs(ux), fabs(uy)), fabs(uz)) + c2 * frsqrt(c2);
        if (!(out[0] > 0.0) || !(pn > 0.0) || !(sp <= 1.7976931348623157e308)) bad = 1;
        smax = fmax(smax, sp);
    }
};

struct GasCarry {
    double rho, ir, vx, vy, vz, p;        // primitives of the current plane j (own cell)
    double amx, amy, amz, aE;             // U*(j) under construction
    double eps, adv;                      // GP_OD: rho*eps of plane j; 2 x (sum of V_hi - V_lo over the faces done so far)
    double wxm, wym, wx0, wy0;            // GP_TZREG: w*_x, w*_y of planes j-2 and j-1
};

struct GasShared {
    double *rp, *vx, *vy, *phi, *fy, *fyv, *ring, *tz;
};

// Prologue of one Eulerian cell column: primitives of plane z0-2, then plane z0-1 with the z face between them;
// publishes the primitives of plane z0-1.
__device__ __forceinline__ GasCarry gas_prologue(const FusedArgs<NFG>& a, const Geo& g, const Blk& b, const Foot& f, const GasShared& S,
                                                 double th, double gm1) {
    GasCarry c;
    const int t = f.t;
    int zm = map_safe(b.z0 - 2, g.nz, g.bcz);
    size_t off = f.base + (size_t)zm * f.nxny;
    constexpr int ES = OD ? BSTR : 1;        // the energy is paired with rho*eps under GP_OD
    double rho = a.U[0][BSTR * off], mx = a.U[1][BSTR * off], my = a.U[2][BSTR * off], mz = a.U[3][BSTR * off], E = a.U[4][ES * off];
    double ir = frcp(rho);
    const double vz_a = mz * ir;
    // same expression as the main loop, so that a 1-D problem stays bitwise 1-D across the chunk edge
    const double p_a = OD ? gm1 * a.U[IEPS][BSTR * off] : gm1 * (E - 0.5 * fma(mx, mx * ir, fma(my, my * ir, mz * vz_a)));
    const double rho_a = rho;
    zm = map_safe(b.z0 - 1, g.nz, g.bcz);
    off = f.base + (size_t)zm * f.nxny;
    rho = a.U[0][BSTR * off]; mx = a.U[1][BSTR * off]; my = a.U[2][BSTR * off]; mz = a.U[3][BSTR * off]; E = a.U[4][ES * off];
    ir = frcp(rho);
    c.rho = rho; c.ir = ir; c.vx = mx * ir; c.vy = my * ir; c.vz = mz * ir;
    c.eps = OD ? a.U[IEPS][BSTR * off] : 0.0;
    c.p = OD ? gm1 * c.eps : gm1 * (E - 0.5 * fma(mx, c.vx, fma(my, c.vy, mz * c.vz)));
    double Pz, PVz, Vz;
    gas_face(a.gamma, rho_a, vz_a, p_a, c.rho, c.vz, c.p, Pz, PVz, Vz);
    c.adv = -Vz;
    c.amx = mx; c.amy = my; c.amz = fma(0.5 * th, Pz, mz); c.aE = fma(0.25 * th, PVz, E);
    sts2(S.rp + 2 * t, c.rho, c.p); S.vx[t] = c.vx; S.vy[t] = c.vy;
    return c;
}

template <bool ST>
__device__ __forceinline__ void gas_iter(const FusedArgs<NFG>& a, BlockTab* T, const Blk& b, const Foot& f, const GasShared& S,
                                         GasCarry& c, int j, double tau, double th, double inv2h) {
    const Geo& g = a.g;
    const int t = f.t;
    const double gamma = a.gamma, gm1 = a.gamma - 1.0;
    const double th2 = 0.5 * th, th4 = 0.25 * th;
    const bool zout = g.bcz == GP_BC_OUTFLOW;
    const bool top_copy = !ST && zout && j == g.nz;
    const bool bot_dup = !ST && zout && j == 0;
    const bool do_out = ST || j - 1 >= b.z0;
    const int it = j - (b.z0 - 1);
    const double* ph0 = S.phi + pslot(it + 1) * PL;   // Phi(j); Phi(j-1) and Phi(j+1) sit in the slots either side
    if (it > 0 && f.ty < FY - 1) mbar_wait_at<OP_UP>(f.rowbar, (it - 1) & 1);   // primitives of plane j of the row above are published

    // B: x and y faces of plane j, each computed once (hi face per thread), in one basic block so
    // that the two solvers interleave
    double Pyh = 0.0, PVyh = 0.0, Vyh = 0.0, gy = 0.0;
    if (f.star_row) {
        const int tr = f.tx < FX - 1 ? t + 1 : t;
        const double2 ry = lds2(S.rp + 2 * (t + FX)), rx = lds2(S.rp + 2 * tr);
        const double vyr = S.vy[t + FX], vxr = S.vx[tr];
        const double phe = ph0[tr], phn = ph0[t + FX];
        const double phw = ph0[f.tx > 0 ? t - 1 : t], phs = ph0[t - FX];
        double Pxh, PVxh, Vxh;
        gas_face(gamma, c.rho, c.vy, c.p, ry.x, vyr, ry.y, Pyh, PVyh, Vyh);
        gas_face(gamma, c.rho, c.vx, c.p, rx.x, vxr, rx.y, Pxh, PVxh, Vxh);
        sts2(S.fy + 2 * t, Pyh, PVyh);
        if (OD) { S.fyv[t] = Vyh; c.adv += Vxh - __shfl_up_sync(0xffffffffu, Vxh, 1); }
        const double Pxl = __shfl_up_sync(0xffffffffu, Pxh, 1);
        const double PVxl = __shfl_up_sync(0xffffffffu, PVxh, 1);
        const double gx = (phe - phw) * inv2h;
        gy = (phn - phs) * inv2h;
        const double trg = tau * c.rho * gx;
        const double mx = c.rho * c.vx;
        c.amx = c.amx - th2 * (Pxh - Pxl) - trg;
        c.aE = c.aE - th4 * (PVxh - PVxl) - fma(-0.5 * tau, trg, tau * mx) * gx;
    } else if (f.ty == 0) {
        // the lowest halo row only supplies the y face between itself and row 1; the top halo row supplies nothing
        const double2 ry = lds2(S.rp + 2 * (t + FX));
        gas_face(gamma, c.rho, c.vy, c.p, ry.x, S.vy[t + FX], ry.y, Pyh, PVyh, Vyh);
        sts2(S.fy + 2 * t, Pyh, PVyh);
        if (OD) S.fyv[t] = Vyh;
    }
    row_arrive_at<OY_OWN>(f.rowbar);                                  // y fluxes of this row are written
    if (f.ty > 0) mbar_wait_at<OY_LO>(f.rowbar, it & 1);       // ... and those of the row below

    // C: y-flux difference
    if (f.star_row) {
        const double2 lo = lds2(S.fy + 2 * (t - FX));
        const double trg = tau * c.rho * gy;
        const double my = c.rho * c.vy;
        c.amy = c.amy - th2 * (Pyh - lo.x) - trg;
        c.aE = c.aE - th4 * (PVyh - lo.y) - fma(-0.5 * tau, trg, tau * my) * gy;
        if (OD) c.adv += Vyh - S.fyv[t - FX];
    }

    // E: plane j+1 has arrived in ring slot `it`; z face (j, j+1); U*(j) complete -> the same slot;
    // publish primitives(j+1)
    double* rs = S.ring + rslot(it) * GasTraits::SLOT;
    const unsigned slotbar = f.tabbar + 8 * rslot(it);
    mbar_wait_at<0>(slotbar, rpar(it));
    const double2 s0 = lds2(rs + 2 * t), s1 = lds2(rs + PP + 2 * t);
    double E_n, eps_n = 0.0;
    if (OD) { const double2 s2 = lds2(rs + 2 * PP + 2 * t); E_n = s2.x; eps_n = s2.y; }
    else E_n = rs[2 * PP + t];
    const double rho_n = s0.x, mx_n = s0.y, my_n = s1.x, mz_n = s1.y;
    const double ir_n = frcp(rho_n);
    const double vx_n = mx_n * ir_n, vy_n = my_n * ir_n, vz_n = mz_n * ir_n;
    // GP_OD: the pressure comes from the carried internal energy (4th equation)
    const double p_n = OD ? gm1 * eps_n : gm1 * (E_n - 0.5 * fma(mx_n, vx_n, fma(my_n, vy_n, mz_n * vz_n)));
    if (EARLYPUB) {
        sts2(S.rp + 2 * t, rho_n, p_n); S.vx[t] = vx_n; S.vy[t] = vy_n;
        row_arrive_at<OP_OWN>(f.rowbar);                              // primitives of plane j+1 of this row are published
    }
    double Pz = 0.0, PVz = 0.0, Vz = 0.0;
    if (f.star_row) {
        gas_face(gamma, c.rho, c.vz, c.p, rho_n, vz_n, p_n, Pz, PVz, Vz);
        double wx, wy, wz, Es, dens, epss = 0.0;
        if (top_copy) {                       // outflow: U*(nz) := U*(nz-1)
            const double* rq = S.ring + rslot(it + NS - 1) * GasTraits::SLOT;
            const double2 q0 = lds2(rq + 2 * t), q1 = lds2(rq + PP + 2 * t);
            dens = q0.x; wz = q0.y; wx = q1.x; wy = q1.y;
            if (OD) { const double2 q2 = lds2(rq + 2 * PP + 2 * t); Es = q2.x; epss = q2.y; }
            else Es = rq[2 * PP + t];
        } else {
            const double gz = (S.phi[pslot(it + 2) * PL + t] - S.phi[pslot(it) * PL + t]) * inv2h;
            const double trg = tau * c.rho * gz;
            const double mz = c.rho * c.vz;
            const double mzs = c.amz - th2 * Pz - trg;
            Es = c.aE - th4 * PVz - fma(-0.5 * tau, trg, tau * mz) * gz;
            dens = c.rho; wx = c.amx * c.ir; wy = c.amy * c.ir; wz = mzs * c.ir;
            // (rho eps)* = rho eps - tau (gamma-1) rho eps div V, V the face values of PAPER.md:112
            if (OD) epss = fma(-(th2 * gm1) * c.eps, c.adv + Vz, c.eps);
        }
        sts2(rs + 2 * t, dens, wz); sts2(rs + PP + 2 * t, wx, wy);
        if (OD) sts2(rs + 2 * PP + 2 * t, Es, epss); else rs[2 * PP + t] = Es;
        if (bot_dup) {                        // outflow: U*(-1) := U*(0)
            double* rg = S.ring + rslot(it + NS - 1) * GasTraits::SLOT;
            sts2(rg + 2 * t, dens, wz); sts2(rg + PP + 2 * t, wx, wy);
            if (OD) sts2(rg + 2 * PP + 2 * t, Es, epss); else rg[2 * PP + t] = Es;
        }
        if (do_out) {                         // 4 x z-average of w*_x, w*_y for plane j-1
            if (TZREG) {
                sts2(S.tz + (it % NTZ) * PP + 2 * t, sum3(c.wxm, c.wx0, wx), sum3(c.wym, c.wy0, wy));
            } else {
                const double2 wm = lds2(S.ring + rslot(it + NS - 2) * GasTraits::SLOT + PP + 2 * t);
                const double2 w0 = lds2(S.ring + rslot(it + NS - 1) * GasTraits::SLOT + PP + 2 * t);
                sts2(S.tz + (it % NTZ) * PP + 2 * t, sum3(wm.x, w0.x, wx), sum3(wm.y, w0.y, wy));
            }
        }
        if (TZREG) {
            c.wxm = bot_dup ? wx : c.wx0; c.wym = bot_dup ? wy : c.wy0;
            c.wx0 = wx; c.wy0 = wy;
        }
    }
    if (!EARLYPUB) { sts2(S.rp + 2 * t, rho_n, p_n); S.vx[t] = vx_n; S.vy[t] = vy_n; }
    c.amx = mx_n; c.amy = my_n; c.amz = fma(th2, Pz, mz_n); c.aE = fma(th4, PVz, E_n);
    c.rho = rho_n; c.ir = ir_n; c.vx = vx_n; c.vy = vy_n; c.vz = vz_n; c.p = p_n;
    if (OD) { c.eps = eps_n; c.adv = -Vz; }
    if (!EARLYPUB) row_arrive_at<OP_OWN>(f.rowbar);                   // primitives of plane j+1 of this row are published

    if (b.block_fix) {
        group_sync(&T->esync, 1);                  // phases: prologue 0, then two per plane
        if (f.fix) {
#pragma unroll
            for (int P = 0; P < GasTraits::NPAIR; ++P) {
                const double2 v = lds2(rs + P * PP + 2 * f.fix_src);
                sts2(rs + P * PP + 2 * t, v.x, v.y);
                if (bot_dup) sts2(S.ring + rslot(it + NS - 1) * GasTraits::SLOT + P * PP + 2 * t, v.x, v.y);
            }
            if (GasTraits::LAST1) {
                const double e = rs[2 * PP + f.fix_src];
                rs[2 * PP + t] = e;
                if (bot_dup) S.ring[rslot(it + NS - 1) * GasTraits::SLOT + 2 * PP + t] = e;
            }
            const double2 v = lds2(S.tz + (it % NTZ) * PP + 2 * f.fix_src);
            sts2(S.tz + (it % NTZ) * PP + 2 * t, v.x, v.y);
        }
        group_sync(&T->esync, 0);
    }
    __syncwarp();
    if (f.tx == 0) mbar_arrive_at<8 * NS>(slotbar);   // this row's U*(j) is complete
}

#if GP_EROWS == 2
// Two footprint rows per thread (rows 2w and 2w+1 of Eulerian warp w): the y face between them is solved once and
// stays in registers, the face above the upper row goes to the warp above through shared memory as before.
// Publishes the primitives of the next plane before the z face solves.
template <bool ST>
__device__ __forceinline__ void gas_iter2(const FusedArgs<NFG>& a, BlockTab* T, const Blk& b, const Foot (&f)[2], const GasShared& S,
                                          GasCarry (&c)[2], int j, double tau, double th, double inv2h) {
    const Geo& g = a.g;
    const int w = threadIdx.x >> 5;
    const int t0 = f[0].t, t1 = f[1].t, tx = f[0].tx;
    const double gamma = a.gamma, gm1 = a.gamma - 1.0;
    const double th2 = 0.5 * th, th4 = 0.25 * th;
    const bool zout = g.bcz == GP_BC_OUTFLOW;
    const bool top_copy = !ST && zout && j == g.nz;
    const bool bot_dup = !ST && zout && j == 0;
    const bool do_out = ST || j - 1 >= b.z0;
    const int it = j - (b.z0 - 1);
    const double* ph0 = S.phi + pslot(it + 1) * PL;
    const unsigned rowbar = f[0].rowbar;
    if (it > 0 && w < NEW - 1) mbar_wait_at<OP_UP>(rowbar, (it - 1) & 1);   // primitives of plane j of the warp above are published

    // B: the y face between the two rows, the y face above the upper row, the x faces of both rows
    const bool s0 = f[0].star_row, s1 = f[1].star_row;      // warp 0: row 0 is halo; last warp: row 1 is halo
    double Pym, PVym, Vym, Pyh = 0.0, PVyh = 0.0, Vyh = 0.0, gy0 = 0.0, gy1 = 0.0;
    gas_face(gamma, c[0].rho, c[0].vy, c[0].p, c[1].rho, c[1].vy, c[1].p, Pym, PVym, Vym);
    {
        const int e0 = tx < FX - 1 ? t0 + 1 : t0, e1 = e0 + FX, w0 = tx > 0 ? t0 - 1 : t0, w1 = w0 + FX;
        if (s1) {
            const double2 ry = lds2(S.rp + 2 * (t1 + FX)), rx = lds2(S.rp + 2 * e1);
            double Pxh, PVxh, Vxh;
            gas_face(gamma, c[1].rho, c[1].vy, c[1].p, ry.x, S.vy[t1 + FX], ry.y, Pyh, PVyh, Vyh);
            gas_face(gamma, c[1].rho, c[1].vx, c[1].p, rx.x, S.vx[e1], rx.y, Pxh, PVxh, Vxh);
            sts2(S.fy + 2 * t1, Pyh, PVyh);
            if (OD) { S.fyv[t1] = Vyh; c[1].adv += Vxh - __shfl_up_sync(0xffffffffu, Vxh, 1); }
            const double Pxl = __shfl_up_sync(0xffffffffu, Pxh, 1), PVxl = __shfl_up_sync(0xffffffffu, PVxh, 1);
            const double gx = (ph0[e1] - ph0[w1]) * inv2h;
            gy1 = (ph0[t1 + FX] - ph0[t0]) * inv2h;
            const double trg = tau * c[1].rho * gx, mx = c[1].rho * c[1].vx;
            c[1].amx = c[1].amx - th2 * (Pxh - Pxl) - trg;
            c[1].aE = c[1].aE - th4 * (PVxh - PVxl) - fma(-0.5 * tau, trg, tau * mx) * gx;
        }
        if (s0) {
            const double2 rx = lds2(S.rp + 2 * e0);
            double Pxh, PVxh, Vxh;
            gas_face(gamma, c[0].rho, c[0].vx, c[0].p, rx.x, S.vx[e0], rx.y, Pxh, PVxh, Vxh);
            if (OD) c[0].adv += Vxh - __shfl_up_sync(0xffffffffu, Vxh, 1);
            const double Pxl = __shfl_up_sync(0xffffffffu, Pxh, 1), PVxl = __shfl_up_sync(0xffffffffu, PVxh, 1);
            const double gx = (ph0[e0] - ph0[w0]) * inv2h;
            gy0 = (ph0[t1] - ph0[t0 - FX]) * inv2h;
            const double trg = tau * c[0].rho * gx, mx = c[0].rho * c[0].vx;
            c[0].amx = c[0].amx - th2 * (Pxh - Pxl) - trg;
            c[0].aE = c[0].aE - th4 * (PVxh - PVxl) - fma(-0.5 * tau, trg, tau * mx) * gx;
        }
    }
    row_arrive_at<OY_OWN>(rowbar);                                    // y fluxes above this warp's upper row are written
    if (w > 0) mbar_wait_at<OY_LO>(rowbar, it & 1);                 // ... and those above the warp below

    // C: y-flux differences
    if (s1) {
        const double trg = tau * c[1].rho * gy1, my = c[1].rho * c[1].vy;
        c[1].amy = c[1].amy - th2 * (Pyh - Pym) - trg;
        c[1].aE = c[1].aE - th4 * (PVyh - PVym) - fma(-0.5 * tau, trg, tau * my) * gy1;
        if (OD) c[1].adv += Vyh - Vym;
    }
    if (s0) {
        const double2 lo = lds2(S.fy + 2 * (t0 - FX));
        const double trg = tau * c[0].rho * gy0, my = c[0].rho * c[0].vy;
        c[0].amy = c[0].amy - th2 * (Pym - lo.x) - trg;
        c[0].aE = c[0].aE - th4 * (PVym - lo.y) - fma(-0.5 * tau, trg, tau * my) * gy0;
        if (OD) c[0].adv += Vym - S.fyv[t0 - FX];
    }

    // E: plane j+1 has arrived in ring slot `it`
    double* rs = S.ring + rslot(it) * GasTraits::SLOT;
    const unsigned slotbar = f[0].tabbar + 8 * rslot(it);
    mbar_wait_at<0>(slotbar, rpar(it));
    double rho_n[2], mx_n[2], my_n[2], mz_n[2], E_n[2], eps_n[2], ir_n[2], vx_n[2], vy_n[2], vz_n[2], p_n[2];
#pragma unroll
    for (int q = 0; q < 2; ++q) {
        const int t = f[q].t;
        const double2 a0 = lds2(rs + 2 * t), a1 = lds2(rs + PP + 2 * t);
        if (OD) { const double2 a2 = lds2(rs + 2 * PP + 2 * t); E_n[q] = a2.x; eps_n[q] = a2.y; }
        else { E_n[q] = rs[2 * PP + t]; eps_n[q] = 0.0; }
        rho_n[q] = a0.x; mx_n[q] = a0.y; my_n[q] = a1.x; mz_n[q] = a1.y;
        ir_n[q] = frcp(rho_n[q]);
        vx_n[q] = mx_n[q] * ir_n[q]; vy_n[q] = my_n[q] * ir_n[q]; vz_n[q] = mz_n[q] * ir_n[q];
        // GP_OD: the pressure comes from the carried internal energy (4th equation)
        p_n[q] = OD ? gm1 * eps_n[q] : gm1 * (E_n[q] - 0.5 * fma(mx_n[q], vx_n[q], fma(my_n[q], vy_n[q], mz_n[q] * vz_n[q])));
        sts2(S.rp + 2 * t, rho_n[q], p_n[q]); S.vx[t] = vx_n[q]; S.vy[t] = vy_n[q];
    }
    row_arrive_at<OP_OWN>(rowbar);                                    // primitives of plane j+1 of both rows are published
#pragma unroll
    for (int q = 0; q < 2; ++q) {
        const int t = f[q].t;
        GasCarry& cq = c[q];
        double Pz = 0.0, PVz = 0.0, Vz = 0.0;
        if (f[q].star_row) {
            gas_face(gamma, cq.rho, cq.vz, cq.p, rho_n[q], vz_n[q], p_n[q], Pz, PVz, Vz);
            double wx, wy, wz, Es, dens, epss = 0.0;
            if (top_copy) {                       // outflow: U*(nz) := U*(nz-1)
                const double* rq = S.ring + rslot(it + NS - 1) * GasTraits::SLOT;
                const double2 q0 = lds2(rq + 2 * t), q1 = lds2(rq + PP + 2 * t);
                dens = q0.x; wz = q0.y; wx = q1.x; wy = q1.y;
                if (OD) { const double2 q2 = lds2(rq + 2 * PP + 2 * t); Es = q2.x; epss = q2.y; }
                else Es = rq[2 * PP + t];
            } else {
                const double gz = (S.phi[pslot(it + 2) * PL + t] - S.phi[pslot(it) * PL + t]) * inv2h;
                const double trg = tau * cq.rho * gz;
                const double mz = cq.rho * cq.vz;
                const double mzs = cq.amz - th2 * Pz - trg;
                Es = cq.aE - th4 * PVz - fma(-0.5 * tau, trg, tau * mz) * gz;
                dens = cq.rho; wx = cq.amx * cq.ir; wy = cq.amy * cq.ir; wz = mzs * cq.ir;
                if (OD) epss = fma(-(th2 * gm1) * cq.eps, cq.adv + Vz, cq.eps);
            }
            sts2(rs + 2 * t, dens, wz); sts2(rs + PP + 2 * t, wx, wy);
            if (OD) sts2(rs + 2 * PP + 2 * t, Es, epss); else rs[2 * PP + t] = Es;
            if (bot_dup) {                        // outflow: U*(-1) := U*(0)
                double* rg = S.ring + rslot(it + NS - 1) * GasTraits::SLOT;
                sts2(rg + 2 * t, dens, wz); sts2(rg + PP + 2 * t, wx, wy);
                if (OD) sts2(rg + 2 * PP + 2 * t, Es, epss); else rg[2 * PP + t] = Es;
            }
            if (do_out) sts2(S.tz + (it % NTZ) * PP + 2 * t, sum3(cq.wxm, cq.wx0, wx), sum3(cq.wym, cq.wy0, wy));
            cq.wxm = bot_dup ? wx : cq.wx0; cq.wym = bot_dup ? wy : cq.wy0;
            cq.wx0 = wx; cq.wy0 = wy;
        }
        cq.amx = mx_n[q]; cq.amy = my_n[q]; cq.amz = fma(th2, Pz, mz_n[q]); cq.aE = fma(th4, PVz, E_n[q]);
        cq.rho = rho_n[q]; cq.ir = ir_n[q]; cq.vx = vx_n[q]; cq.vy = vy_n[q]; cq.vz = vz_n[q]; cq.p = p_n[q];
        if (OD) { cq.eps = eps_n[q]; cq.adv = -Vz; }
    }

    if (b.block_fix) {
        group_sync(&T->esync, 1);                  // phases: prologue 0, then two per plane
#pragma unroll
        for (int q = 0; q < 2; ++q)
            if (f[q].fix) {
                const int t = f[q].t, src = f[q].fix_src;
#pragma unroll
                for (int P = 0; P < GasTraits::NPAIR; ++P) {
                    const double2 v = lds2(rs + P * PP + 2 * src);
                    sts2(rs + P * PP + 2 * t, v.x, v.y);
                    if (bot_dup) sts2(S.ring + rslot(it + NS - 1) * GasTraits::SLOT + P * PP + 2 * t, v.x, v.y);
                }
                if (GasTraits::LAST1) {
                    const double e = rs[2 * PP + src];
                    rs[2 * PP + t] = e;
                    if (bot_dup) S.ring[rslot(it + NS - 1) * GasTraits::SLOT + 2 * PP + t] = e;
                }
                const double2 v = lds2(S.tz + (it % NTZ) * PP + 2 * src);
                sts2(S.tz + (it % NTZ) * PP + 2 * t, v.x, v.y);
            }
        group_sync(&T->esync, 0);
    }
    __syncwarp();
    if (tx == 0) mbar_arrive_at<8 * NS>(slotbar);   // this warp's U*(j) is complete
}
#endif  // GP_EROWS == 2

__global__ void __launch_bounds__(NT, 1)
k_fused_gas(const __grid_constant__ FusedArgs<NFG> a) {
    extern __shared__ __align__(128) unsigned char smraw[];
    BlockTab* T = reinterpret_cast<BlockTab*>(smraw);
    double* sm = reinterpret_cast<double*>(smraw + sizeof(BlockTab));
    GasShared S;
    S.rp = sm; S.vx = sm + 2 * PL; S.vy = sm + 3 * PL; S.phi = sm + 4 * PL; S.fy = S.phi + NPHI * PL;
    S.fyv = S.fy + 2 * PL;
    S.ring = S.fyv + (OD ? PL : 0); S.tz = S.ring + NS * GasTraits::SLOT;

    const Geo& g = a.g;
    const Blk b = make_blk(g, a.zchunk);
    if (threadIdx.x == 0) {
        build_tab(T, g, a.phi, b, a.use_tma);
        const unsigned cnt = T->percell ? NTD : 1;
        for (int s = 0; s < NS; ++s) { mbar_init(&T->landed[s], cnt); mbar_init(&T->ufull[s], NEW); }
        mbar_init(&T->pro, cnt);
        mbar_init(&T->dsync, NDW);
        mbar_init(&T->esync, NEW);
        for (int r = 0; r < FY; ++r) { mbar_init(&T->yrdy[r], 1); mbar_init(&T->prdy[r], 1); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const double tau = a.dt_ptr ? *a.dt_ptr : a.dt_val;
    const double th = tau / a.h, inv2h = 0.5 / a.h, gm1 = a.gamma - 1.0;

    double smax = 0.0, kap = 0.0;
    int bad = 0;
    if (threadIdx.x >= NTE) {
#if GP_REG_D
        reg_dealloc<GP_REG_D>();
#endif
        LagRows L;
        lag_warps<GasTraits>(a, T, b, S.ring, S.tz, S.phi, th, L);
        smax = L.smax; bad = L.bad; kap = L.kap;
    } else {
#if GP_REG_E
        reg_alloc<GP_REG_E>();
#endif
        if ((int)threadIdx.x < NEW * 32) {
#if GP_EROWS == 2
        const int w = threadIdx.x >> 5;
        const Foot f[2] = {make_foot(g, b, T, 2 * w), make_foot(g, b, T, 2 * w + 1)};
        GasCarry c[2] = {gas_prologue(a, g, b, f[0], S, th, gm1), gas_prologue(a, g, b, f[1], S, th, gm1)};
#else
        const Foot f = make_foot(g, b, T, threadIdx.x >> 5);
        GasCarry c = gas_prologue(a, g, b, f, S, th, gm1);
#endif
        mbar_wait(&T->pro, 0);
        group_sync(&T->esync, 0);

        int j = b.z0 - 1;
#if GP_EROWS == 2
        for (; j <= b.z0 && j <= b.z1; ++j) gas_iter2<false>(a, T, b, f, S, c, j, tau, th, inv2h);
        for (; j <= b.z1 - 1; ++j) gas_iter2<true>(a, T, b, f, S, c, j, tau, th, inv2h);
        for (; j <= b.z1; ++j) gas_iter2<false>(a, T, b, f, S, c, j, tau, th, inv2h);
#else
        for (; j <= b.z0 && j <= b.z1; ++j) gas_iter<false>(a, T, b, f, S, c, j, tau, th, inv2h);
        for (; j <= b.z1 - 1; ++j) gas_iter<true>(a, T, b, f, S, c, j, tau, th, inv2h);
        for (; j <= b.z1; ++j) gas_iter<false>(a, T, b, f, S, c, j, tau, th, inv2h);
#endif
        }   // real Eulerian warps (the padding warps of the register split skip to the reduction)
    }
    block_max_commit(smax, bad, a.smax_bits, a.flag, S.rp, kap, a.kappa);
}

#endif  // GP_FUSED_GAS

#ifdef GP_FUSED_BME
// =================================================================================================
// Collisionless component: fields n, nu (3), nE_ij (6: xx xy xz yy yz zz).
// Shared planes (of PL doubles): primitives (n,ux) (uy,uz) (Pxx,Pxz) (Pyy,Pyz) pairs 8 + Pxy 1,
// Phi ring 8, y-flux (Ps0,Ps1) (Ps2,EF0) (EF1,EF2) (EF3,EF4) pairs 8 + EF5 1, U* ring 4 x 5 pair planes = 40,
// z-averaged (w*_x,w*_y) pair 2 x 2 = 4  ->  70 planes (210 KB at FY = 12).
// =================================================================================================
// GP_OD: six more fields, Pi_ij, as three more pairs (Pi_xx,Pi_xy) (Pi_xz,Pi_yy) (Pi_yz,Pi_zz) in HBM and in the
// ring; the y-flux exchange carries 2u* as three more values: (EF5,us0) (us1,us2).
constexpr int NFB = NBME + (OD ? NODB : 0);
constexpr int PI0 = OD ? NBME : 0;        // first carried Pi_ij among the fields (only used under GP_OD; in range either way)
__device__ __forceinline__ constexpr int symi(int i, int j) {      // (i,j) -> index in xx xy xz yy yz zz
    return i == 0 ? j : (j == 0 ? i : (i == 1 ? (j == 1 ? 3 : 4) : (j == 1 ? 4 : 5)));
}
struct BmeTraits {
    static constexpr int NPAIR = OD ? 8 : 5, NP2 = NPAIR - 2;
    static constexpr bool LAST1 = false;
    static constexpr int SLOT = NPAIR * PP;
    static constexpr int NFY = OD ? 12 : 9;      // planes of the y-flux exchange
    static constexpr int PLANES = 9 + NPHI + NFY + NS * 2 * NPAIR + 2 * NTZ;
    __device__ static __forceinline__ double early(const FusedArgs<NFB>&, size_t, bool) { return 0.0; }
    __device__ static __forceinline__ void emit(const FusedArgs<NFB>& a, size_t off, double out[NFB], double, double& smax, int& bad,
                                                double& kap) {
        const double inn = frcp(out[0]);
        if (OD) {
            // correctness check of the state as the two stages left it, then the energy balance (G15)
            const double u[3] = {out[1] * inn, out[2] * inn, out[3] * inn};
            double Pc[6];                                 // Pi_ij as the total-energy tensor implies it
#pragma unroll
            for (int i = 0; i < 3; ++i)
#pragma unroll
                for (int j = i; j < 3; ++j) {
                    Pc[symi(i, j)] = fma(-out[1 + i], u[j], out[4 + symi(i, j)]);
                    kap += fabs(Pc[symi(i, j)] - out[PI0 + symi(i, j)]);
                }
            if (a.balance) {
                if (Pc[0] > 0.0 && Pc[3] > 0.0 && Pc[5] > 0.0) {
#pragma unroll
                    for (int q = 0; q < 6; ++q) out[PI0 + q] = Pc[q];
                } else {                                  // the carried tensor wins
#pragma unroll
                    for (int i = 0; i < 3; ++i)
#pragma unroll
                        for (int j = i; j < 3; ++j) out[4 + symi(i, j)] = fma(out[1 + i], u[j], out[PI0 + symi(i, j)]);
                }
            }
        }
#pragma unroll
        for (int P = 0; P < NPAIR; ++P)
            *reinterpret_cast<double2*>(a.Un[2 * P] + BSTR * off) = make_double2(out[2 * P], out[2 * P + 1]);
        // CFL of the new state (reading G4): |u_d| + sqrt(3 Pi_dd / n)
        const int dd[3] = {4, 7, 9};
        if (!(out[0] > 0.0)) bad = 1;
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            const double ud = out[1 + d] * inn;
            const double Pdd = OD ? out[PI0 + dd[d] - 4] : fma(-out[1 + d], ud, out[dd[d]]);   // GP_OD: carried (G16)
            const double c2 = 3.0 * Pdd * inn;
            const double sp = fabs(ud) + c2 * frsqrt(c2);
            if (!(Pdd > 0.0) || !(sp <= 1.7976931348623157e308)) bad = 1;
            smax = fmax(smax, sp);
        }
    }
};

struct BmeCarry {
    double n, in, u[3], Pi[6];            // primitives of the current plane j (own cell)
    double acc[9];                        // U*(j) under construction: nu (3), nE (6)
    double accP[6];                       // GP_OD: Pi*(j) under construction
    double wxm, wym, wx0, wy0;            // GP_TZREG: w*_x, w*_y of planes j-2 and j-1
};

// y-flux exchange of one cell: Py (3), EFy (6) and, under GP_OD, 2u* (3)
__device__ __forceinline__ void fy_store(double* fy, int t, const double Py[3], const double EFy[6], const double usy[3]) {
    sts2(fy + 2 * t, Py[0], Py[1]); sts2(fy + PP + 2 * t, Py[2], EFy[0]);
    sts2(fy + 2 * PP + 2 * t, EFy[1], EFy[2]); sts2(fy + 3 * PP + 2 * t, EFy[3], EFy[4]);
    if (OD) { sts2(fy + 4 * PP + 2 * t, EFy[5], usy[0]); sts2(fy + 5 * PP + 2 * t, usy[1], usy[2]); }
    else fy[4 * PP + t] = EFy[5];
}

// GP_OD, PAPER.md:65 without advection: Pi*_ab -= (tau/h) [Pi_bk du_a + Pi_ak du_b] for the faces normal to axis K,
// du2 = 2 x (u*_hi - u*_lo) of that axis, Pi the carried tensor of the cell at time n; sg = -1 for the hi - lo
// difference, +1 when only the lo face is entered (with du2 = 2 u*_lo)
template <int K>
__device__ __forceinline__ void pi_source(double accP[6], const double Pi[6], const double du2[3], double sth2) {
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = i; j < 3; ++j)
            accP[symi(i, j)] = fma(sth2, fma(Pi[symi(j, K)], du2[i], Pi[symi(i, K)] * du2[j]), accP[symi(i, j)]);
}

struct BmeShared {
    double *nu, *uu, *px, *py, *pxy, *phi, *fy, *ring, *tz;
};

// Prologue of one Eulerian cell column: primitives of plane z0-2, then plane z0-1 with the z face between them;
// publishes the primitives of plane z0-1.
__device__ __forceinline__ BmeCarry bme_prologue(const FusedArgs<NFB>& a, const Geo& g, const Blk& b, const Foot& f, const BmeShared& S,
                                                 double th) {
    BmeCarry c;
    const int t = f.t;
    int zm = map_safe(b.z0 - 2, g.nz, g.bcz);
    size_t off = f.base + (size_t)zm * f.nxny;
    double U0[NFB];
#pragma unroll
    for (int q = 0; q < NFB; ++q) U0[q] = a.U[q][BSTR * off];
    const double n_a = U0[0];
    double in = frcp(n_a);
    const double u_a[3] = {U0[1] * in, U0[2] * in, U0[3] * in};
    double Pz_a[3] = {fma(-U0[1], u_a[2], U0[6]), fma(-U0[2], u_a[2], U0[8]), fma(-U0[3], u_a[2], U0[9])};
    if (OD) { Pz_a[0] = U0[PI0 + 2]; Pz_a[1] = U0[PI0 + 4]; Pz_a[2] = U0[PI0 + 5]; }   // carried Pi_xz, Pi_yz, Pi_zz
    zm = map_safe(b.z0 - 1, g.nz, g.bcz);
    off = f.base + (size_t)zm * f.nxny;
#pragma unroll
    for (int q = 0; q < NFB; ++q) U0[q] = a.U[q][BSTR * off];
    c.n = U0[0]; c.in = frcp(c.n);
#pragma unroll
    for (int d = 0; d < 3; ++d) c.u[d] = U0[1 + d] * c.in;
    if (OD) {
#pragma unroll
        for (int q = 0; q < 6; ++q) c.Pi[q] = U0[PI0 + q];
    } else {
        c.Pi[0] = fma(-U0[1], c.u[0], U0[4]); c.Pi[1] = fma(-U0[1], c.u[1], U0[5]); c.Pi[2] = fma(-U0[1], c.u[2], U0[6]);
        c.Pi[3] = fma(-U0[2], c.u[1], U0[7]); c.Pi[4] = fma(-U0[2], c.u[2], U0[8]); c.Pi[5] = fma(-U0[3], c.u[2], U0[9]);
    }
    const double Pr[3] = {c.Pi[2], c.Pi[4], c.Pi[5]};
    double Pz[3], EFz[6], usz[3];
    bme_face<2>(n_a, u_a, Pz_a, c.n, c.u, Pr, Pz, EFz, usz);
    if (OD) {
#pragma unroll
        for (int q = 0; q < 6; ++q) c.accP[q] = c.Pi[q];
        pi_source<2>(c.accP, c.Pi, usz, 0.5 * th);
    }
#pragma unroll
    for (int d = 0; d < 3; ++d) c.acc[d] = fma(0.5 * th, Pz[d], U0[1 + d]);
#pragma unroll
    for (int q = 0; q < 6; ++q) c.acc[3 + q] = fma(0.25 * th, EFz[q], U0[4 + q]);
    sts2(S.nu + 2 * t, c.n, c.u[0]); sts2(S.uu + 2 * t, c.u[1], c.u[2]); sts2(S.px + 2 * t, c.Pi[0], c.Pi[2]);
    sts2(S.py + 2 * t, c.Pi[3], c.Pi[4]); S.pxy[t] = c.Pi[1];
    return c;
}

template <bool ST>
__device__ __forceinline__ void bme_iter(const FusedArgs<NFB>& a, BlockTab* T, const Blk& b, const Foot& f, const BmeShared& S,
                                         BmeCarry& c, int j, double tau, double th, double inv2h) {
    const Geo& g = a.g;
    const int t = f.t;
    const double th2 = 0.5 * th, th4 = 0.25 * th;
    const bool zout = g.bcz == GP_BC_OUTFLOW;
    const bool top_copy = !ST && zout && j == g.nz;
    const bool bot_dup = !ST && zout && j == 0;
    const bool do_out = ST || j - 1 >= b.z0;
    const int it = j - (b.z0 - 1);
    const double* ph0 = S.phi + pslot(it + 1) * PL;   // Phi(j); Phi(j-1) and Phi(j+1) sit in the slots either side
    if (it > 0 && f.ty < FY - 1) mbar_wait_at<OP_UP>(f.rowbar, (it - 1) & 1);   // primitives of plane j of the row above are published

    // B: x and y faces of plane j (hi face per thread), both solvers in ONE basic block so that their
    // dependent chains interleave
    double Py[3] = {0.0, 0.0, 0.0}, EFy[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0}, usy[3] = {0.0, 0.0, 0.0};
    double gx = 0.0, gy = 0.0;
    if (f.star_row) {
        const int tn = t + FX, te = f.tx < FX - 1 ? t + 1 : t;
        const double2 y0 = lds2(S.nu + 2 * tn), y1 = lds2(S.uu + 2 * tn), y2 = lds2(S.py + 2 * tn);
        const double2 x0 = lds2(S.nu + 2 * te), x1 = lds2(S.uu + 2 * te), x2 = lds2(S.px + 2 * te);
        const double pxy_n = S.pxy[tn], pxy_e = S.pxy[te];
        const double ury[3] = {y0.y, y1.x, y1.y}, urx[3] = {x0.y, x1.x, x1.y};
        const double Ply[3] = {c.Pi[1], c.Pi[3], c.Pi[4]}, Plx[3] = {c.Pi[0], c.Pi[1], c.Pi[2]};
        const double Pry[3] = {pxy_n, y2.x, y2.y}, Prx[3] = {x2.x, pxy_e, x2.y};
        double Px[3], EFx[6], usx[3];
        bme_face<1>(c.n, c.u, Ply, y0.x, ury, Pry, Py, EFy, usy);
        bme_face<0>(c.n, c.u, Plx, x0.x, urx, Prx, Px, EFx, usx);
        fy_store(S.fy, t, Py, EFy, usy);
        if (OD) {
            double du2[3];
#pragma unroll
            for (int q = 0; q < 3; ++q) du2[q] = usx[q] - __shfl_up_sync(0xffffffffu, usx[q], 1);
            pi_source<0>(c.accP, c.Pi, du2, -th2);
        }
#pragma unroll
        for (int q = 0; q < 3; ++q) c.acc[q] -= th2 * (Px[q] - __shfl_up_sync(0xffffffffu, Px[q], 1));
#pragma unroll
        for (int q = 0; q < 6; ++q) c.acc[3 + q] -= th4 * (EFx[q] - __shfl_up_sync(0xffffffffu, EFx[q], 1));
        gx = (ph0[te] - ph0[f.tx > 0 ? t - 1 : t]) * inv2h;
        gy = (ph0[tn] - ph0[t - FX]) * inv2h;
    } else if (f.ty == 0) {
        // the lowest halo row only supplies the y face between itself and row 1; the top halo row supplies nothing
        const int tn = t + FX;
        const double2 y0 = lds2(S.nu + 2 * tn), y1 = lds2(S.uu + 2 * tn), y2 = lds2(S.py + 2 * tn);
        const double ury[3] = {y0.y, y1.x, y1.y};
        const double Ply[3] = {c.Pi[1], c.Pi[3], c.Pi[4]};
        const double Pry[3] = {S.pxy[tn], y2.x, y2.y};
        bme_face<1>(c.n, c.u, Ply, y0.x, ury, Pry, Py, EFy, usy);
        fy_store(S.fy, t, Py, EFy, usy);
    }
    row_arrive_at<OY_OWN>(f.rowbar);                                  // y fluxes of this row are written
    if (f.ty > 0) mbar_wait_at<OY_LO>(f.rowbar, it & 1);       // ... and those of the row below

    // C: y-flux difference, then everything of U*(j) but the upper z face
    if (f.star_row) {
        const double* fy = S.fy + 2 * (t - FX);
        const double2 l0 = lds2(fy), l1 = lds2(fy + PP), l2 = lds2(fy + 2 * PP), l3 = lds2(fy + 3 * PP);
        double l4;
        if (OD) {
            const double2 m4 = lds2(fy + 4 * PP), m5 = lds2(fy + 5 * PP);
            l4 = m4.x;
            const double du2[3] = {usy[0] - m4.y, usy[1] - m5.x, usy[2] - m5.y};
            pi_source<1>(c.accP, c.Pi, du2, -th2);
        } else {
            l4 = S.fy[4 * PP + t - FX];
        }
        c.acc[0] -= th2 * (Py[0] - l0.x); c.acc[1] -= th2 * (Py[1] - l0.y); c.acc[2] -= th2 * (Py[2] - l1.x);
        c.acc[3] -= th4 * (EFy[0] - l1.y); c.acc[4] -= th4 * (EFy[1] - l2.x); c.acc[5] -= th4 * (EFy[2] - l2.y);
        c.acc[6] -= th4 * (EFy[3] - l3.x); c.acc[7] -= th4 * (EFy[4] - l3.y); c.acc[8] -= th4 * (EFy[5] - l4);
        // gravity (reading G5): -tau n g_i and -tau n [(u_i - tau g_i/2) g_j + (u_j - tau g_j/2) g_i]
        const double gr[3] = {gx, gy, (S.phi[pslot(it + 2) * PL + t] - S.phi[pslot(it) * PL + t]) * inv2h};
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


    // E: plane j+1 has arrived in ring slot `it`; z face (j, j+1); U*(j) complete -> the same slot;
    // publish primitives(j+1)
    double* rs = S.ring + rslot(it) * BmeTraits::SLOT;
    const unsigned slotbar = f.tabbar + 8 * rslot(it);
    mbar_wait_at<0>(slotbar, rpar(it));
    double Un[NFB];
    {
        const double2 s0 = lds2(rs + 2 * t), s1 = lds2(rs + PP + 2 * t);
        Un[0] = s0.x; Un[1] = s0.y; Un[2] = s1.x; Un[3] = s1.y;
#pragma unroll
        for (int P = 2; P < BmeTraits::NPAIR; ++P) {
            const double2 sp = lds2(rs + P * PP + 2 * t);
            Un[2 * P] = sp.x; Un[2 * P + 1] = sp.y;
        }
    }
    const double n_n = Un[0];
    const double in_n = frcp(n_n);
    const double u_n[3] = {Un[1] * in_n, Un[2] * in_n, Un[3] * in_n};
    double Pi_n[6];
    if (OD) {        // the dispersion tensor as carried
#pragma unroll
        for (int q = 0; q < 6; ++q) Pi_n[q] = Un[PI0 + q];
    } else {
        Pi_n[0] = fma(-Un[1], u_n[0], Un[4]); Pi_n[1] = fma(-Un[1], u_n[1], Un[5]); Pi_n[2] = fma(-Un[1], u_n[2], Un[6]);
        Pi_n[3] = fma(-Un[2], u_n[1], Un[7]); Pi_n[4] = fma(-Un[2], u_n[2], Un[8]); Pi_n[5] = fma(-Un[3], u_n[2], Un[9]);
    }
    if (EARLYPUB) {
        sts2(S.nu + 2 * t, n_n, u_n[0]); sts2(S.uu + 2 * t, u_n[1], u_n[2]); sts2(S.px + 2 * t, Pi_n[0], Pi_n[2]);
        sts2(S.py + 2 * t, Pi_n[3], Pi_n[4]); S.pxy[t] = Pi_n[1];
        row_arrive_at<OP_OWN>(f.rowbar);                              // primitives of plane j+1 of this row are published
    }
    double Pz[3] = {0.0, 0.0, 0.0}, EFz[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0}, usz[3] = {0.0, 0.0, 0.0};
    if (f.star_row) {
        const double Pl[3] = {c.Pi[2], c.Pi[4], c.Pi[5]};
        const double Pr[3] = {Pi_n[2], Pi_n[4], Pi_n[5]};
        bme_face<2>(c.n, c.u, Pl, n_n, u_n, Pr, Pz, EFz, usz);
        double o[NFB];      // n, w (3), nE (6) [, Pi (6)]
        if (top_copy) {                       // outflow: U*(nz) := U*(nz-1)
            const double* rq = S.ring + rslot(it + NS - 1) * BmeTraits::SLOT;
            const double2 q0 = lds2(rq + 2 * t), q1 = lds2(rq + PP + 2 * t);
            o[0] = q0.x; o[3] = q0.y; o[1] = q1.x; o[2] = q1.y;
#pragma unroll
            for (int P = 2; P < BmeTraits::NPAIR; ++P) {
                const double2 qp = lds2(rq + P * PP + 2 * t);
                o[2 * P] = qp.x; o[2 * P + 1] = qp.y;
            }
        } else {
            o[0] = c.n;
#pragma unroll
            for (int d = 0; d < 3; ++d) o[1 + d] = fma(-th2, Pz[d], c.acc[d]) * c.in;
#pragma unroll
            for (int q = 0; q < 6; ++q) o[4 + q] = fma(-th4, EFz[q], c.acc[3 + q]);
            if (OD) {
                pi_source<2>(c.accP, c.Pi, usz, -th2);        // the upper z face completes Pi*(j)
#pragma unroll
                for (int q = 0; q < 6; ++q) o[PI0 + q] = c.accP[q];
            }
        }
        sts2(rs + 2 * t, o[0], o[3]); sts2(rs + PP + 2 * t, o[1], o[2]);
#pragma unroll
        for (int P = 2; P < BmeTraits::NPAIR; ++P) sts2(rs + P * PP + 2 * t, o[2 * P], o[2 * P + 1]);
        if (bot_dup) {                        // outflow: U*(-1) := U*(0)
            double* rg = S.ring + rslot(it + NS - 1) * BmeTraits::SLOT;
            sts2(rg + 2 * t, o[0], o[3]); sts2(rg + PP + 2 * t, o[1], o[2]);
#pragma unroll
            for (int P = 2; P < BmeTraits::NPAIR; ++P) sts2(rg + P * PP + 2 * t, o[2 * P], o[2 * P + 1]);
        }
        if (do_out) {                         // 4 x z-average of w*_x, w*_y for plane j-1
            if (TZREG) {
                sts2(S.tz + (it % NTZ) * PP + 2 * t, sum3(c.wxm, c.wx0, o[1]), sum3(c.wym, c.wy0, o[2]));
            } else {
                const double2 wm = lds2(S.ring + rslot(it + NS - 2) * BmeTraits::SLOT + PP + 2 * t);
                const double2 w0 = lds2(S.ring + rslot(it + NS - 1) * BmeTraits::SLOT + PP + 2 * t);
                sts2(S.tz + (it % NTZ) * PP + 2 * t, sum3(wm.x, w0.x, o[1]), sum3(wm.y, w0.y, o[2]));
            }
        }
        if (TZREG) {
            c.wxm = bot_dup ? o[1] : c.wx0; c.wym = bot_dup ? o[2] : c.wy0;
            c.wx0 = o[1]; c.wy0 = o[2];
        }
    }
    if (!EARLYPUB) {
        sts2(S.nu + 2 * t, n_n, u_n[0]); sts2(S.uu + 2 * t, u_n[1], u_n[2]); sts2(S.px + 2 * t, Pi_n[0], Pi_n[2]);
        sts2(S.py + 2 * t, Pi_n[3], Pi_n[4]); S.pxy[t] = Pi_n[1];
    }
#pragma unroll
    for (int d = 0; d < 3; ++d) c.acc[d] = fma(th2, Pz[d], Un[1 + d]);
#pragma unroll
    for (int q = 0; q < 6; ++q) c.acc[3 + q] = fma(th4, EFz[q], Un[4 + q]);
    c.n = n_n; c.in = in_n;
#pragma unroll
    for (int d = 0; d < 3; ++d) c.u[d] = u_n[d];
#pragma unroll
    for (int q = 0; q < 6; ++q) c.Pi[q] = Pi_n[q];
    if (OD) {        // Pi*(j+1) starts from the carried tensor and the lower z face
#pragma unroll
        for (int q = 0; q < 6; ++q) c.accP[q] = Pi_n[q];
        pi_source<2>(c.accP, Pi_n, usz, th2);
    }
    if (!EARLYPUB) row_arrive_at<OP_OWN>(f.rowbar);     // primitives of plane j+1 of this row are published

    if (b.block_fix) {
        group_sync(&T->esync, 1);                  // phases: prologue 0, then two per plane
        if (f.fix) {
#pragma unroll
            for (int P = 0; P < BmeTraits::NPAIR; ++P) {
                const double2 v = lds2(rs + P * PP + 2 * f.fix_src);
                sts2(rs + P * PP + 2 * t, v.x, v.y);
                if (bot_dup) sts2(S.ring + rslot(it + NS - 1) * BmeTraits::SLOT + P * PP + 2 * t, v.x, v.y);
            }
            const double2 v = lds2(S.tz + (it % NTZ) * PP + 2 * f.fix_src);
            sts2(S.tz + (it % NTZ) * PP + 2 * t, v.x, v.y);
        }
        group_sync(&T->esync, 0);
    }
    __syncwarp();
    if (f.tx == 0) mbar_arrive_at<8 * NS>(slotbar);   // this row's U*(j) is complete
}


__global__ void __launch_bounds__(NT, 1)
k_fused_bme(const __grid_constant__ FusedArgs<NFB> a) {
    extern __shared__ __align__(128) unsigned char smraw[];
    BlockTab* T = reinterpret_cast<BlockTab*>(smraw);
    double* sm = reinterpret_cast<double*>(smraw + sizeof(BlockTab));
    BmeShared S;
    S.nu = sm; S.uu = sm + 2 * PL; S.px = sm + 4 * PL; S.py = sm + 6 * PL; S.pxy = sm + 8 * PL; S.phi = sm + 9 * PL;
    S.fy = S.phi + NPHI * PL; S.ring = S.fy + BmeTraits::NFY * PL; S.tz = S.ring + NS * BmeTraits::SLOT;

    const Geo& g = a.g;
    const Blk b = make_blk(g, a.zchunk);
    if (threadIdx.x == 0) {
        build_tab(T, g, a.phi, b, a.use_tma);
        const unsigned cnt = T->percell ? NTD : 1;
        for (int s = 0; s < NS; ++s) { mbar_init(&T->landed[s], cnt); mbar_init(&T->ufull[s], NEW); }
        mbar_init(&T->pro, cnt);
        mbar_init(&T->dsync, NDW);
        mbar_init(&T->esync, NEW);
        for (int r = 0; r < FY; ++r) { mbar_init(&T->yrdy[r], 1); mbar_init(&T->prdy[r], 1); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const double tau = a.dt_ptr ? *a.dt_ptr : a.dt_val;
    const double th = tau / a.h, inv2h = 0.5 / a.h;

    double smax = 0.0, kap = 0.0;
    int bad = 0;
    if (threadIdx.x >= NTE) {
#if GP_REG_D
        reg_dealloc<GP_REG_D>();
#endif
        LagRows L;
        lag_warps<BmeTraits>(a, T, b, S.ring, S.tz, S.phi, th, L);
        smax = L.smax; bad = L.bad; kap = L.kap;
    } else {
#if GP_REG_E
        reg_alloc<GP_REG_E>();
#endif
        if ((int)threadIdx.x < NEW * 32) {
        const Foot f = make_foot(g, b, T, threadIdx.x >> 5);
        BmeCarry c = bme_prologue(a, g, b, f, S, th);
        mbar_wait(&T->pro, 0);
        group_sync(&T->esync, 0);

        int j = b.z0 - 1;
        for (; j <= b.z0 && j <= b.z1; ++j) bme_iter<false>(a, T, b, f, S, c, j, tau, th, inv2h);
        for (; j <= b.z1 - 1; ++j) bme_iter<true>(a, T, b, f, S, c, j, tau, th, inv2h);
        for (; j <= b.z1; ++j) bme_iter<false>(a, T, b, f, S, c, j, tau, th, inv2h);
        }   // real Eulerian warps (the padding warps of the register split skip to the reduction)
    }
    block_max_commit(smax, bad, a.smax_bits, a.flag, S.nu, kap, a.kappa);
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

// Tensor maps of one launch (host side; encoded at the first launch on each half of the double buffer, then taken
// from the context's TmCache): field pairs as rows of 2 nx doubles, the gas energy and
// the padded Phi as rows of doubles; boxes of one footprint plane.  Returns false if TMA cannot describe the grid
// (odd nx: rows not 16-byte aligned) or the driver entry point is missing; the kernel then stages cell by cell.
typedef CUresult (*EncodeTiled)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static bool encode_map(CUtensorMap* tm, const void* base, size_t row_doubles, size_t ny, size_t nz, unsigned box_doubles) {
    static EncodeTiled enc = nullptr;
    static std::once_flag looked;
    std::call_once(looked, [] {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess)
            enc = (EncodeTiled)fn;
    });
    if (!enc || (row_doubles & 1)) return false;
    const cuuint64_t dims[3] = {row_doubles, ny, nz};
    const cuuint64_t strides[2] = {row_doubles * sizeof(double), row_doubles * ny * sizeof(double)};
    const cuuint32_t box[3] = {box_doubles, (cuuint32_t)FY, 1}, estr[3] = {1, 1, 1};
    return enc(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, const_cast<void*>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
               CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <int NF, class K>
static int launch_fused_t(gp_ctx* c, int which, K kernel, const int* fields, int planes, int kid, double dt, const double* d_dt,
                          const double* src_in = nullptr, double* src_out = nullptr, int balance = 0, double* kappa = nullptr) {
    FusedArgs<NF> a;
    a.src_in = src_in; a.src_out = src_out;
    a.balance = balance; a.kappa = kappa;
    a.g = Geo{c->g.nx, c->g.ny, c->g.nz, c->bc.x, c->bc.y, c->bc.z};
    for (int f = 0; f < NF; ++f) { a.U[f] = c->U[fields[f]]; a.Un[f] = c->Us[fields[f]]; }
    a.phi = phipad_of(c);
    // tensor maps: encoded once per half of the double buffer and kept with the context (gp_internal.h, TmCache)
    constexpr int NTM = (NF + 1) / 2 + 1;
    static_assert(NTM <= TM_MAX, "TmCache holds every map of one launch");
    TmCache*& tc = c->tmc[which];
    if (!tc) { tc = new (std::nothrow) TmCache; if (tc) std::memset((void*)tc, 0, sizeof(*tc)); }
    int set = -1;
    if (tc)
        for (int q = 0; q < 2; ++q)
            if (tc->key_u[q] == (const void*)a.U[0] && tc->key_phi[q] == (const void*)a.phi.p) set = q;
    if (set < 0) {
        CUtensorMap* tm = tc ? tc->tm[tc->next] : a.tm;
        bool ok = true;
        for (int P = 0; P < NF / 2; ++P) ok = ok && encode_map(&tm[P], a.U[2 * P], 2 * (size_t)c->g.nx, c->g.ny, c->g.nz, 2 * FX);
        if (NF & 1) ok = ok && encode_map(&tm[NF / 2], a.U[NF - 1], c->g.nx, c->g.ny, c->g.nz, FX);
        ok = ok && encode_map(&tm[(NF + 1) / 2], a.phi.p, a.phi.pitch, a.phi.py, (size_t)c->g.nz + 4, FX);
        a.use_tma = ok ? 1 : 0;
        if (tc) {
            set = tc->next;
            tc->key_u[set] = a.U[0]; tc->key_phi[set] = a.phi.p; tc->ok[set] = a.use_tma;
            tc->next ^= 1;
        }
    }
    if (tc) {
        a.use_tma = tc->ok[set];
        std::memcpy((void*)a.tm, (const void*)tc->tm[set], NTM * sizeof(CUtensorMap));
    }
    a.h = c->g.h; a.gamma = c->gamma; a.dt_val = dt; a.dt_ptr = d_dt;
    a.smax_bits = c->d_smax_next; a.flag = c->d_flag_next;
    const int tx = (c->g.nx + TXO - 1) / TXO, ty = (c->g.ny + TYO - 1) / TYO;
    a.zchunk = pick_zchunk(c, tx * ty);
    const int tz = (c->g.nz + a.zchunk - 1) / a.zchunk;
    const size_t smem = (size_t)planes * PL * sizeof(double) + sizeof(BlockTab);
    // the opt-in is per device and cheap: set it on every launch (a context may live on any device)
    GP_CUDA(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    tic(c, kid);
    kernel<<<dim3(tx, ty, tz), dim3(NT, 1, 1), smem, c->stream>>>(a);
    toc(c);
    c->n_own++;
    GP_CUDA(cudaGetLastError());
    return GP_OK;
}

#ifdef GP_FUSED_GAS
static int launch_gas_impl(gp_ctx* c, double dt, const double* d_dt, const double* src_in, double* src_out, int balance) {
    const int fields[NGAS + NODG] = {0, 1, 2, 3, 4, F_EPS};
    return launch_fused_t<NFG>(c, 0, k_fused_gas, fields, GasTraits::PLANES, K_FUSED_GAS, dt, d_dt, src_in, src_out, balance,
                               OD ? c->d_kappa : nullptr);
}
#endif
#ifdef GP_FUSED_BME
static int launch_bme_impl(gp_ctx* c, double dt, const double* d_dt, int balance) {
    int fields[NBME + NODB];
    for (int f = 0; f < NBME; ++f) fields[f] = NGAS + f;
    for (int q = 0; q < NODB; ++q) fields[NBME + q] = F_PI + q;
    return launch_fused_t<NFB>(c, 1, k_fused_bme, fields, BmeTraits::PLANES, K_FUSED_BME, dt, d_dt, nullptr, nullptr, balance,
                               OD ? c->d_kappa + 1 : nullptr);
}
#endif

#if defined(GP_FUSED_GAS) && !GP_OVERDET
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

#if defined(GP_FUSED_GAS) && !GP_OVERDET
int launch_fused_gas(gp_ctx* c, double dt, const double* d_dt, const double* src_in, double* src_out) {
    return GP_FUSED_NS::launch_gas_impl(c, dt, d_dt, src_in, src_out, 0);
}
int math_selftest(int n, const double* x, double* rcp, double* rsq) { return GP_FUSED_NS::math_selftest_impl(n, x, rcp, rsq); }
#endif
#if defined(GP_FUSED_BME) && !GP_OVERDET
int launch_fused_bme(gp_ctx* c, double dt, const double* d_dt) { return GP_FUSED_NS::launch_bme_impl(c, dt, d_dt, 0); }
#endif
#if defined(GP_FUSED_GAS) && GP_OVERDET
int launch_fused_gas_od(gp_ctx* c, double dt, const double* d_dt, const double* src_in, double* src_out, int balance) {
    return GP_FUSED_NS::launch_gas_impl(c, dt, d_dt, src_in, src_out, balance);
}
#endif
#if defined(GP_FUSED_BME) && GP_OVERDET
int launch_fused_bme_od(gp_ctx* c, double dt, const double* d_dt, int balance) { return GP_FUSED_NS::launch_bme_impl(c, dt, d_dt, balance); }
#endif

}  // namespace gp
