// nb_force.cu — the pairwise evaluation: acceleration, jerk, snap and
// potential of eq. (1)-(2) and their time derivatives (R3), for
// the active particles against all N predicted j-records.  fp64 on the FP64 ALU pipe; tensor cores
// are not used (no dense contraction).  Kernel shapes, all writing per-slice partial sums that a
// reduction kernel adds in a fixed order (the "Bfactor" j-split of PAPER.md:59-65, made deterministic):
//   force_li_kernel<EPS0, W, ORDER>  lanes-over-i: a thread owns one active particle in registers; the CTA
//                    streams j-tiles into shared memory with 1-D TMA bulk copies (UBLKCP) signalled
//                    on mbarriers, double-buffered; every lane reads the same j-record (broadcast LDS).
//                    W = 1: i-tiles of 128 particles.  W = 4 (17..96 active): i-tiles of 32, the four warps
//                    take different parts of each j-tile.
//   force_lj_kernel<EPS0, ORDER>  lanes-over-j (<= 16 active): a warp owns one active particle (same in every
//                    lane); its 32 lanes read 32 different j-records straight from global memory (coalesced)
//                    and the sums are combined with a warp-shuffle butterfly.
// ORDER = 6 is the scheme of the north star (a, jerk, snap, pot); 4 (a, jerk, pot) and 8 (+ crackle) are the other
// Hermite orders the paper names (R21, R22).
// Work items (i-unit, j-slice) are handed out by an atomic queue, not by a static stride: warps of
// co-resident CTAs do NOT get equal shares of the FP64 pipe (measured: of three CTAs with equal work on
// one SM the first finished after 40 % of the time the last one needed), so a static partition ends in a
// long tail of under-occupied SMs.  Where an item's sums are stored depends only on the item, so the
// results stay bitwise reproducible.
#include "nb_internal.h"
#include "nb_plan.h"

namespace {

// ---------------------------------------------------------------------------------------------
// One pair, 6th order.  53 FP64-pipe instructions (32 DFMA + 11 DMUL + 10 DADD) + 1 MUFU.RSQ64H.  Used by the
// lanes-over-j kernel; the lanes-over-i kernel uses pair2 below.
// ---------------------------------------------------------------------------------------------
struct Sums { double ax, ay, az, jx, jy, jz, sx, sy, sz, p, cx, cy, cz; };   // cx..cz: crackle, 8th order only

struct IPart { double x, y, z, vx, vy, vz, ax, ay, az, jx, jy, jz; };        // jx..jz: predicted jerk, 8th order only

// fp64 reciprocal-square-root seed: MUFU.RSQ64H works on the high word only (about 20 good bits).
__device__ __forceinline__ double rsqrt_seed(double s)
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(s));
    return y;
}

// fma / mul with the operand order fixed in PTX.  A DFMA that reads three different register pairs occupies
// the FP64 pipe for 3 cycles instead of 2 unless one operand comes from the operand-reuse cache of its slot
// (measured); keeping the shared factor (q, c1, c2, c3, dx) in the same slot of consecutive
// instructions lets ptxas mark it .reuse.
__device__ __forceinline__ double F(double a, double b, double c)
{
    double d;
    asm("fma.rn.f64 %0, %1, %2, %3;" : "=d"(d) : "d"(a), "d"(b), "d"(c));
    return d;
}
__device__ __forceinline__ double M(double a, double b)
{
    double d;
    asm("mul.rn.f64 %0, %1, %2;" : "=d"(d) : "d"(a), "d"(b));
    return d;
}
// 2 c by incrementing the exponent field (integer pipe, not the FP64 pipe).  Exact for every normal c; for
// c = +-0 it returns +-2^-1022 instead of 0, which only ever multiplies a finite u and is added to da.
__device__ __forceinline__ double twice(double c)
{
    return __hiloint2double(__double2hiint(c) + 0x00100000, __double2loint(c));
}

// MASK = false: the caller knows that no lane meets its own record here (self is ignored).
template <bool EPS0, bool MASK = true>
__device__ __forceinline__ void pair(const IPart& pi, const double4 p0, const double4 p1, const double2 p2,
                                     const double eps2, const bool self, Sums& S)
{
    const double dx = p0.x - pi.x, dy = p0.y - pi.y, dz = p0.z - pi.z;
    const double dvx = p1.x - pi.vx, dvy = p1.y - pi.vy, dvz = p1.z - pi.vz;
    const double dax = p1.w - pi.ax, day = p2.x - pi.ay, daz = p2.y - pi.az;
    double s = F(dx, dx, F(dy, dy, F(dz, dz, eps2)));
    if (EPS0 && MASK) s = self ? 1.0 : s;                // eps = 0: keep the masked self pair finite
    // y = s^(-1/2): seed e0 ~ 2^-20, one cubic (Halley) step leaves 5/16 e0^3 < 2^-60
    const double y0 = rsqrt_seed(s);
    const double e = F(-s, M(y0, y0), 1.0);
    const double y = F(M(y0, e), F(e, 0.375, 0.5), y0);
    // rv = dx.dv and B = dv.dv + dx.da, interleaved so that dx_k is shared by consecutive FMAs
    double rv = M(dz, dvz);
    double B = M(dvz, dvz);
    B = F(dz, daz, B);
    B = F(dvy, dvy, B);
    rv = F(dy, dvy, rv);
    B = F(dy, day, B);
    B = F(dvx, dvx, B);
    rv = F(dx, dvx, rv);
    B = F(dx, dax, B);
    const double yy = M(y, y);                           // 1/s
    const double z = M(yy, -3.0);
    const double mr = M(y, p0.w);                        // m_j / sqrt(s)
    const double q = M(yy, mr);                          // m_j s^(-3/2)
    const double alpha = M(yy, rv);
    const double c1 = M(z, rv);                          // -3 alpha
    const double c3 = F(c1, alpha, M(z, B));             // -3 beta = -3 (B/s + alpha^2)
    const double c2 = twice(c1);                         // -6 alpha
    const double ux = F(c1, dx, dvx), uy = F(c1, dy, dvy), uz = F(c1, dz, dvz);      // dv - 3 alpha dx
    double wx = F(c3, dx, dax), wy = F(c3, dy, day), wz = F(c3, dz, daz);            // da - 3 beta dx ...
    wx = F(c2, ux, wx); wy = F(c2, uy, wy); wz = F(c2, uz, wz);                      // ... - 6 alpha u
    S.ax = F(q, dx, S.ax); S.ay = F(q, dy, S.ay); S.az = F(q, dz, S.az);
    S.jx = F(q, ux, S.jx); S.jy = F(q, uy, S.jy); S.jz = F(q, uz, S.jz);
    S.sx = F(q, wx, S.sx); S.sy = F(q, wy, S.sy); S.sz = F(q, wz, S.sz);
    S.p += (MASK && self) ? 0.0 : mr;                    // j != i (eq. 1); a, jerk, snap get exactly 0 from the self pair
}

// ---------------------------------------------------------------------------------------------
// Two pairs (one i against records J[0], J[1]) with the ORDER of the FP64 instructions fixed by `asm volatile`.
// Why: on sm_100a a DFMA that reads three different register pairs holds the FP64 pipe for 3 cycles, not 2.
// It takes 2 only if one source is a duplicate, an immediate or uniform register, or comes from the
// operand-reuse cache, i.e. the instruction issued just before it BY THE SAME WARP read that register in the
// same operand slot (measured with DFMA chains).  Left to itself ptxas interleaves the pairs and
// loses most of these reuses (28 of 64 DFMAs took 3 cycles).  Here every three-source DFMA sits in a run whose
// neighbours share a source in the same slot, dependent instructions inside a run are >= 5 issue slots apart
// (DFMA latency is 8 cycles = 4 slots), and what reads at most two registers (DADD, DMUL, the rsqrt refinement)
// alternates between the two pairs; a stall there costs nothing while another warp has work.
// 53 FP64 instructions per pair (32 DFMA + 11 DMUL + 10 DADD) + 1 MUFU.RSQ64H, as in pair().
// ---------------------------------------------------------------------------------------------
#define VSUB(d, a, b) asm volatile("sub.rn.f64 %0, %1, %2;" : "=d"(d) : "d"(a), "d"(b))
#define VADD(d, a, b) asm volatile("add.rn.f64 %0, %1, %2;" : "=d"(d) : "d"(a), "d"(b))
#define VMUL(d, a, b) asm volatile("mul.rn.f64 %0, %1, %2;" : "=d"(d) : "d"(a), "d"(b))
#define VFMA(d, a, b, c) asm volatile("fma.rn.f64 %0, %1, %2, %3;" : "=d"(d) : "d"(a), "d"(b), "d"(c))
#define VFNMA(d, a, b, c) /* d = c - a b */ \
    asm volatile("{\n\t.reg .f64 n;\n\tneg.f64 n, %1;\n\tfma.rn.f64 %0, n, %2, %3;\n\t}" : "=d"(d) : "d"(a), "d"(b), "d"(c))
#define VRSQ(d, a) asm volatile("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(d) : "d"(a))
#define BOTH for (int k = 0; k < 2; ++k)

struct JRec { double4 p0, p1; double2 p2; };

template <bool EPS0, bool MASK>
__device__ __forceinline__ void pair2(const IPart& pi, const JRec (&J)[2], const double eps2, const bool (&self)[2], Sums& S)
{
    // PIN(v): a branch that is never taken (v > 0) but that ptxas cannot see through.  The sums are live on its
    // taken side, so the run of DFMAs that updates them cannot be moved across it: each pair's run stays in one piece.
#define PIN(v) if (__double2hiint(v) < 0) return;
    double dx[2], dy[2], dz[2], dvx[2], dvy[2], dvz[2], dax[2], day[2], daz[2];
    double s[2], rv[2], rv2[2], B[2], y0[2], t[2], e[2], h[2], y[2], yy[2], mr[2], z[2], q[2], c1[2], c2[2], c3[2];
    // differences, with B = dv.dv (operands are duplicates: two-cycle DFMAs) threaded through them
#pragma unroll
    BOTH VSUB(dvz[k], J[k].p1.z, pi.vz);
#pragma unroll
    BOTH VSUB(dvy[k], J[k].p1.y, pi.vy);
#pragma unroll
    BOTH VSUB(dvx[k], J[k].p1.x, pi.vx);
#pragma unroll
    BOTH VMUL(B[k], dvz[k], dvz[k]);
#pragma unroll
    BOTH VSUB(dz[k], J[k].p0.z, pi.z);
#pragma unroll
    BOTH VSUB(daz[k], J[k].p2.y, pi.az);
#pragma unroll
    BOTH VFMA(B[k], dvy[k], dvy[k], B[k]);
#pragma unroll
    BOTH VSUB(dy[k], J[k].p0.y, pi.y);
#pragma unroll
    BOTH VSUB(day[k], J[k].p2.x, pi.ay);
#pragma unroll
    BOTH VFMA(B[k], dvx[k], dvx[k], B[k]);
#pragma unroll
    BOTH VSUB(dx[k], J[k].p0.x, pi.x);
#pragma unroll
    BOTH VSUB(dax[k], J[k].p1.w, pi.ax);
    // s = dx.dx + eps2, rv = dx.dv, B += dx.da: runs of three that share d_c in slot A
#pragma unroll
    BOTH { VFMA(s[k], dz[k], dz[k], eps2); VMUL(rv[k], dz[k], dvz[k]); VFMA(B[k], dz[k], daz[k], B[k]); }
#pragma unroll
    BOTH { VFMA(s[k], dy[k], dy[k], s[k]); VFMA(rv[k], dy[k], dvy[k], rv[k]); VFMA(B[k], dy[k], day[k], B[k]); }
#pragma unroll
    BOTH { VFMA(s[k], dx[k], dx[k], s[k]); VFMA(rv[k], dx[k], dvx[k], rv[k]); VFMA(B[k], dx[k], dax[k], B[k]); }
    if (EPS0 && MASK) {                                   // eps = 0: keep the masked self pair finite
#pragma unroll
        BOTH s[k] = self[k] ? 1.0 : s[k];
    }
    // y = s^(-1/2): MUFU.RSQ64H seed (e ~ 2^-20), then one cubic step y = y0 + y0 e (1/2 + 3/8 e), e = 1 - s y0^2,
    // which leaves 5/16 e^3 < 2^-60
#pragma unroll
    BOTH VRSQ(y0[k], s[k]);
#pragma unroll
    BOTH VMUL(rv2[k], rv[k], rv[k]);
#pragma unroll
    BOTH VMUL(t[k], y0[k], y0[k]);
#pragma unroll
    BOTH VFNMA(e[k], s[k], t[k], 1.0);
#pragma unroll
    BOTH VFMA(h[k], e[k], 0.375, 0.5);
#pragma unroll
    BOTH VMUL(t[k], e[k], h[k]);
#pragma unroll
    BOTH VFMA(y[k], y0[k], t[k], y0[k]);
    // scalars: yy = 1/s, mr = m_j/sqrt(s), q = m_j s^(-3/2), c1 = -3 alpha, c2 = -6 alpha, c3 = -3 beta
    //          with alpha = rv/s, beta = B/s + alpha^2 = (B + rv^2/s)/s
#pragma unroll
    BOTH VMUL(yy[k], y[k], y[k]);
#pragma unroll
    BOTH VMUL(mr[k], y[k], J[k].p0.w);
#pragma unroll
    BOTH VMUL(z[k], yy[k], -3.0);
#pragma unroll
    BOTH { VMUL(q[k], mr[k], yy[k]); VFMA(B[k], rv2[k], yy[k], B[k]); }     // yy stays in slot B
#pragma unroll
    BOTH VMUL(c1[k], z[k], rv[k]);
#pragma unroll
    BOTH VMUL(c3[k], z[k], B[k]);
#pragma unroll
    BOTH c2[k] = twice(c1[k]);
    PIN(s[0])
    {
        const double m0 = (MASK && self[0]) ? 0.0 : mr[0];   // j != i (eq. 1); a, jerk, snap get exactly 0 from the self pair
        VADD(S.p, S.p, m0);
    }
    // u = dv + c1 dx, w = da + c3 dx + c2 u, sums += q (dx, u, w): 18 three-source DFMAs per pair in one run;
    // each shares a source with its predecessor in the same slot (A: c1, c3, q, c2; B: d_c, u_c)
#pragma unroll
    BOTH {
        double ux, uy, uz, wx, wy, wz;
        VFMA(ux, c1[k], dx[k], dvx[k]);
        VFMA(uy, c1[k], dy[k], dvy[k]);
        VFMA(uz, c1[k], dz[k], dvz[k]);
        VFMA(wz, c3[k], dz[k], daz[k]);
        VFMA(wy, c3[k], dy[k], day[k]);
        VFMA(wx, c3[k], dx[k], dax[k]);
        VFMA(S.ax, q[k], dx[k], S.ax);
        VFMA(S.ay, q[k], dy[k], S.ay);
        VFMA(S.az, q[k], dz[k], S.az);
        VFMA(S.jx, q[k], ux, S.jx);
        VFMA(wx, c2[k], ux, wx);
        VFMA(wy, c2[k], uy, wy);
        VFMA(wz, c2[k], uz, wz);
        VFMA(S.jz, q[k], uz, S.jz);
        VFMA(S.jy, q[k], uy, S.jy);
        VFMA(S.sx, q[k], wx, S.sx);
        VFMA(S.sy, q[k], wy, S.sy);
        VFMA(S.sz, q[k], wz, S.sz);
        PIN(yy[k])
        if (k == 0) {
            const double m1 = (MASK && self[1]) ? 0.0 : mr[1];
            VADD(S.p, S.p, m1);
        }
    }
}

// ---------------------------------------------------------------------------------------------
// 4th-order variant (R21): acceleration, jerk and potential only.  32 FP64-pipe instructions per
// pair (17 DFMA + 8 DMUL + 7 DADD) + 1 MUFU.RSQ64H; the snap sums stay 0.
// ---------------------------------------------------------------------------------------------
template <bool EPS0, bool MASK = true>
__device__ __forceinline__ void pair_o4(const IPart& pi, const double4 p0, const double4 p1, const double eps2, const bool self, Sums& S)
{
    const double dx = p0.x - pi.x, dy = p0.y - pi.y, dz = p0.z - pi.z;
    const double dvx = p1.x - pi.vx, dvy = p1.y - pi.vy, dvz = p1.z - pi.vz;
    double s = F(dx, dx, F(dy, dy, F(dz, dz, eps2)));
    if (EPS0 && MASK) s = self ? 1.0 : s;
    const double y0 = rsqrt_seed(s);
    const double e = F(-s, M(y0, y0), 1.0);
    const double y = F(M(y0, e), F(e, 0.375, 0.5), y0);
    const double rv = F(dx, dvx, F(dy, dvy, M(dz, dvz)));
    const double yy = M(y, y);
    const double mr = M(y, p0.w);
    const double q = M(yy, mr);
    const double c1 = M(M(yy, -3.0), rv);                // -3 alpha
    const double ux = F(c1, dx, dvx), uy = F(c1, dy, dvy), uz = F(c1, dz, dvz);
    S.ax = F(q, dx, S.ax); S.ay = F(q, dy, S.ay); S.az = F(q, dz, S.az);
    S.jx = F(q, ux, S.jx); S.jy = F(q, uy, S.jy); S.jz = F(q, uz, S.jz);
    S.p += (MASK && self) ? 0.0 : mr;
}

// two j-records at a time, FP64 instruction order as in pair2 (the nine three-source DFMAs of a pair in one pinned run)
template <bool EPS0, bool MASK>
__device__ __forceinline__ void pair2_o4(const IPart& pi, const JRec (&J)[2], const double eps2, const bool (&self)[2], Sums& S)
{
    double dx[2], dy[2], dz[2], dvx[2], dvy[2], dvz[2];
    double s[2], rv[2], y0[2], t[2], e[2], h[2], y[2], yy[2], mr[2], z[2], q[2], c1[2];
#pragma unroll
    BOTH { VSUB(dz[k], J[k].p0.z, pi.z); VSUB(dvz[k], J[k].p1.z, pi.vz); }
#pragma unroll
    BOTH { VSUB(dy[k], J[k].p0.y, pi.y); VSUB(dvy[k], J[k].p1.y, pi.vy); }
#pragma unroll
    BOTH { VSUB(dx[k], J[k].p0.x, pi.x); VSUB(dvx[k], J[k].p1.x, pi.vx); }
#pragma unroll
    BOTH { VFMA(s[k], dz[k], dz[k], eps2); VMUL(rv[k], dz[k], dvz[k]); }
#pragma unroll
    BOTH { VFMA(s[k], dy[k], dy[k], s[k]); VFMA(rv[k], dy[k], dvy[k], rv[k]); }
#pragma unroll
    BOTH { VFMA(s[k], dx[k], dx[k], s[k]); VFMA(rv[k], dx[k], dvx[k], rv[k]); }
    if (EPS0 && MASK) {
#pragma unroll
        BOTH s[k] = self[k] ? 1.0 : s[k];
    }
#pragma unroll
    BOTH VRSQ(y0[k], s[k]);
#pragma unroll
    BOTH VMUL(t[k], y0[k], y0[k]);
#pragma unroll
    BOTH VFNMA(e[k], s[k], t[k], 1.0);
#pragma unroll
    BOTH VFMA(h[k], e[k], 0.375, 0.5);
#pragma unroll
    BOTH VMUL(t[k], e[k], h[k]);
#pragma unroll
    BOTH VFMA(y[k], y0[k], t[k], y0[k]);
#pragma unroll
    BOTH VMUL(yy[k], y[k], y[k]);
#pragma unroll
    BOTH VMUL(mr[k], y[k], J[k].p0.w);
#pragma unroll
    BOTH VMUL(z[k], yy[k], -3.0);
#pragma unroll
    BOTH VMUL(q[k], mr[k], yy[k]);
#pragma unroll
    BOTH VMUL(c1[k], z[k], rv[k]);
    {
        const double m0 = (MASK && self[0]) ? 0.0 : mr[0];
        VADD(S.p, S.p, m0);
    }
    PIN(s[0])
#pragma unroll
    BOTH {
        double ux, uy, uz;
        VFMA(ux, c1[k], dx[k], dvx[k]);
        VFMA(uy, c1[k], dy[k], dvy[k]);
        VFMA(uz, c1[k], dz[k], dvz[k]);
        VFMA(S.az, q[k], dz[k], S.az);
        VFMA(S.ay, q[k], dy[k], S.ay);
        VFMA(S.ax, q[k], dx[k], S.ax);
        VFMA(S.jx, q[k], ux, S.jx);
        VFMA(S.jy, q[k], uy, S.jy);
        VFMA(S.jz, q[k], uz, S.jz);
        PIN(yy[k])
        if (k == 0) {
            const double m1 = (MASK && self[1]) ? 0.0 : mr[1];
            VADD(S.p, S.p, m1);
        }
    }
}

// ---------------------------------------------------------------------------------------------
// 8th-order variant (R22): crackle added.  With T3 = 3 dv.da + dx.dj and
// gamma = T3/s + alpha (3 beta - 4 alpha^2):  crackle term = q (dj - 9 alpha w - 9 beta u - 3 gamma dx).
// 84 FP64-pipe instructions per pair + 1 MUFU.RSQ64H; one pair at a time (ptxas schedules it; 2 x 12 differences would
// not fit the register budget).
// ---------------------------------------------------------------------------------------------
template <bool EPS0, bool MASK = true>
__device__ __forceinline__ void pair_o8(const IPart& pi, const double4 p0, const double4 p1, const double2 p2, const double4 p3,
                                        const double eps2, const bool self, Sums& S)
{
    const double dx = p0.x - pi.x, dy = p0.y - pi.y, dz = p0.z - pi.z;
    const double dvx = p1.x - pi.vx, dvy = p1.y - pi.vy, dvz = p1.z - pi.vz;
    const double dax = p1.w - pi.ax, day = p2.x - pi.ay, daz = p2.y - pi.az;
    const double djx = p3.x - pi.jx, djy = p3.y - pi.jy, djz = p3.z - pi.jz;
    double s = F(dx, dx, F(dy, dy, F(dz, dz, eps2)));
    if (EPS0 && MASK) s = self ? 1.0 : s;
    const double y0 = rsqrt_seed(s);
    const double e = F(-s, M(y0, y0), 1.0);
    const double y = F(M(y0, e), F(e, 0.375, 0.5), y0);
    const double rv = F(dx, dvx, F(dy, dvy, M(dz, dvz)));
    double B = M(dvz, dvz);
    B = F(dz, daz, B); B = F(dvy, dvy, B); B = F(dy, day, B); B = F(dvx, dvx, B); B = F(dx, dax, B);
    const double va = F(dvx, dax, F(dvy, day, M(dvz, daz)));
    const double xj = F(dx, djx, F(dy, djy, M(dz, djz)));
    const double T3 = F(va, 3.0, xj);
    const double yy = M(y, y);
    const double z = M(yy, -3.0);
    const double mr = M(y, p0.w);
    const double q = M(yy, mr);
    const double alpha = M(yy, rv);
    const double c1 = M(z, rv);                          // -3 alpha
    const double c3 = F(c1, alpha, M(z, B));             // -3 beta
    const double c2 = twice(c1);                         // -6 alpha
    const double g3 = F(alpha, F(c3, 3.0, M(M(alpha, alpha), 12.0)), M(z, T3));   // -3 gamma = z T3 + alpha (-9 beta + 12 alpha^2)
    const double c9a = M(c1, 3.0), c9b = M(c3, 3.0);     // -9 alpha, -9 beta
    const double ux = F(c1, dx, dvx), uy = F(c1, dy, dvy), uz = F(c1, dz, dvz);
    double wx = F(c3, dx, dax), wy = F(c3, dy, day), wz = F(c3, dz, daz);
    wx = F(c2, ux, wx); wy = F(c2, uy, wy); wz = F(c2, uz, wz);
    double kx = F(g3, dx, djx), ky = F(g3, dy, djy), kz = F(g3, dz, djz);
    kx = F(c9b, ux, kx); ky = F(c9b, uy, ky); kz = F(c9b, uz, kz);
    kx = F(c9a, wx, kx); ky = F(c9a, wy, ky); kz = F(c9a, wz, kz);
    S.ax = F(q, dx, S.ax); S.ay = F(q, dy, S.ay); S.az = F(q, dz, S.az);
    S.jx = F(q, ux, S.jx); S.jy = F(q, uy, S.jy); S.jz = F(q, uz, S.jz);
    S.sx = F(q, wx, S.sx); S.sy = F(q, wy, S.sy); S.sz = F(q, wz, S.sz);
    S.cx = F(q, kx, S.cx); S.cy = F(q, ky, S.cy); S.cz = F(q, kz, S.cz);
    S.p += (MASK && self) ? 0.0 : mr;
}

template <int ORDER>
__device__ __forceinline__ IPart load_ipart(const ForceArgs& A, int i)
{
    const double4 a = A.pj0[i], b = A.pj1[i];
    const double2 c = A.pj2[i];
    IPart p{a.x, a.y, a.z, b.x, b.y, b.z, b.w, c.x, c.y, 0.0, 0.0, 0.0};
    if (ORDER == 8) { const double4 d = A.pj3[i]; p.jx = d.x; p.jy = d.y; p.jz = d.z; }
    return p;
}

// partial planes are [plane][NC][ld] with NC = 10 (a, jerk, snap, pot), 13 at the 8th order (+ crackle)
template <int ORDER>
__device__ __forceinline__ void store_sums(const ForceArgs& A, int slice, int k, bool valid, const Sums& S)
{
    constexpr int NC = ORDER == 8 ? 13 : 10;
    if (A.n_planes > 1) {
        double* P = A.partial + (size_t)slice * NC * A.ld + k;      // plane (slice, c) is contiguous in k
        const size_t ld = A.ld;
        P[0] = S.ax; P[ld] = S.ay; P[2 * ld] = S.az;
        P[3 * ld] = S.jx; P[4 * ld] = S.jy; P[5 * ld] = S.jz;
        P[6 * ld] = S.sx; P[7 * ld] = S.sy; P[8 * ld] = S.sz; P[9 * ld] = S.p;
        if (ORDER == 8) { P[10 * ld] = S.cx; P[11 * ld] = S.cy; P[12 * ld] = S.cz; }
    } else if (valid) {
        A.out_a[3 * k] = S.ax; A.out_a[3 * k + 1] = S.ay; A.out_a[3 * k + 2] = S.az;
        A.out_j[3 * k] = S.jx; A.out_j[3 * k + 1] = S.jy; A.out_j[3 * k + 2] = S.jz;
        A.out_s[3 * k] = S.sx; A.out_s[3 * k + 1] = S.sy; A.out_s[3 * k + 2] = S.sz;
        A.out_p[k] = -S.p;
        if (ORDER == 8) { A.out_c[3 * k] = S.cx; A.out_c[3 * k + 1] = S.cy; A.out_c[3 * k + 2] = S.cz; }
    }
}

// ---------------------------------------------------------------------------------------------
// mbarrier / TMA bulk-copy helpers (PTX; SASS: SYNCS.*, UBLKCP)
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    uint32_t done;
    do {
        asm volatile("{\n\t.reg .pred p;\n\t"
                     "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
                     "selp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(done) : "r"(bar), "r"(parity) : "memory");
    } while (!done);
}

// Device-planned launch (nb_run_blocks): take the plan the scheduler left in device memory.  False: this kernel shape
// is not the one the plan names (or the step is not taken) and the whole grid returns.
__device__ __forceinline__ bool take_devplan(ForceArgs& A, int kernel_id)
{
    if (!A.dp) return true;
    const DevPlan* d = A.dp;
    if (d->stop || d->kernel != kernel_id) return false;
    A.n_act = d->n_act; A.n_units = d->n_units; A.n_split = d->n_split; A.slice_tiles = d->slice_tiles;
    A.n_items = d->n_items; A.ld = d->ld; A.n_planes = d->n_planes;
    return true;
}

// The CTA (or warp) that finds the queue empty last puts both counters back to 0 for the next launch.
__device__ __forceinline__ void queue_retire(int* queue, int n_workers)
{
    __threadfence();
    if (atomicAdd(queue + 1, 1) == n_workers - 1) { queue[0] = 0; queue[1] = 0; }
}

// ---------------------------------------------------------------------------------------------
// lanes-over-i
// ---------------------------------------------------------------------------------------------
static_assert((LI_STAGES & (LI_STAGES - 1)) == 0, "LI_STAGES must be a power of two");
static_assert(LI_TJ % 2 == 0, "pair2 takes two j-records at a time");

// W = 1: a work item is (i-tile of LI_THREADS particles, j-slice).  W = 4 (17..96 active particles): the CTA's four
// warps hold the SAME 32 particles and each takes its own quarter of every j-tile, so an item is (32 particles,
// j-slice) and writes four partial planes (slice * 4 + warp) that the reduction adds like any other slices.
template <bool EPS0, int W, int ORDER>
__global__ void __launch_bounds__(LI_THREADS, LI_CTAS_PER_SM) force_li_kernel(const ForceArgs A_)
{
    ForceArgs A = A_;
    if (!take_devplan(A, W == 1 ? 0 : 2)) return;
    constexpr int UNIT = LI_UNIT / W;                      // active particles per work item
    constexpr int TJW = LI_TJ / W;                         // records of each j-tile one warp group takes
    static_assert(W == 1 || (LI_I == 1 && UNIT == 32 && TJW % 2 == 0), "W > 1: one warp per group");
    __shared__ alignas(128) double4 s0[LI_STAGES][LI_TJ];
    __shared__ alignas(128) double4 s1[LI_STAGES][LI_TJ];
    __shared__ alignas(128) double2 s2[LI_STAGES][LI_TJ];
    __shared__ alignas(128) double4 s3[LI_STAGES][ORDER == 8 ? LI_TJ : 1];   // predicted jerk, 8th order only
    __shared__ alignas(8) unsigned long long full[LI_STAGES];
    __shared__ int next_item;

    const int tid = threadIdx.x;
    const int wg = W == 1 ? 0 : tid / UNIT;                // warp group: which part of each j-tile
    const int til = W == 1 ? tid : tid % UNIT;             // lane within the i-tile
    if (tid == 0) {
        for (int s = 0; s < LI_STAGES; ++s) mbar_init(smem_u32(&full[s]), 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    // one elected thread stages j-tile `tile` into stage `st`: three bulk copies, one barrier
    auto stage_tile = [&](int tile, int st) {
        const uint32_t bar = smem_u32(&full[st]);
        const size_t j0 = (size_t)tile * LI_TJ;
        mbar_expect_tx(bar, LI_TJ * (ORDER == 8 ? 112 : 80));
        bulk_g2s(smem_u32(&s0[st][0]), A.pj0 + j0, LI_TJ * 32, bar);
        bulk_g2s(smem_u32(&s1[st][0]), A.pj1 + j0, LI_TJ * 32, bar);
        bulk_g2s(smem_u32(&s2[st][0]), A.pj2 + j0, LI_TJ * 16, bar);
        if (ORDER == 8) bulk_g2s(smem_u32(&s3[st][0]), A.pj3 + j0, LI_TJ * 32, bar);
    };

    uint32_t uses = 0;   // j-tiles this CTA has consumed so far: stage = uses % STAGES, parity = (uses / STAGES) & 1
    for (;;) {
        if (tid == 0) next_item = atomicAdd(A.queue, 1);
        __syncthreads();
        const int item = next_item;
        __syncthreads();                                   // everyone has read next_item before it is overwritten
        if (item >= A.n_items) break;
        const int unit = item % A.n_units, slice = item / A.n_units;
        const int t0 = slice * A.slice_tiles;
        const int nt = min(A.slice_tiles, A.n_tiles - t0);

        if (tid == 0)
            for (int f = 0; f < LI_STAGES && f < nt; ++f) stage_tile(t0 + f, (uses + f) & (LI_STAGES - 1));

        int ii[LI_I];
        bool valid[LI_I];
        IPart pi[LI_I];
        Sums acc[LI_I];
#pragma unroll
        for (int q = 0; q < LI_I; ++q) {
            const int k = unit * UNIT + q * LI_THREADS + til;
            valid[q] = k < A.n_act;
            const int kk = valid[q] ? k : 0;
            ii[q] = A.idx ? A.idx[kk] : kk;
            pi[q] = load_ipart<ORDER>(A, ii[q]);
            acc[q] = Sums{0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
        }

        for (int t = 0; t < nt; ++t) {
            const uint32_t u = uses + t;
            const int st = u & (LI_STAGES - 1);
            mbar_wait(smem_u32(&full[st]), (u / LI_STAGES) & 1);
            const int jbase = (t0 + t) * LI_TJ + wg * TJW;
            // the self pair (reading R4) lies in one j-tile per particle: only a warp that has one of its own
            // particles in this tile runs the loop that masks by index
            bool own = false;
#pragma unroll
            for (int q = 0; q < LI_I; ++q) own |= (unsigned)(ii[q] - jbase) < (unsigned)TJW;
            const double4 *t0p = &s0[st][wg * TJW], *t1p = &s1[st][wg * TJW];
            const double2* t2p = &s2[st][wg * TJW];
            if (ORDER == 8) {
                const double4* t3p = &s3[st][ORDER == 8 ? wg * TJW : 0];
                if (__any_sync(0xffffffffu, own)) {
#pragma unroll 2
                    for (int jj = 0; jj < TJW; ++jj) {
#pragma unroll
                        for (int q = 0; q < LI_I; ++q)
                            pair_o8<EPS0, true>(pi[q], t0p[jj], t1p[jj], t2p[jj], t3p[jj], A.eps2, jbase + jj == ii[q], acc[q]);
                    }
                } else {
#pragma unroll 2
                    for (int jj = 0; jj < TJW; ++jj) {
#pragma unroll
                        for (int q = 0; q < LI_I; ++q) pair_o8<EPS0, false>(pi[q], t0p[jj], t1p[jj], t2p[jj], t3p[jj], A.eps2, false, acc[q]);
                    }
                }
            } else if (__any_sync(0xffffffffu, own)) {
#pragma unroll 1
                for (int jj = 0; jj < TJW; jj += 2) {
                    const JRec J[2] = {{t0p[jj], t1p[jj], t2p[jj]}, {t0p[jj + 1], t1p[jj + 1], t2p[jj + 1]}};
#pragma unroll
                    for (int q = 0; q < LI_I; ++q) {
                        const bool self[2] = {jbase + jj == ii[q], jbase + jj + 1 == ii[q]};
                        if (ORDER == 4) pair2_o4<EPS0, true>(pi[q], J, A.eps2, self, acc[q]);
                        else pair2<EPS0, true>(pi[q], J, A.eps2, self, acc[q]);
                    }
                }
            } else {
#pragma unroll 1
                for (int jj = 0; jj < TJW; jj += 2) {
                    const JRec J[2] = {{t0p[jj], t1p[jj], t2p[jj]}, {t0p[jj + 1], t1p[jj + 1], t2p[jj + 1]}};
                    const bool self[2] = {false, false};
#pragma unroll
                    for (int q = 0; q < LI_I; ++q) {
                        if (ORDER == 4) pair2_o4<EPS0, false>(pi[q], J, A.eps2, self, acc[q]);
                        else pair2<EPS0, false>(pi[q], J, A.eps2, self, acc[q]);
                    }
                }
            }
            __syncthreads();                                   // every warp is done with stage st
            if (tid == 0 && t + LI_STAGES < nt) stage_tile(t0 + t + LI_STAGES, st);
        }
        uses += nt;

#pragma unroll
        for (int q = 0; q < LI_I; ++q) store_sums<ORDER>(A, slice * W + wg, unit * UNIT + q * LI_THREADS + til, valid[q], acc[q]);
    }
    if (tid == 0) queue_retire(A.queue, gridDim.x);
}

// ---------------------------------------------------------------------------------------------
// lanes-over-j
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

template <bool EPS0, int ORDER>
__global__ void __launch_bounds__(LJ_THREADS, ORDER == 8 ? 1 : LJ_CTAS_PER_SM) force_lj_kernel(const ForceArgs A_)
{
    ForceArgs A = A_;
    if (!take_devplan(A, 1)) return;
    const int lane = threadIdx.x & 31;
    for (;;) {
        int wi = 0;
        if (lane == 0) wi = atomicAdd(A.queue, 1);
        wi = __shfl_sync(0xffffffffu, wi, 0);
        if (wi >= A.n_items) break;
        const int unit = wi % A.n_units, slice = wi / A.n_units;
        const int t0 = slice * A.slice_tiles;
        const int nt = min(A.slice_tiles, A.n_tiles - t0);

        int ii[LJ_I];
        bool valid[LJ_I];
        IPart pi[LJ_I];
        Sums acc[LJ_I];
#pragma unroll
        for (int q = 0; q < LJ_I; ++q) {
            const int k = unit * LJ_I + q;
            valid[q] = k < A.n_act;
            const int kk = valid[q] ? k : 0;
            ii[q] = A.idx ? A.idx[kk] : kk;
            pi[q] = load_ipart<ORDER>(A, ii[q]);
            acc[q] = Sums{0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
        }

        int j = t0 * LJ_TJ + lane;
        double4 n0 = A.pj0[j], n1 = A.pj1[j];
        double2 n2 = A.pj2[j];
        double4 n3 = ORDER == 8 ? A.pj3[j] : make_double4(0, 0, 0, 0);
        for (int t = 0; t < nt; ++t) {
            const double4 p0 = n0, p1 = n1, p3 = n3;
            const double2 p2 = n2;
            if (t + 1 < nt) {                                                                            // prefetch
                n0 = A.pj0[j + LJ_TJ]; n1 = A.pj1[j + LJ_TJ]; n2 = A.pj2[j + LJ_TJ];
                if (ORDER == 8) n3 = A.pj3[j + LJ_TJ];
            }
#pragma unroll
            for (int q = 0; q < LJ_I; ++q) {
                if (ORDER == 4) pair_o4<EPS0>(pi[q], p0, p1, A.eps2, j == ii[q], acc[q]);
                else if (ORDER == 8) pair_o8<EPS0>(pi[q], p0, p1, p2, p3, A.eps2, j == ii[q], acc[q]);
                else pair<EPS0>(pi[q], p0, p1, p2, A.eps2, j == ii[q], acc[q]);
            }
            j += LJ_TJ;
        }

#pragma unroll
        for (int q = 0; q < LJ_I; ++q) {
            Sums& S = acc[q];
            S.ax = warp_sum(S.ax); S.ay = warp_sum(S.ay); S.az = warp_sum(S.az);
            S.jx = warp_sum(S.jx); S.jy = warp_sum(S.jy); S.jz = warp_sum(S.jz);
            S.sx = warp_sum(S.sx); S.sy = warp_sum(S.sy); S.sz = warp_sum(S.sz);
            S.p = warp_sum(S.p);
            if (ORDER == 8) { S.cx = warp_sum(S.cx); S.cy = warp_sum(S.cy); S.cz = warp_sum(S.cz); }
            if (lane == 0) store_sums<ORDER>(A, slice, unit * LJ_I + q, valid[q], S);
        }
    }
    if (lane == 0) queue_retire(A.queue, gridDim.x * LJ_WARPS);
}

// ---------------------------------------------------------------------------------------------
// partial-sum reduction (row a3).  T threads per active particle (T a power of two chosen from S on the host):
// thread `lane` adds slices lane, lane + T, ... in increasing order, then the T lane sums are combined by a binary
// tree in shared memory.  The order depends only on (S, T): bitwise reproducible.  T = 1 is the plain loop over
// slices (large active sets, few slices: the loads of neighbouring threads coalesce over k).
// ---------------------------------------------------------------------------------------------
template <int NC>
__global__ void __launch_bounds__(RED_THREADS) reduce_partials_kernel(const ForceArgs A_, int T)
{
    __shared__ double sm[NC][RED_THREADS];
    ForceArgs A = A_;
    if (A.dp) {                                            // device-planned: any kernel shape, T from the plan
        if (A.dp->stop) return;
        A.n_act = A.dp->n_act; A.ld = A.dp->ld; A.n_planes = A.dp->n_planes; T = A.dp->red_T;
        if (A.n_planes <= 1) return;                       // the force kernel wrote the results itself
    }
    const int R = RED_THREADS / T;                         // active particles per block and pass
    const int kl = threadIdx.x % R, lane = threadIdx.x / R;
    for (int k0 = blockIdx.x * R; k0 < A.n_act; k0 += gridDim.x * R) {      // uniform over the block
        const int k = k0 + kl;
        double r[NC];
#pragma unroll
        for (int c = 0; c < NC; ++c) r[c] = 0.0;
        if (k < A.n_act) {
            const size_t plane = (size_t)NC * A.ld;
            const double* P = A.partial + (size_t)lane * plane + k;
            for (int s = lane; s < A.n_planes; s += T, P += (size_t)T * plane) {
#pragma unroll
                for (int c = 0; c < NC; ++c) r[c] += P[(size_t)c * A.ld];
            }
        }
        for (int off = T >> 1; off > 0; off >>= 1) {
            if (lane >= off && lane < 2 * off) {
#pragma unroll
                for (int c = 0; c < NC; ++c) sm[c][threadIdx.x] = r[c];
            }
            __syncthreads();
            if (lane < off) {
#pragma unroll
                for (int c = 0; c < NC; ++c) r[c] += sm[c][threadIdx.x + off * R];
            }
            __syncthreads();
        }
        if (lane != 0 || k >= A.n_act) continue;
        A.out_a[3 * k] = r[0]; A.out_a[3 * k + 1] = r[1]; A.out_a[3 * k + 2] = r[2];
        A.out_j[3 * k] = r[3]; A.out_j[3 * k + 1] = r[4]; A.out_j[3 * k + 2] = r[5];
        A.out_s[3 * k] = r[6]; A.out_s[3 * k + 1] = r[7]; A.out_s[3 * k + 2] = r[8];
        A.out_p[k] = -r[9];
        if (NC == 13) { A.out_c[3 * k] = r[10]; A.out_c[3 * k + 1] = r[11]; A.out_c[3 * k + 2] = r[12]; }
    }
}

}  // namespace

// kernel instantiation for (eps == 0, order)
#define NB_DISPATCH(CALL)                                               \
    do {                                                                \
        if (order == 4)      { if (eps_is_zero) { CALL(true, 4); } else { CALL(false, 4); } } \
        else if (order == 8) { if (eps_is_zero) { CALL(true, 8); } else { CALL(false, 8); } } \
        else                 { if (eps_is_zero) { CALL(true, 6); } else { CALL(false, 6); } } \
    } while (0)

cudaError_t nb_launch_force(const nb_plan& plan, const ForceArgs& args, bool eps_is_zero, int order, cudaStream_t st, int* launches)
{
#define LI1(E, O) force_li_kernel<E, 1, O><<<plan.grid, LI_THREADS, 0, st>>>(args)
#define LIW(E, O) force_li_kernel<E, LI_W, O><<<plan.grid, LI_THREADS, 0, st>>>(args)
#define LJ(E, O) force_lj_kernel<E, O><<<plan.grid, LJ_THREADS, 0, st>>>(args)
    if (plan.kernel == 0) NB_DISPATCH(LI1);
    else if (plan.kernel == 2) NB_DISPATCH(LIW);
    else NB_DISPATCH(LJ);
#undef LI1
#undef LIW
#undef LJ
    ++*launches;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    if (args.n_planes > 1) {
        const int T = nb_reduce_threads(args.n_act, args.n_planes);
        const int R = RED_THREADS / T;
        if (order == 8) reduce_partials_kernel<13><<<(args.n_act + R - 1) / R, RED_THREADS, 0, st>>>(args, T);
        else reduce_partials_kernel<10><<<(args.n_act + R - 1) / R, RED_THREADS, 0, st>>>(args, T);
        ++*launches;
        e = cudaGetLastError();
    }
    return e;
}

cudaError_t nb_launch_force_devplan(const ForceArgs& args_, bool eps_is_zero, int order, int n_sm, int Npad, cudaStream_t st, int* launches)
{
    ForceArgs args = args_, args_lj = args_;
    args.n_tiles = Npad / LI_TJ; args_lj.n_tiles = Npad / LJ_TJ;
    const int g_li = n_sm * LI_CTAS_PER_SM, g_lj = n_sm * LJ_CTAS_PER_SM;
#define ALL3(E, O)                                                      \
    force_lj_kernel<E, O><<<g_lj, LJ_THREADS, 0, st>>>(args_lj);        \
    force_li_kernel<E, LI_W, O><<<g_li, LI_THREADS, 0, st>>>(args);     \
    force_li_kernel<E, 1, O><<<g_li, LI_THREADS, 0, st>>>(args)
    NB_DISPATCH(ALL3);
#undef ALL3
    if (order == 8) reduce_partials_kernel<13><<<n_sm * 4, RED_THREADS, 0, st>>>(args, 1);
    else reduce_partials_kernel<10><<<n_sm * 4, RED_THREADS, 0, st>>>(args, 1);
    *launches += 4;
    return cudaGetLastError();
}

void nb_force_occupancy(int* li, int* lj)
{
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(li, force_li_kernel<false, 1, 6>, LI_THREADS, 0);
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(lj, force_lj_kernel<false, 6>, LJ_THREADS, 0);
}
