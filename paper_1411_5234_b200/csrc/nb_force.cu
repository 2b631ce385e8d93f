// nb_force.cu — the pairwise evaluation: acceleration, jerk, snap and
// potential of eq. (1)-(2) and their time derivatives (R3), for
// the active particles against all N predicted j-records.  fp64 on the FP64 ALU pipe; tensor cores
// are not used (no dense contraction).  Two kernel shapes, both writing per-slice partial sums that are
// added in a fixed order (the "Bfactor" j-split of PAPER.md:59-65, made deterministic):
//   li_body  "CTA tiles" (n_act >= LI_MIN_ACT): a thread owns one active particle in registers; the CTA streams
//            j-tiles of 128 records into shared memory with 1-D TMA bulk copies (UBLKCP) signalled on mbarriers,
//            double-buffered; every lane reads the same j-record (broadcast LDS).
//   wu_body  "warp units" (smaller active sets, the paper's Bfactor regime): every warp is its own worker with a
//            private double-buffered ring of 64-record tiles (one bulk copy per tile).  A unit is p = 32, 16, .. 1
//            particles: the lanes are split p ways over particles and 32/p ways over the records of a step, from
//            lanes-over-i (p = 32) to lanes-over-j (p = 1); the 32/p lane sums of a particle are combined with a
//            warp-shuffle butterfly.  In a device-planned block step with few units the warp PREDICTS the records of
//            its slice from the state instead of reading them (the predictor's pass over all N is skipped).
// The FP64 instructions of the pair evaluation are written one per source line between NB_SCHED_BEGIN / NB_SCHED_END, in the order
// the FP64 pipe is to see them (operand-reuse chains); build.py passes this file's cubin through sass_sched.py, which
// puts the machine code of the CTA-tile loops back into that order after ptxas (results bit-identical, tests compare).
// ORDER = 6 is the scheme of the north star (a, jerk, snap, pot); 4 (a, jerk, pot) and 8 (+ crackle) are the other
// Hermite orders the paper names (R21, R22).
// Work items (i-unit, j-slice) are handed out by an atomic queue, not by a static stride: warps of
// co-resident CTAs do NOT get equal shares of the FP64 pipe (measured: of three CTAs with equal work on
// one SM the first finished after 40 % of the time the last one needed), so a static partition ends in a
// long tail of under-occupied SMs.  Where an item's sums are stored depends only on the item, so the
// results stay bitwise reproducible.
#include "nb_internal.h"
#include "nb_plan.h"
#include "nb_predict.h"
#include "nb_reduce.h"

namespace {

struct Sums { double ax, ay, az, jx, jy, jz, sx, sy, sz, p, cx, cy, cz; };   // cx..cz: crackle, 8th order only

struct IPart { double x, y, z, vx, vy, vz, ax, ay, az, jx, jy, jz; };        // jx..jz: predicted jerk, 8th order only

struct JRec { double x, y, z, m, vx, vy, vz, ax, ay, az, jx, jy, jz; };      // one predicted j-record in registers

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
// fp64 reciprocal-square-root seed: MUFU.RSQ64H works on the high word only (about 20 good bits).
__device__ __forceinline__ double rsqrt_seed(double s)
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(s));
    return y;
}
// 2 c by incrementing the exponent field (integer pipe, not the FP64 pipe).  Exact for every normal c; for
// c = +-0 it returns +-2^-1022 instead of 0, which only ever multiplies a finite u and is added to da.
__device__ __forceinline__ double twice(double c)
{
    return __hiloint2double(__double2hiint(c) + 0x00100000, __double2loint(c));
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
// 2 c by incrementing the exponent field (integer pipe): see twice()
#define VTWICE(d, a) asm volatile("{\n\t.reg .b32 lo, hi;\n\tmov.b64 {lo, hi}, %1;\n\tadd.s32 hi, hi, 0x100000;\n\tmov.b64 %0, {lo, hi};\n\t}" : "=d"(d) : "d"(a))
#define BOTH for (int k = 0; k < 2; ++k)


// NB_SCHED_BEGIN (sass_sched.py puts the machine code of these lines back into the order written here)
// PINNED: for the instantiations sass_sched.py does not reschedule (warp units and block steps at the 6th order).  There a
// branch that is never taken (v >= 0) but that ptxas cannot see through stands before each pair's run of 18 DFMAs; the sums are
// live on its taken side, so ptxas cannot interleave the two runs and chains the sources through the reuse cache itself
// (21-25 of 48 three-source DFMAs left uncovered instead of 29-33).
#define PIN(v) if (PINNED && __double2hiint(v) < 0) return;
#ifndef NB_PIN_UNSCHEDULED
#define NB_PIN_UNSCHEDULED true        // build.py: false with NB_SASS_SCHED=all (then sass_sched.py reschedules those loops too)
#endif
template <bool EPS0, bool MASK, bool PINNED = false>
__device__ __forceinline__ void pair2(const IPart& pi, const JRec (&J)[2], const double eps2, const bool (&self)[2], Sums& S)
{
    // ONE FP64 instruction per source line, in the order the pipe is to see them (pair 0 and pair 1 of the two records):
    // sass_sched.py sorts the machine code of a basic block by these line numbers.
    double dx0, dy0, dz0, dvx0, dvy0, dvz0, dax0, day0, daz0, s0, rv0, rq0, B0, y00, t0, e0, h0, y0, yy0, mr0, z0, q0, c10, c20, c30;
    double dx1, dy1, dz1, dvx1, dvy1, dvz1, dax1, day1, daz1, s1, rv1, rq1, B1, y01, t1, e1, h1, y1, yy1, mr1, z1, q1, c11, c21, c31;
    double ux0, uy0, uz0, wx0, wy0, wz0, ux1, uy1, uz1, wx1, wy1, wz1;
    // differences, with B = dv.dv (duplicate operands: two-cycle DFMAs) threaded through them
    VSUB(dvz0, J[0].vz, pi.vz);
    VSUB(dvz1, J[1].vz, pi.vz);
    VSUB(dvy0, J[0].vy, pi.vy);
    VSUB(dvy1, J[1].vy, pi.vy);
    VSUB(dvx0, J[0].vx, pi.vx);
    VSUB(dvx1, J[1].vx, pi.vx);
    VMUL(B0, dvz0, dvz0);
    VMUL(B1, dvz1, dvz1);
    VSUB(dz0, J[0].z, pi.z);
    VSUB(dz1, J[1].z, pi.z);
    VSUB(daz0, J[0].az, pi.az);
    VSUB(daz1, J[1].az, pi.az);
    VFMA(B0, dvy0, dvy0, B0);
    VFMA(B1, dvy1, dvy1, B1);
    VSUB(dy0, J[0].y, pi.y);
    VSUB(dy1, J[1].y, pi.y);
    VSUB(day0, J[0].ay, pi.ay);
    VSUB(day1, J[1].ay, pi.ay);
    VFMA(B0, dvx0, dvx0, B0);
    VFMA(B1, dvx1, dvx1, B1);
    VSUB(dx0, J[0].x, pi.x);
    VSUB(dx1, J[1].x, pi.x);
    VSUB(dax0, J[0].ax, pi.ax);
    VSUB(dax1, J[1].ax, pi.ax);
    // s = dx.dx + eps2, rv = dx.dv, B += dx.da: groups of three that share d_c in slot A
    VFMA(s0, dz0, dz0, eps2);
    VMUL(rv0, dz0, dvz0);
    VFMA(B0, dz0, daz0, B0);
    VFMA(s1, dz1, dz1, eps2);
    VMUL(rv1, dz1, dvz1);
    VFMA(B1, dz1, daz1, B1);
    VFMA(s0, dy0, dy0, s0);
    VFMA(rv0, dy0, dvy0, rv0);
    VFMA(B0, dy0, day0, B0);
    VFMA(s1, dy1, dy1, s1);
    VFMA(rv1, dy1, dvy1, rv1);
    VFMA(B1, dy1, day1, B1);
    VFMA(s0, dx0, dx0, s0);
    VFMA(rv0, dx0, dvx0, rv0);
    VFMA(B0, dx0, dax0, B0);
    VFMA(s1, dx1, dx1, s1);
    VFMA(rv1, dx1, dvx1, rv1);
    VFMA(B1, dx1, dax1, B1);
    if (EPS0 && MASK) {                                   // eps = 0: keep the masked self pair finite
        s0 = self[0] ? 1.0 : s0;
        s1 = self[1] ? 1.0 : s1;
    }
    // y = s^(-1/2): MUFU.RSQ64H seed (e ~ 2^-20), then one cubic step y = y0 + y0 e (1/2 + 3/8 e), e = 1 - s y0^2,
    // which leaves 5/16 e^3 < 2^-60
    VRSQ(y00, s0);
    VRSQ(y01, s1);
    VMUL(rq0, rv0, rv0);
    VMUL(rq1, rv1, rv1);
    VMUL(t0, y00, y00);
    VMUL(t1, y01, y01);
    VFNMA(e0, s0, t0, 1.0);
    VFNMA(e1, s1, t1, 1.0);
    VFMA(h0, e0, 0.375, 0.5);
    VFMA(h1, e1, 0.375, 0.5);
    VMUL(t0, e0, h0);
    VMUL(t1, e1, h1);
    VFMA(y0, y00, t0, y00);
    VFMA(y1, y01, t1, y01);
    // scalars: yy = 1/s, mr = m_j/sqrt(s), q = m_j s^(-3/2), c1 = -3 alpha, c2 = -6 alpha, c3 = -3 beta
    //          with alpha = rv/s, beta = B/s + alpha^2 = (B + rv^2/s)/s
    VMUL(yy0, y0, y0);
    VMUL(yy1, y1, y1);
    VMUL(mr0, y0, J[0].m);
    VMUL(mr1, y1, J[1].m);
    VMUL(z0, yy0, -3.0);
    VMUL(z1, yy1, -3.0);
    VMUL(q0, mr0, yy0);
    VFMA(B0, rq0, yy0, B0);                            // yy stays in slot B
    VMUL(q1, mr1, yy1);
    VFMA(B1, rq1, yy1, B1);                            // yy stays in slot B
    VMUL(c10, z0, rv0);
    VMUL(c11, z1, rv1);
    VMUL(c30, z0, B0);
    VMUL(c31, z1, B1);
    VTWICE(c20, c10);
    VTWICE(c21, c11);
    PIN(s0)
    // u = dv + c1 dx, w = da + c3 dx + c2 u, sums += q (dx, u, w): 18 three-source DFMAs per pair in one run;
    // each shares a source with its predecessor in the same slot (A: c1, c3, q, c2; B: d_c, u_c)
    if (MASK) mr0 = self[0] ? 0.0 : mr0;              // j != i (eq. 1); a, jerk, snap get exactly 0 from the self pair
    VADD(S.p, S.p, mr0);
    VFMA(ux0, c10, dx0, dvx0);
    VFMA(uy0, c10, dy0, dvy0);
    VFMA(uz0, c10, dz0, dvz0);
    VFMA(wz0, c30, dz0, daz0);
    VFMA(wy0, c30, dy0, day0);
    VFMA(wx0, c30, dx0, dax0);
    VFMA(S.ax, q0, dx0, S.ax);
    VFMA(S.ay, q0, dy0, S.ay);
    VFMA(S.az, q0, dz0, S.az);
    VFMA(S.jx, q0, ux0, S.jx);
    VFMA(wx0, c20, ux0, wx0);
    VFMA(wy0, c20, uy0, wy0);
    VFMA(wz0, c20, uz0, wz0);
    VFMA(S.jz, q0, uz0, S.jz);
    VFMA(S.jy, q0, uy0, S.jy);
    VFMA(S.sx, q0, wx0, S.sx);
    VFMA(S.sy, q0, wy0, S.sy);
    VFMA(S.sz, q0, wz0, S.sz);
    PIN(yy0)
    if (MASK) mr1 = self[1] ? 0.0 : mr1;              // j != i (eq. 1); a, jerk, snap get exactly 0 from the self pair
    VADD(S.p, S.p, mr1);
    VFMA(ux1, c11, dx1, dvx1);
    VFMA(uy1, c11, dy1, dvy1);
    VFMA(uz1, c11, dz1, dvz1);
    VFMA(wz1, c31, dz1, daz1);
    VFMA(wy1, c31, dy1, day1);
    VFMA(wx1, c31, dx1, dax1);
    VFMA(S.ax, q1, dx1, S.ax);
    VFMA(S.ay, q1, dy1, S.ay);
    VFMA(S.az, q1, dz1, S.az);
    VFMA(S.jx, q1, ux1, S.jx);
    VFMA(wx1, c21, ux1, wx1);
    VFMA(wy1, c21, uy1, wy1);
    VFMA(wz1, c21, uz1, wz1);
    VFMA(S.jz, q1, uz1, S.jz);
    VFMA(S.jy, q1, uy1, S.jy);
    VFMA(S.sx, q1, wx1, S.sx);
    VFMA(S.sy, q1, wy1, S.sy);
    VFMA(S.sz, q1, wz1, S.sz);
    PIN(yy1)
}

// ---------------------------------------------------------------------------------------------
// 4th-order variant (R21): acceleration, jerk and potential only.  32 FP64-pipe instructions per
// pair (17 DFMA + 8 DMUL + 7 DADD) + 1 MUFU.RSQ64H; the snap sums stay 0.  Two j-records at a time, FP64 instruction
// order as in pair2 (the nine three-source DFMAs of a pair in one pinned run).
// ---------------------------------------------------------------------------------------------
template <bool EPS0, bool MASK>
__device__ __forceinline__ void pair2_o4(const IPart& pi, const JRec (&J)[2], const double eps2, const bool (&self)[2], Sums& S)
{
    double dx0, dy0, dz0, dvx0, dvy0, dvz0, s0, rv0, y00, t0, e0, h0, y0, yy0, mr0, z0, q0, c10, ux0, uy0, uz0;
    double dx1, dy1, dz1, dvx1, dvy1, dvz1, s1, rv1, y01, t1, e1, h1, y1, yy1, mr1, z1, q1, c11, ux1, uy1, uz1;
    VSUB(dz0, J[0].z, pi.z);
    VSUB(dz1, J[1].z, pi.z);
    VSUB(dvz0, J[0].vz, pi.vz);
    VSUB(dvz1, J[1].vz, pi.vz);
    VSUB(dy0, J[0].y, pi.y);
    VSUB(dy1, J[1].y, pi.y);
    VSUB(dvy0, J[0].vy, pi.vy);
    VSUB(dvy1, J[1].vy, pi.vy);
    VSUB(dx0, J[0].x, pi.x);
    VSUB(dx1, J[1].x, pi.x);
    VSUB(dvx0, J[0].vx, pi.vx);
    VSUB(dvx1, J[1].vx, pi.vx);
    VFMA(s0, dz0, dz0, eps2);
    VMUL(rv0, dz0, dvz0);
    VFMA(s1, dz1, dz1, eps2);
    VMUL(rv1, dz1, dvz1);
    VFMA(s0, dy0, dy0, s0);
    VFMA(rv0, dy0, dvy0, rv0);
    VFMA(s1, dy1, dy1, s1);
    VFMA(rv1, dy1, dvy1, rv1);
    VFMA(s0, dx0, dx0, s0);
    VFMA(rv0, dx0, dvx0, rv0);
    VFMA(s1, dx1, dx1, s1);
    VFMA(rv1, dx1, dvx1, rv1);
    if (EPS0 && MASK) {
        s0 = self[0] ? 1.0 : s0;
        s1 = self[1] ? 1.0 : s1;
    }
    VRSQ(y00, s0);
    VRSQ(y01, s1);
    VMUL(t0, y00, y00);
    VMUL(t1, y01, y01);
    VFNMA(e0, s0, t0, 1.0);
    VFNMA(e1, s1, t1, 1.0);
    VFMA(h0, e0, 0.375, 0.5);
    VFMA(h1, e1, 0.375, 0.5);
    VMUL(t0, e0, h0);
    VMUL(t1, e1, h1);
    VFMA(y0, y00, t0, y00);
    VFMA(y1, y01, t1, y01);
    VMUL(yy0, y0, y0);
    VMUL(yy1, y1, y1);
    VMUL(mr0, y0, J[0].m);
    VMUL(mr1, y1, J[1].m);
    VMUL(z0, yy0, -3.0);
    VMUL(z1, yy1, -3.0);
    VMUL(q0, mr0, yy0);
    VMUL(q1, mr1, yy1);
    VMUL(c10, z0, rv0);
    VMUL(c11, z1, rv1);
    if (MASK) mr0 = self[0] ? 0.0 : mr0;
    VADD(S.p, S.p, mr0);
    VFMA(ux0, c10, dx0, dvx0);
    VFMA(uy0, c10, dy0, dvy0);
    VFMA(uz0, c10, dz0, dvz0);
    VFMA(S.az, q0, dz0, S.az);
    VFMA(S.ay, q0, dy0, S.ay);
    VFMA(S.ax, q0, dx0, S.ax);
    VFMA(S.jx, q0, ux0, S.jx);
    VFMA(S.jy, q0, uy0, S.jy);
    VFMA(S.jz, q0, uz0, S.jz);
    if (MASK) mr1 = self[1] ? 0.0 : mr1;
    VADD(S.p, S.p, mr1);
    VFMA(ux1, c11, dx1, dvx1);
    VFMA(uy1, c11, dy1, dvy1);
    VFMA(uz1, c11, dz1, dvz1);
    VFMA(S.az, q1, dz1, S.az);
    VFMA(S.ay, q1, dy1, S.ay);
    VFMA(S.ax, q1, dx1, S.ax);
    VFMA(S.jx, q1, ux1, S.jx);
    VFMA(S.jy, q1, uy1, S.jy);
    VFMA(S.jz, q1, uz1, S.jz);
}

// ---------------------------------------------------------------------------------------------
// 8th-order variant (R22): crackle added.  With T3 = 3 dv.da + dx.dj and
// gamma = T3/s + alpha (3 beta - 4 alpha^2):  crackle term = q (dj - 9 alpha w - 9 beta u - 3 gamma dx).
// 84 FP64-pipe instructions per pair + 1 MUFU.RSQ64H; one pair at a time (ptxas schedules it; 2 x 12 differences would
// not fit the register budget).
// ---------------------------------------------------------------------------------------------
template <bool EPS0, bool MASK>
__device__ __forceinline__ void pair_o8(const IPart& pi, const JRec& J, const double eps2, const bool self, Sums& S)
{
    const double dx = J.x - pi.x, dy = J.y - pi.y, dz = J.z - pi.z;
    const double dvx = J.vx - pi.vx, dvy = J.vy - pi.vy, dvz = J.vz - pi.vz;
    const double dax = J.ax - pi.ax, day = J.ay - pi.ay, daz = J.az - pi.az;
    const double djx = J.jx - pi.jx, djy = J.jy - pi.jy, djz = J.jz - pi.jz;
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
    const double mr = M(y, J.m);
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

// NB_SCHED_END
// ---------------------------------------------------------------------------------------------
// Mixed precision (nb_config.precision = NB_PREC_MIXED; HiGPUs uses DP "to calculate reciprocal distances
// and to cumulate accelerations" and SP elsewhere).  Position differences in fp64, converted once; everything else of the
// pair in fp32 (46 FP32-pipe instructions + 3 DADD + 3 F2F + 1 MUFU.RSQ); the fp32 sums of one j-tile are flushed into
// fp64 accumulators by the caller.  The formulas are those of pair2 (R3); the order is left to ptxas.
// ---------------------------------------------------------------------------------------------
struct IPartM { double x, y, z; float vx, vy, vz, ax, ay, az; };
struct SumsF { float ax, ay, az, jx, jy, jz, sx, sy, sz, p; };
struct JRecM { double x, y, z; float m, vx, vy, vz, ax, ay, az; };

__device__ __forceinline__ double f2_as_double(float lo, float hi) { return __hiloint2double(__float_as_int(hi), __float_as_int(lo)); }

__device__ __forceinline__ JRecM load_recm(const float4* r)
{
    const float4 a = r[0], b = r[1], c = r[2], d = r[3];
    return JRecM{f2_as_double(a.x, a.y), f2_as_double(a.z, a.w), f2_as_double(b.x, b.y), b.z, b.w, c.x, c.y, c.z, c.w, d.x};
}

__device__ __forceinline__ float rsqrt_f32(float s)
{
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(s));
    return y;
}

template <bool EPS0, bool MASK>
__device__ __forceinline__ void pair_mixed(const IPartM& pi, const JRecM& J, const float eps2, const bool self, SumsF& S)
{
    const float dx = (float)(J.x - pi.x), dy = (float)(J.y - pi.y), dz = (float)(J.z - pi.z);   // DP difference, then SP
    const float dvx = J.vx - pi.vx, dvy = J.vy - pi.vy, dvz = J.vz - pi.vz;
    const float dax = J.ax - pi.ax, day = J.ay - pi.ay, daz = J.az - pi.az;
    float s = fmaf(dx, dx, fmaf(dy, dy, fmaf(dz, dz, eps2)));
    if (EPS0 && MASK) s = self ? 1.f : s;                // eps = 0: keep the masked self pair finite
    const float y = rsqrt_f32(s);                        // MUFU.RSQ: about 2^-22 relative
    const float rv = fmaf(dx, dvx, fmaf(dy, dvy, dz * dvz));
    const float B = fmaf(dx, dax, fmaf(dy, day, fmaf(dz, daz, fmaf(dvx, dvx, fmaf(dvy, dvy, dvz * dvz)))));
    const float yy = y * y, mr = J.m * y, q = mr * yy, z = -3.f * yy;
    const float alpha = yy * rv, c1 = z * rv;            // c1 = -3 alpha
    const float c3 = fmaf(c1, alpha, z * B), c2 = c1 + c1;   // -3 beta, -6 alpha
    const float ux = fmaf(c1, dx, dvx), uy = fmaf(c1, dy, dvy), uz = fmaf(c1, dz, dvz);
    const float wx = fmaf(c2, ux, fmaf(c3, dx, dax)), wy = fmaf(c2, uy, fmaf(c3, dy, day)), wz = fmaf(c2, uz, fmaf(c3, dz, daz));
    S.ax = fmaf(q, dx, S.ax); S.ay = fmaf(q, dy, S.ay); S.az = fmaf(q, dz, S.az);
    S.jx = fmaf(q, ux, S.jx); S.jy = fmaf(q, uy, S.jy); S.jz = fmaf(q, uz, S.jz);
    S.sx = fmaf(q, wx, S.sx); S.sy = fmaf(q, wy, S.sy); S.sz = fmaf(q, wz, S.sz);
    S.p += (MASK && self) ? 0.f : mr;                    // j != i (eq. 1)
}

// ---------------------------------------------------------------------------------------------
// records: one predicted particle is Q = 5 (7 at the 8th order) double2, nb_internal.h
// ---------------------------------------------------------------------------------------------
template <int ORDER>
__device__ __forceinline__ JRec load_rec(const double2* r)
{
    const double2 a = r[0], b = r[1], c = r[2], d = r[3], e = r[4];
    JRec J{a.x, a.y, b.x, b.y, c.x, c.y, d.x, d.y, e.x, e.y, 0.0, 0.0, 0.0};
    if (ORDER == 8) { const double2 f = r[5], g = r[6]; J.jx = f.x; J.jy = f.y; J.jz = g.x; }
    return J;
}

__device__ __forceinline__ IPart ipart_of(const JRec& J) { return IPart{J.x, J.y, J.z, J.vx, J.vy, J.vz, J.ax, J.ay, J.az, J.jx, J.jy, J.jz}; }

// the i-particle's own predicted record: read from the record array, or predicted from the state with the predictor's
// fma chain (bit-identical)
template <int ORDER, bool PREDICT>
__device__ __forceinline__ IPart load_ipart(const ForceArgs& A, int i)
{
    constexpr int Q = nb_rec_q(ORDER);
    if (PREDICT) {
        double2 r[Q];
        nb_predict_record<ORDER>(nb_load_pstate<ORDER>(A.st0, A.st1, A.st2, A.st3, A.st4, A.st5, A.st6, i), A.t_pred, false, r);
        return ipart_of(load_rec<ORDER>(r));
    }
    return ipart_of(load_rec<ORDER>(A.rec + (size_t)i * Q));
}

// partial sums: NC = 10 components (a, jerk, snap, pot), 13 at the 8th order (+ crackle), per slice and row
template <int ORDER>
__device__ __forceinline__ void store_sums(const ForceArgs& A, int slice, int k, const Sums& S)
{
    constexpr int NC = ORDER == 8 ? 13 : 10;
    if (A.n_split > 1) {
        const PartialLayout L(NC, A.ld, A.n_split, A.slice_minor != 0);     // nb_reduce.h: [s][c][k] or [c][k][s]
        double* P = A.partial + (size_t)slice * L.stride_s + (size_t)k * L.stride_k;
        const size_t sc = L.stride_c;
        P[0] = S.ax; P[sc] = S.ay; P[2 * sc] = S.az;
        P[3 * sc] = S.jx; P[4 * sc] = S.jy; P[5 * sc] = S.jz;
        P[6 * sc] = S.sx; P[7 * sc] = S.sy; P[8 * sc] = S.sz; P[9 * sc] = S.p;
        if (ORDER == 8) { P[10 * sc] = S.cx; P[11 * sc] = S.cy; P[12 * sc] = S.cz; }
    } else {
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

constexpr int N_BARS = WU_WARPS * WU_STAGES > LI_STAGES ? WU_WARPS * WU_STAGES : LI_STAGES;
static_assert((LI_STAGES & (LI_STAGES - 1)) == 0 && (WU_STAGES & (WU_STAGES - 1)) == 0, "stage counts must be powers of two");
static_assert(LI_TJ % 2 == 0 && WU_TJ == 64, "pair2 takes two j-records at a time; a warp predicts a tile as lane, lane + 32");

__device__ __forceinline__ void init_barriers(unsigned long long* bars)
{
    if (threadIdx.x == 0) {
        for (int s = 0; s < N_BARS; ++s) mbar_init(smem_u32(&bars[s]), 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
}

// Device-planned launch (nb_run_blocks): take the plan the scheduler left in device memory.  False: the step is not taken.
__device__ __forceinline__ bool take_devplan(ForceArgs& A)
{
    const DevPlan* d = A.dp;
    if (d->stop) return false;
    A.n_act = d->n_act; A.n_units = d->n_units; A.n_split = d->n_split; A.slice_tiles = d->slice_tiles;
    A.n_items = d->n_items; A.ld = d->ld; A.predict = d->predict; A.t_pred = d->t_next; A.slice_minor = nb_slice_minor(d->red_T);
    return true;
}

// The worker that finds the queue empty last puts both counters back to 0 for the next launch.
__device__ __forceinline__ void queue_retire(int* queue, int n_workers)
{
    __threadfence();
    if (atomicAdd(queue + 1, 1) == n_workers - 1) { queue[0] = 0; queue[1] = 0; }
}

// ---------------------------------------------------------------------------------------------
// CTA tiles: a work item is (i-tile of 128 particles, j-slice)
// ---------------------------------------------------------------------------------------------
template <bool EPS0, int ORDER>
__device__ __forceinline__ void li_body(const ForceArgs& A, double2* smem, unsigned long long* full)
{
    constexpr int Q = nb_rec_q(ORDER);
    constexpr uint32_t TILE_BYTES = LI_TJ * Q * 16;
    __shared__ int next_item;
    const int tid = threadIdx.x;

    // one elected thread stages j-tile `tile` into stage `st`: one bulk copy, one barrier
    auto stage_tile = [&](int tile, int st) {
        const uint32_t bar = smem_u32(&full[st]);
        mbar_expect_tx(bar, TILE_BYTES);
        bulk_g2s(smem_u32(smem + (size_t)st * LI_TJ * Q), A.rec + (size_t)tile * LI_TJ * Q, TILE_BYTES, bar);
    };

    uint32_t uses = 0;   // j-tiles this CTA has consumed so far: stage = uses % STAGES, parity = (uses / STAGES) & 1
    for (int round = 0;; ++round) {
        // the first item is the CTA's own number, further ones come from the queue (which counts from gridDim.x)
        if (tid == 0) next_item = round == 0 ? (int)blockIdx.x : (int)gridDim.x + atomicAdd(A.queue, 1);
        __syncthreads();
        const int item = next_item;
        __syncthreads();                                   // everyone has read next_item before it is overwritten
        if (item >= A.n_items) break;
        const int unit = item % A.n_units, slice = item / A.n_units;
        const int t0 = slice * A.slice_tiles;
        const int nt = min(A.slice_tiles, A.n_tiles - t0);

        if (tid == 0)
            for (int f = 0; f < LI_STAGES && f < nt; ++f) stage_tile(t0 + f, (uses + f) & (LI_STAGES - 1));

        const int k = unit * LI_UNIT + tid;
        const bool valid = k < A.n_act;
        const int kk = valid ? k : 0;
        const int ii = A.idx ? A.idx[kk] : kk;
        const IPart pi = load_ipart<ORDER, false>(A, ii);
        Sums acc{0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0};

        for (int t = 0; t < nt; ++t) {
            const uint32_t u = uses + t;
            const int st = u & (LI_STAGES - 1);
            mbar_wait(smem_u32(&full[st]), (u / LI_STAGES) & 1);
            const int jbase = (t0 + t) * LI_TJ;
            // the self pair (reading R4) lies in one j-tile per particle: only a warp that has one of its own
            // particles in this tile runs the loop that masks by index
            const bool own = (unsigned)(ii - jbase) < (unsigned)LI_TJ;
            const double2* tp = smem + (size_t)st * LI_TJ * Q;
            if (ORDER == 8) {
                if (__any_sync(0xffffffffu, own)) {
#pragma unroll 2
                    for (int jj = 0; jj < LI_TJ; ++jj) pair_o8<EPS0, true>(pi, load_rec<ORDER>(tp + jj * Q), A.eps2, jbase + jj == ii, acc);
                } else {
#pragma unroll 2
                    for (int jj = 0; jj < LI_TJ; ++jj) pair_o8<EPS0, false>(pi, load_rec<ORDER>(tp + jj * Q), A.eps2, false, acc);
                }
            } else if (__any_sync(0xffffffffu, own)) {
#pragma unroll 1
                for (int jj = 0; jj < LI_TJ; jj += 2) {
                    const JRec J[2] = {load_rec<ORDER>(tp + jj * Q), load_rec<ORDER>(tp + (jj + 1) * Q)};
                    const bool self[2] = {jbase + jj == ii, jbase + jj + 1 == ii};
                    if (ORDER == 4) pair2_o4<EPS0, true>(pi, J, A.eps2, self, acc);
                    else pair2<EPS0, true>(pi, J, A.eps2, self, acc);
                }
            } else {
#pragma unroll 1
                for (int jj = 0; jj < LI_TJ; jj += 2) {
                    const JRec J[2] = {load_rec<ORDER>(tp + jj * Q), load_rec<ORDER>(tp + (jj + 1) * Q)};
                    const bool self[2] = {false, false};
                    if (ORDER == 4) pair2_o4<EPS0, false>(pi, J, A.eps2, self, acc);
                    else pair2<EPS0, false>(pi, J, A.eps2, self, acc);
                }
            }
            __syncthreads();                                   // every warp is done with stage st
            if (tid == 0 && t + LI_STAGES < nt) stage_tile(t0 + t + LI_STAGES, st);
        }
        uses += nt;
        if (valid || A.n_split > 1) store_sums<ORDER>(A, slice, k, acc);
    }
    if (tid == 0) queue_retire(A.queue, gridDim.x);
}

// ---------------------------------------------------------------------------------------------
// CTA tiles in mixed precision (6th order): li_body's structure over the 64-B records; the fp32 sums of a j-tile (128
// pairs per particle) are added into the fp64 accumulators after every tile ("DP ... to cumulate")
// ---------------------------------------------------------------------------------------------
constexpr uint32_t LIM_TILE_BYTES = LI_TJ * 64;

template <bool EPS0>
__device__ __forceinline__ void li_mixed_body(const ForceArgs& A, double2* smem_, unsigned long long* full)
{
    float4* smem = (float4*)smem_;
    __shared__ int next_item_m;
    const int tid = threadIdx.x;
    const float eps2 = (float)A.eps2;

    auto stage_tile = [&](int tile, int st) {
        const uint32_t bar = smem_u32(&full[st]);
        mbar_expect_tx(bar, LIM_TILE_BYTES);
        bulk_g2s(smem_u32(smem + (size_t)st * LI_TJ * 4), A.recm + (size_t)tile * LI_TJ * 4, LIM_TILE_BYTES, bar);
    };

    uint32_t uses = 0;
    for (int round = 0;; ++round) {
        if (tid == 0) next_item_m = round == 0 ? (int)blockIdx.x : (int)gridDim.x + atomicAdd(A.queue, 1);
        __syncthreads();
        const int item = next_item_m;
        __syncthreads();
        if (item >= A.n_items) break;
        const int unit = item % A.n_units, slice = item / A.n_units;
        const int t0 = slice * A.slice_tiles;
        const int nt = min(A.slice_tiles, A.n_tiles - t0);
        if (tid == 0)
            for (int f = 0; f < LI_STAGES && f < nt; ++f) stage_tile(t0 + f, (uses + f) & (LI_STAGES - 1));

        const int k = unit * LI_UNIT + tid;
        const bool valid = k < A.n_act;
        const int kk = valid ? k : 0;
        const int ii = A.idx ? A.idx[kk] : kk;
        const JRecM me = load_recm(A.recm + (size_t)ii * 4);
        const IPartM pi{me.x, me.y, me.z, me.vx, me.vy, me.vz, me.ax, me.ay, me.az};
        Sums acc{0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0};

        for (int t = 0; t < nt; ++t) {
            const uint32_t u = uses + t;
            const int st = u & (LI_STAGES - 1);
            mbar_wait(smem_u32(&full[st]), (u / LI_STAGES) & 1);
            const int jbase = (t0 + t) * LI_TJ;
            const bool own = (unsigned)(ii - jbase) < (unsigned)LI_TJ;
            const float4* tp = smem + (size_t)st * LI_TJ * 4;
            SumsF f{0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
            if (__any_sync(0xffffffffu, own)) {
#pragma unroll 4
                for (int jj = 0; jj < LI_TJ; ++jj) pair_mixed<EPS0, true>(pi, load_recm(tp + jj * 4), eps2, jbase + jj == ii, f);
            } else {
#pragma unroll 4
                for (int jj = 0; jj < LI_TJ; ++jj) pair_mixed<EPS0, false>(pi, load_recm(tp + jj * 4), eps2, false, f);
            }
            acc.ax += (double)f.ax; acc.ay += (double)f.ay; acc.az += (double)f.az;
            acc.jx += (double)f.jx; acc.jy += (double)f.jy; acc.jz += (double)f.jz;
            acc.sx += (double)f.sx; acc.sy += (double)f.sy; acc.sz += (double)f.sz; acc.p += (double)f.p;
            __syncthreads();
            if (tid == 0 && t + LI_STAGES < nt) stage_tile(t0 + t + LI_STAGES, st);
        }
        uses += nt;
        if (valid || A.n_split > 1) store_sums<6>(A, slice, k, acc);
    }
    if (tid == 0) queue_retire(A.queue, gridDim.x);
}

// ---------------------------------------------------------------------------------------------
// warp units: a work item is (unit of p particles, j-slice), one warp per item
// ---------------------------------------------------------------------------------------------
template <bool EPS0, int ORDER, bool PREDICT>
__device__ __forceinline__ void wu_body(const ForceArgs& A, double2* smem, unsigned long long* full_all)
{
    constexpr int Q = nb_rec_q(ORDER);
    constexpr uint32_t TILE_BYTES = WU_TJ * Q * 16;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double2* ring = smem + (size_t)warp * WU_STAGES * WU_TJ * Q;        // this warp's private stages
    unsigned long long* full = full_all + warp * WU_STAGES;

    auto stage_tile = [&](int tile, int st) {                          // lane 0 only
        const uint32_t bar = smem_u32(&full[st]);
        mbar_expect_tx(bar, TILE_BYTES);
        bulk_g2s(smem_u32(ring + (size_t)st * WU_TJ * Q), A.rec + (size_t)tile * WU_TJ * Q, TILE_BYTES, bar);
    };

    // every worker's first item is its own number (no queue traffic at all when there is at most one item per warp);
    // further items come from the queue, which counts from n_workers
    const int n_workers = gridDim.x * WU_WARPS;
    const bool queued = A.n_items > n_workers;
    uint32_t uses = 0;
    for (int round = 0;; ++round) {
        int item;
        if (round == 0) item = (int)(blockIdx.x * WU_WARPS + warp);
        else if (queued) {
            item = 0;
            if (lane == 0) item = n_workers + atomicAdd(A.queue, 1);
            item = __shfl_sync(0xffffffffu, item, 0);
        } else item = A.n_items;
        if (item >= A.n_items) break;
        const int unit = item % A.n_units, slice = item / A.n_units;
        const int t0 = slice * A.slice_tiles;
        const int nt = min(A.slice_tiles, A.n_tiles - t0);
        if (!PREDICT && lane == 0)
            for (int f = 0; f < WU_STAGES && f < nt; ++f) stage_tile(t0 + f, (uses + f) & (WU_STAGES - 1));

        // lanes: p ways over the unit's particles, LJ = 32 / p ways over the records of a step
        int k0, p, nvalid;
        nb_wu_unit(A.n_act, unit, &k0, &p, &nvalid);
        const int LJ = 32 / p;                              // powers of two
        const int lj = lane & (LJ - 1), part = lane >> (__ffs(LJ) - 1);
        const bool valid = part < nvalid;
        const int k = k0 + (valid ? part : 0);
        const int ii = A.idx ? A.idx[k] : k;
        const IPart pi = load_ipart<ORDER, PREDICT>(A, ii);
        Sums acc{0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0};

        for (int t = 0; t < nt; ++t) {
            const int jbase = (t0 + t) * WU_TJ;
            const double2* tp;
            if (PREDICT) {
                // the warp predicts this tile's 64 records itself: lane -> records lane and lane + 32
                tp = ring;
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const int r = lane + 32 * h;
                    double2 rec[Q];
                    nb_predict_record<ORDER>(nb_load_pstate<ORDER>(A.st0, A.st1, A.st2, A.st3, A.st4, A.st5, A.st6, jbase + r), A.t_pred, false, rec);
#pragma unroll
                    for (int q = 0; q < Q; ++q) ring[r * Q + q] = rec[q];
                }
                __syncwarp();
            } else {
                const uint32_t u = uses + t;
                const int st = u & (WU_STAGES - 1);
                mbar_wait(smem_u32(&full[st]), (u / WU_STAGES) & 1);
                tp = ring + (size_t)st * WU_TJ * Q;
            }
            // the self pair (reading R4) lies in one j-tile per particle
            const bool own = (unsigned)(ii - jbase) < (unsigned)WU_TJ;
            const double2* lp = tp + lj * Q;                 // this lane's first record of the tile; a step advances LJ records
            const int jl = jbase + lj;
            if (ORDER == 8) {
                if (__any_sync(0xffffffffu, own)) {
#pragma unroll 1
                    for (int r = 0; r < WU_TJ; r += LJ) pair_o8<EPS0, true>(pi, load_rec<ORDER>(lp + r * Q), A.eps2, jl + r == ii, acc);
                } else {
#pragma unroll 1
                    for (int r = 0; r < WU_TJ; r += LJ) pair_o8<EPS0, false>(pi, load_rec<ORDER>(lp + r * Q), A.eps2, false, acc);
                }
            } else if (__any_sync(0xffffffffu, own)) {
#pragma unroll 1
                for (int r = 0; r < WU_TJ; r += 2 * LJ) {
                    const JRec J[2] = {load_rec<ORDER>(lp + r * Q), load_rec<ORDER>(lp + (r + LJ) * Q)};
                    const bool self[2] = {jl + r == ii, jl + r + LJ == ii};
                    if (ORDER == 4) pair2_o4<EPS0, true>(pi, J, A.eps2, self, acc);
                    else pair2<EPS0, true, NB_PIN_UNSCHEDULED>(pi, J, A.eps2, self, acc);
                }
            } else {
#pragma unroll 1
                for (int r = 0; r < WU_TJ; r += 2 * LJ) {
                    const JRec J[2] = {load_rec<ORDER>(lp + r * Q), load_rec<ORDER>(lp + (r + LJ) * Q)};
                    const bool self[2] = {false, false};
                    if (ORDER == 4) pair2_o4<EPS0, false>(pi, J, A.eps2, self, acc);
                    else pair2<EPS0, false, NB_PIN_UNSCHEDULED>(pi, J, A.eps2, self, acc);
                }
            }
            __syncwarp();                                      // every lane is done with the stage
            if (!PREDICT && lane == 0 && t + WU_STAGES < nt) stage_tile(t0 + t + WU_STAGES, (uses + t) & (WU_STAGES - 1));
        }
        uses += nt;

        // the LJ lane sums of a particle: shuffle butterfly in a fixed order (the "warp-shuffle reduction" of the north star)
        for (int o = LJ >> 1; o > 0; o >>= 1) {
            acc.ax += __shfl_xor_sync(0xffffffffu, acc.ax, o); acc.ay += __shfl_xor_sync(0xffffffffu, acc.ay, o);
            acc.az += __shfl_xor_sync(0xffffffffu, acc.az, o); acc.jx += __shfl_xor_sync(0xffffffffu, acc.jx, o);
            acc.jy += __shfl_xor_sync(0xffffffffu, acc.jy, o); acc.jz += __shfl_xor_sync(0xffffffffu, acc.jz, o);
            acc.p += __shfl_xor_sync(0xffffffffu, acc.p, o);
            if (ORDER != 4) {
                acc.sx += __shfl_xor_sync(0xffffffffu, acc.sx, o); acc.sy += __shfl_xor_sync(0xffffffffu, acc.sy, o);
                acc.sz += __shfl_xor_sync(0xffffffffu, acc.sz, o);
            }
            if (ORDER == 8) {
                acc.cx += __shfl_xor_sync(0xffffffffu, acc.cx, o); acc.cy += __shfl_xor_sync(0xffffffffu, acc.cy, o);
                acc.cz += __shfl_xor_sync(0xffffffffu, acc.cz, o);
            }
        }
        if (lj == 0 && valid) store_sums<ORDER>(A, slice, k, acc);
    }
    if (queued && lane == 0) queue_retire(A.queue, n_workers);
}

// ---------------------------------------------------------------------------------------------
// kernels: one per shape for nb_force (the host planned the launch), and one that holds both shapes and takes the
// plan from device memory (nb_run_blocks: one force launch per block step whatever the scheduler found)
// ---------------------------------------------------------------------------------------------
extern __shared__ __align__(128) double2 dyn_smem[];

// Register ballast.  sass_sched.py re-allocates the temporaries of the pair loops for the source order, which keeps a few more
// values alive than ptxas's own order; it may use every register up to the kernel's register count, and ptxas sets that
// count to what ITS schedule needs (104-110 of the 128 that four CTAs of 128 threads leave per thread).  This block is never
// executed (n_items is never negative); it needs N doubles at once, so the kernel is compiled with 128 registers.
template <int N>
__device__ __forceinline__ void reg_ballast(const ForceArgs& A)
{
    if (A.n_items >= 0) return;
    double x[N], f = 0.0, g = 0.0;
#pragma unroll
    for (int i = 0; i < N; ++i) asm volatile("ld.volatile.global.f64 %0, [%1];" : "=d"(x[i]) : "l"(A.partial + i));
#pragma unroll
    for (int i = 0; i < N; ++i) f = F(x[i], f, x[i]);
#pragma unroll
    for (int i = N - 1; i >= 0; --i) g = F(x[i], g, f);
    A.partial[0] = g;
}

template <bool EPS0, int ORDER>
__global__ void __launch_bounds__(LI_THREADS, LI_CTAS_PER_SM) force_li_kernel(const ForceArgs A)
{
    __shared__ alignas(8) unsigned long long bars[N_BARS];
    reg_ballast<58>(A);
    init_barriers(bars);
    li_body<EPS0, ORDER>(A, dyn_smem, bars);
}

template <bool EPS0>
__global__ void __launch_bounds__(LI_THREADS, LI_CTAS_PER_SM) force_lim_kernel(const ForceArgs A)
{
    __shared__ alignas(8) unsigned long long bars[N_BARS];
    init_barriers(bars);
    li_mixed_body<EPS0>(A, dyn_smem, bars);
}

template <bool EPS0, int ORDER>
__global__ void __launch_bounds__(WU_THREADS, WU_CTAS_PER_SM) force_wu_kernel(const ForceArgs A)
{
    __shared__ alignas(8) unsigned long long bars[N_BARS];
    if (!NB_PIN_UNSCHEDULED) reg_ballast<58>(A);           // only where sass_sched.py reschedules this kernel too
    init_barriers(bars);
    wu_body<EPS0, ORDER, false>(A, dyn_smem, bars);
}

static_assert(LI_THREADS == WU_THREADS && LI_CTAS_PER_SM == WU_CTAS_PER_SM, "the block-step kernel runs either shape in one launch");

template <bool EPS0, int ORDER>
__global__ void __launch_bounds__(WU_THREADS, WU_CTAS_PER_SM) force_step_kernel(const ForceArgs A_)
{
    __shared__ alignas(8) unsigned long long bars[N_BARS];
    ForceArgs A = A_;
    if (!take_devplan(A)) return;
    const int kernel = A.dp->kernel;
    A.n_tiles = kernel == 0 ? A.n_tiles * (WU_TJ) / LI_TJ : A.n_tiles;      // the host passes Npad / WU_TJ
    // CTAs (warps) beyond the work return before any set-up; with a queue the retire count needs every worker
    if (kernel == 1 && A.n_items <= (int)(gridDim.x * WU_WARPS) && (int)(blockIdx.x * WU_WARPS) >= A.n_items) return;
    init_barriers(bars);
    if (kernel == 0 && ORDER == 6 && A.recm) li_mixed_body<EPS0>(A, dyn_smem, bars);
    else if (kernel == 0) li_body<EPS0, ORDER>(A, dyn_smem, bars);
    else if (A.predict) wu_body<EPS0, ORDER, true>(A, dyn_smem, bars);
    else wu_body<EPS0, ORDER, false>(A, dyn_smem, bars);
}

// ---------------------------------------------------------------------------------------------
// partial-sum reduction (row a3) after nb_force: the fixed-order sum of nb_reduce.h, one pass per RED_THREADS / T particles
// ---------------------------------------------------------------------------------------------
template <int NC>
__global__ void __launch_bounds__(RED_THREADS) reduce_partials_kernel(const ForceArgs A, int T)
{
    __shared__ double sm[NC][RED_THREADS];
    const int R = RED_THREADS / T;
    for (int k0 = blockIdx.x * R; k0 < A.n_act; k0 += gridDim.x * R) {      // uniform over the block
        double r[NC];
        int k;
        if (nb_reduce_pass<NC>(A.partial, A.ld, A.n_split, T, A.n_act, k0, sm, r, &k)) nb_store_totals<NC>(A, k, r);
    }
}

constexpr size_t li_smem(int order) { return (size_t)LI_STAGES * LI_TJ * nb_rec_q(order) * 16; }
constexpr size_t wu_smem(int order) { return (size_t)WU_WARPS * WU_STAGES * WU_TJ * nb_rec_q(order) * 16; }
constexpr size_t step_smem(int order) { return li_smem(order) > wu_smem(order) ? li_smem(order) : wu_smem(order); }

}  // namespace

// kernel instantiation for (eps == 0, order)
#define NB_DISPATCH(CALL)                                               \
    do {                                                                \
        if (order == 4)      { if (eps_is_zero) { CALL(true, 4); } else { CALL(false, 4); } } \
        else if (order == 8) { if (eps_is_zero) { CALL(true, 8); } else { CALL(false, 8); } } \
        else                 { if (eps_is_zero) { CALL(true, 6); } else { CALL(false, 6); } } \
    } while (0)

// dynamic shared memory above 48 KiB has to be allowed per kernel (warp units at the 8th order: 56 KiB), and four CTAs
// of 40-56 KiB per SM need the largest shared-memory carve-out (the default heuristic may leave room for only two)
cudaError_t nb_force_setup()
{
    cudaError_t e = cudaSuccess;
    const bool eps_is_zero_values[2] = {false, true};
    for (int order : {4, 6, 8})
        for (bool eps_is_zero : eps_is_zero_values) {
#define SETUP1(K, BYTES)                                                                                                          \
    if (e == cudaSuccess) e = cudaFuncSetAttribute(K, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(BYTES));                 \
    if (e == cudaSuccess) e = cudaFuncSetAttribute(K, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared)
#define SETUP(E, O)                                                                                                              \
    SETUP1((force_li_kernel<E, O>), li_smem(O)); SETUP1((force_wu_kernel<E, O>), wu_smem(O)); SETUP1((force_step_kernel<E, O>), step_smem(O))
            NB_DISPATCH(SETUP);
#undef SETUP
#undef SETUP1
        }
    return e;
}

cudaError_t nb_launch_force(const nb_plan& plan, const ForceArgs& args, bool eps_is_zero, int order, cudaStream_t st, int* launches)
{
#define LI(E, O)                                                                                         \
    if (O == 6 && args.recm) force_lim_kernel<E><<<plan.grid, LI_THREADS, LI_STAGES * LIM_TILE_BYTES, st>>>(args); \
    else force_li_kernel<E, O><<<plan.grid, LI_THREADS, li_smem(O), st>>>(args)
#define WU(E, O) force_wu_kernel<E, O><<<plan.grid, WU_THREADS, wu_smem(O), st>>>(args)
    if (plan.kernel == 0) NB_DISPATCH(LI);
    else NB_DISPATCH(WU);
#undef LI
#undef WU
    ++*launches;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    if (args.n_split > 1) {
        const int T = nb_reduce_threads(args.n_act, args.n_split);
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
    ForceArgs args = args_;
    args.n_tiles = Npad / WU_TJ;
    const int grid = n_sm * WU_CTAS_PER_SM;
#define STEP(E, O) force_step_kernel<E, O><<<grid, WU_THREADS, step_smem(O), st>>>(args)
    NB_DISPATCH(STEP);
#undef STEP
    *launches += 1;
    return cudaGetLastError();
}

void nb_force_occupancy(int order, int* li, int* wu)
{
    const bool eps_is_zero = false;
#define OCC(E, O)                                                                                                   \
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(li, force_li_kernel<E, O>, LI_THREADS, li_smem(O));                \
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(wu, force_wu_kernel<E, O>, WU_THREADS, wu_smem(O))
    NB_DISPATCH(OCC);
#undef OCC
}
