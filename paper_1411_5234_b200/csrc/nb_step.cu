// nb_step.cu — the O(N) / O(n_act) steps around the pairwise evaluation (SURVEY.md 8a rows a0, a1,
// a4, a5, a6): predictor, corrector with the time-step criterion, block scheduler, state I/O,
// energy.  All are HBM-bandwidth bound; see DESIGN.md for the bytes per particle of each.
#include "nb_internal.h"
#include "nb_plan.h"
#include "nb_predict.h"
#include "nb_reduce.h"

namespace {

constexpr int TPB = 256;
inline int nblocks(int64_t n, int tpb = TPB) { return (int)((n + tpb - 1) / tpb); }

// massless record far away: contributes exactly 0 to every sum and never overflows
__device__ __forceinline__ void write_pad_record(const StateArrays& s, int64_t i)
{
    double2* r = s.rec + i * nb_rec_q(s.order);
    r[0] = make_double2(3e33, 3e33);
    r[1] = make_double2(3e33, 0.0);
    for (int q = 2; q < nb_rec_q(s.order); ++q) r[q] = make_double2(0.0, 0.0);
    if (s.recm) {
        const double far = 3e33;
        const float lo = __int_as_float(__double2loint(far)), hi = __int_as_float(__double2hiint(far));
        s.recm[4 * i] = make_float4(lo, hi, lo, hi);
        s.recm[4 * i + 1] = make_float4(lo, hi, 0.f, 0.f);
        s.recm[4 * i + 2] = make_float4(0.f, 0.f, 0.f, 0.f);
        s.recm[4 * i + 3] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
}

// ------------------------------------------------------------------ init: AoS inputs -> packed state
__global__ void init_state_kernel(StateArrays s, int64_t N, int64_t Npad, const double* m, const double* x, const double* v)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= Npad) return;
    const double4 zero = make_double4(0, 0, 0, 0);
    if (i < N) {
        s.st0[i] = make_double4(x[3 * i], x[3 * i + 1], x[3 * i + 2], m[i]);
        s.st1[i] = make_double4(v[3 * i], v[3 * i + 1], v[3 * i + 2], 0.0);
        s.dt[i] = 0.0; s.tn[i] = 0.0;
    } else {
        s.st0[i] = make_double4(3e33, 3e33, 3e33, 0.0);
        s.st1[i] = zero;
        s.dt[i] = 1e300; s.tn[i] = 1e300;
        write_pad_record(s, i);
    }
    s.st2[i] = zero; s.st3[i] = zero; s.st4[i] = zero; s.st5[i] = zero; s.st6[i] = zero;
}

// ------------------------------------------------------------------ a1: predictor (reading R6)
// Reads 160 B, writes 80 B per particle (224 B / 112 B at the 8th order).  own_time: D = 0 for every particle (records :=
// stored state).  The arithmetic is nb_predict_record (nb_predict.h), shared with the force kernel.
template <int ORDER>
__global__ void __launch_bounds__(TPB) predict_kernel(StateArrays s, int64_t N, double t, bool own_time, const DevPlan* dp)
{
    if (dp) {                                              // device-planned block step: the time comes from the scheduler
        if (dp->stop || dp->predict) return;               // (predict: the force kernel predicts what it reads)
        t = dp->t_next;
    }
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    constexpr int Q = nb_rec_q(ORDER);
    double2 rec[Q];
    nb_predict_record<ORDER>(nb_load_pstate<ORDER>(s.st0, s.st1, s.st2, s.st3, s.st4, s.st5, s.st6, i), t, own_time, rec);
    double2* out = s.rec + i * Q;
#pragma unroll
    for (int q = 0; q < Q; ++q) out[q] = rec[q];
    if (s.recm) {                                          // mixed precision: fp64 position, fp32 copies of the rest
        float4* om = s.recm + i * 4;
        om[0] = make_float4(__int_as_float(__double2loint(rec[0].x)), __int_as_float(__double2hiint(rec[0].x)),
                            __int_as_float(__double2loint(rec[0].y)), __int_as_float(__double2hiint(rec[0].y)));
        om[1] = make_float4(__int_as_float(__double2loint(rec[1].x)), __int_as_float(__double2hiint(rec[1].x)),
                            (float)rec[1].y, (float)rec[2].x);
        om[2] = make_float4((float)rec[2].y, (float)rec[3].x, (float)rec[3].y, (float)rec[4].x);
        om[3] = make_float4((float)rec[4].y, 0.f, 0.f, 0.f);
    }
}

void launch_predict(const StateArrays& s, int64_t N, double t, bool own_time, const DevPlan* dp, cudaStream_t st)
{
    if (s.order == 8) predict_kernel<8><<<nblocks(N), TPB, 0, st>>>(s, N, t, own_time, dp);
    else if (s.order == 4) predict_kernel<4><<<nblocks(N), TPB, 0, st>>>(s, N, t, own_time, dp);
    else predict_kernel<6><<<nblocks(N), TPB, 0, st>>>(s, N, t, own_time, dp);
}

// ------------------------------------------------------------------ time-step level helpers (a5)
__device__ __forceinline__ int clampi(int k, int lo, int hi) { return k < lo ? lo : (k > hi ? hi : k); }

// floor(log2(r)) for finite r > 0 (subnormals report a value below any admissible level)
__device__ __forceinline__ int ilog2_pos(double r)
{
    const int e = (int)((__double2hiint(r) >> 20) & 0x7ff);
    return e == 0 ? -2000 : e - 1023;
}
__device__ __forceinline__ int floordiv3(int e) { return e >= 0 ? e / 3 : -((-e + 2) / 3); }
__device__ __forceinline__ double norm3(double a, double b, double c) { return sqrt(fma(a, a, fma(b, b, c * c))); }

// ------------------------------------------------------------------ a0: startup (reading R8)
// pass 1: store a, jerk from the first evaluation (snap of that evaluation is discarded).
// pass 2: store a, jerk, snap; crackle = 0 (8th order: the evaluated crackle); dt = eta_s |a|/|jerk| floored to a power of two.
__global__ void startup_kernel(StateArrays s, int64_t N, const double* fa, const double* fj, const double* fs, int pass,
                               double eta_s, int k_min, int k_max)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const double ax = fa[3 * i], ay = fa[3 * i + 1], az = fa[3 * i + 2];
    const double jx = fj[3 * i], jy = fj[3 * i + 1], jz = fj[3 * i + 2];
    if (pass == 1 && s.order != 4) {
        s.st2[i] = make_double4(ax, ay, az, jx);
        s.st3[i] = make_double4(jy, jz, 0.0, 0.0);
        return;
    }
    // 4th-order variant: a and jerk are complete after one evaluation; snap := 0
    const bool o4 = s.order == 4;
    const double sx = o4 ? 0.0 : fs[3 * i], sy = o4 ? 0.0 : fs[3 * i + 1], sz = o4 ? 0.0 : fs[3 * i + 2];
    s.st2[i] = make_double4(ax, ay, az, jx);
    s.st3[i] = make_double4(jy, jz, sx, sy);
    const bool c8 = s.order == 8;                           // 8th order: pass 2's records carry a AND jerk, so it gives crackle too
    s.st4[i] = make_double4(sz, c8 ? s.fc[3 * i] : 0.0, c8 ? s.fc[3 * i + 1] : 0.0, c8 ? s.fc[3 * i + 2] : 0.0);
    const double r = eta_s * norm3(ax, ay, az) / norm3(jx, jy, jz);
    int k;
    if (!(r < INFINITY)) k = k_max;
    else if (!(r > 0.0)) k = k_min;
    else k = clampi(ilog2_pos(r), k_min, k_max);
    s.dt[i] = scalbn(1.0, k); s.tn[i] = s.dt[i];               // t_i = 0
}

// ------------------------------------------------------------------ a4 + a5: corrector (reading R10, R11, R12)
// Per active particle: reads 160 B state + 8 B dt + 72 B new a, jerk, snap; writes 160 B + 8 B.
__device__ __forceinline__ void corrector_one(const StateArrays& s, const int32_t* idx, int64_t k, double dt_shared, double t_new,
                                              const double* fa, const double* fj, const double* fs, double eta3, int k_min, int k_max)
{
    const int64_t i = idx ? (int64_t)idx[k] : k;
    const double4 p = s.st0[i], q = s.st1[i], r = s.st2[i], u = s.st3[i], w = s.st4[i];
    const double dt_old = s.dt[i];
    const double h = dt_shared > 0.0 ? dt_shared : dt_old;
    const double hh = 0.5 * h;
    const double x0[3] = {p.x, p.y, p.z}, v0[3] = {q.x, q.y, q.z};
    const double a0[3] = {r.x, r.y, r.z}, j0[3] = {r.w, u.x, u.y}, s0[3] = {u.z, u.w, w.x};
    if (s.order == 8) {
        // 8th-order variant (R22): septic Hermite quadrature; d4a/dt4 .. d7a/dt7 at the end of the step from the interpolant
        const double c0[3] = {w.y, w.z, w.w};
        double a1[3], j1[3], s1[3], c1[3], x1[3], v1[3], d4[3], d5[3], d6[3], d7[3];
        const double h2 = h * h, h3 = h2 * h, h4 = h3 * h;
        const double ihh = 1.0 / hh, ihh2 = ihh * ihh, ihh4 = ihh2 * ihh2;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            a1[c] = fa[3 * k + c]; j1[c] = fj[3 * k + c]; s1[c] = fs[3 * k + c]; c1[c] = s.fc[3 * k + c];
            v1[c] = v0[c] + hh * (a1[c] + a0[c]) - h2 * (3.0 / 28.0) * (j1[c] - j0[c]) + h3 * (1.0 / 84.0) * (s1[c] + s0[c])
                    - h4 * (1.0 / 1680.0) * (c1[c] - c0[c]);
            x1[c] = x0[c] + hh * (v1[c] + v0[c]) - h2 * (3.0 / 28.0) * (a1[c] - a0[c]) + h3 * (1.0 / 84.0) * (j1[c] + j0[c])
                    - h4 * (1.0 / 1680.0) * (s1[c] - s0[c]);
            const double Am = a1[c] - a0[c];
            const double Jp = hh * (j1[c] + j0[c]), Jm = hh * (j1[c] - j0[c]);
            const double Sp = hh * hh * (s1[c] + s0[c]), Sm = hh * hh * (s1[c] - s0[c]);
            const double Cp = hh * hh * hh * (c1[c] + c0[c]), Cm = hh * hh * hh * (c1[c] - c0[c]);
            d4[c] = (0.5 * (-105.0 * Am + 105.0 * Jp + 15.0 * Jm - 45.0 * Sm - 15.0 * Sp) + 5.0 * Cp + 3.0 * Cm) * ihh4;
            d5[c] = (-315.0 * Am + 315.0 * Jp + 0.5 * (45.0 * Jm - 255.0 * Sm - 45.0 * Sp + 45.0 * Cp + 15.0 * Cm)) * (ihh4 * ihh);
            d6[c] = (0.5 * (-1575.0 * Am + 1575.0 * Jp + 45.0 * Jm - 45.0 * Sp + 105.0 * Cp + 15.0 * Cm) - 315.0 * Sm) * (ihh4 * ihh2);
            d7[c] = (0.5 * (-1575.0 * Am + 1575.0 * Jp + 105.0 * Cp) - 315.0 * Sm) * (ihh4 * ihh2 * ihh);
        }
        s.st0[i] = make_double4(x1[0], x1[1], x1[2], p.w);
        s.st1[i] = make_double4(v1[0], v1[1], v1[2], t_new);
        s.st2[i] = make_double4(a1[0], a1[1], a1[2], j1[0]);
        s.st3[i] = make_double4(j1[1], j1[2], s1[0], s1[1]);
        s.st4[i] = make_double4(s1[2], c1[0], c1[1], c1[2]);
        s.st5[i] = make_double4(d4[0], d4[1], d4[2], d5[0]);
        s.st6[i] = make_double4(d5[1], d5[2], 0.0, 0.0);
        if (dt_shared > 0.0) { s.dt[i] = dt_shared; s.tn[i] = t_new + dt_shared; return; }
        // dt_crit = eta (A1/A6)^(1/5); level = floor(log2 dt_crit) = floor(ilogb(dt_crit^5)/5) (eta3 carries eta^5 for this order)
        const double n0 = norm3(a1[0], a1[1], a1[2]), n1 = norm3(j1[0], j1[1], j1[2]), n2 = norm3(s1[0], s1[1], s1[2]);
        const double n5 = norm3(d5[0], d5[1], d5[2]), n6 = norm3(d6[0], d6[1], d6[2]), n7 = norm3(d7[0], d7[1], d7[2]);
        const double r5 = eta3 * (sqrt(fma(n0, n2, n1 * n1)) / sqrt(fma(n5, n7, n6 * n6)));
        int k_crit;
        if (!(r5 < INFINITY)) k_crit = k_max;
        else if (!(r5 > 0.0)) k_crit = k_min;
        else { const int e5 = ilog2_pos(r5); k_crit = clampi(e5 >= 0 ? e5 / 5 : -((-e5 + 4) / 5), k_min, k_max); }
        const int k_old = ilog2_pos(dt_old);
        int k_new = k_old;
        if (k_crit < k_old) k_new = k_crit;
        else if (k_crit > k_old && k_old < k_max) {
            const double mm = scalbn(t_new, -(k_old + 1));
            if (mm == rint(mm)) k_new = k_old + 1;
        }
        s.dt[i] = scalbn(1.0, k_new); s.tn[i] = t_new + s.dt[i];
        return;
    }
    if (s.order == 4) {
        // 4th-order variant (R21): cubic Hermite quadrature; d2a/dt2 at the end of the step and d3a/dt3 from the interpolant
        double a1[3], j1[3], x1[3], v1[3], d2[3], d3[3];
        const double h2_12 = h * h * (1.0 / 12.0), ih = 1.0 / h, ih2 = ih * ih;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            a1[c] = fa[3 * k + c]; j1[c] = fj[3 * k + c];
            v1[c] = v0[c] + hh * (a1[c] + a0[c]) - h2_12 * (j1[c] - j0[c]);
            x1[c] = x0[c] + hh * (v1[c] + v0[c]) - h2_12 * (a1[c] - a0[c]);
            const double Am = a0[c] - a1[c];
            d2[c] = (6.0 * Am + h * (2.0 * j0[c] + 4.0 * j1[c])) * ih2;
            d3[c] = (12.0 * Am + 6.0 * h * (j0[c] + j1[c])) * (ih2 * ih);
        }
        s.st0[i] = make_double4(x1[0], x1[1], x1[2], p.w);
        s.st1[i] = make_double4(v1[0], v1[1], v1[2], t_new);
        s.st2[i] = make_double4(a1[0], a1[1], a1[2], j1[0]);
        s.st3[i] = make_double4(j1[1], j1[2], d2[0], d2[1]);
        s.st4[i] = make_double4(d2[2], d3[0], d3[1], d3[2]);
        if (dt_shared > 0.0) { s.dt[i] = dt_shared; s.tn[i] = t_new + dt_shared; return; }
        // dt_crit = eta A1/A2 (eta3 carries eta itself for this order)
        const double n0 = norm3(a1[0], a1[1], a1[2]), n1 = norm3(j1[0], j1[1], j1[2]);
        const double n2 = norm3(d2[0], d2[1], d2[2]), n3 = norm3(d3[0], d3[1], d3[2]);
        const double r1 = eta3 * (sqrt(fma(n0, n2, n1 * n1)) / sqrt(fma(n1, n3, n2 * n2)));
        int k_crit;
        if (!(r1 < INFINITY)) k_crit = k_max;
        else if (!(r1 > 0.0)) k_crit = k_min;
        else k_crit = clampi(ilog2_pos(r1), k_min, k_max);
        const int k_old = ilog2_pos(dt_old);
        int k_new = k_old;
        if (k_crit < k_old) k_new = k_crit;
        else if (k_crit > k_old && k_old < k_max) {
            const double mm = scalbn(t_new, -(k_old + 1));
            if (mm == rint(mm)) k_new = k_old + 1;
        }
        s.dt[i] = scalbn(1.0, k_new); s.tn[i] = t_new + s.dt[i];
        return;
    }
    double a1[3], j1[3], s1[3], x1[3], v1[3], d3[3], d4[3], d5[3];
    const double h2_10 = h * h * 0.1, h3_120 = h * h * h * (1.0 / 120.0);
    const double ihh = 1.0 / hh, ihh3 = ihh * ihh * ihh;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        a1[c] = fa[3 * k + c]; j1[c] = fj[3 * k + c]; s1[c] = fs[3 * k + c];
        v1[c] = v0[c] + hh * (a1[c] + a0[c]) - h2_10 * (j1[c] - j0[c]) + h3_120 * (s1[c] + s0[c]);
        x1[c] = x0[c] + hh * (v1[c] + v0[c]) - h2_10 * (a1[c] - a0[c]) + h3_120 * (j1[c] + j0[c]);
        // quintic Hermite interpolant of a(t) about the midpoint, derivatives at the end of the step
        const double Am = a1[c] - a0[c];
        const double Jp = hh * (j1[c] + j0[c]), Jm = hh * (j1[c] - j0[c]);
        const double Sp = hh * hh * (s1[c] + s0[c]), Sm = hh * hh * (s1[c] - s0[c]);
        const double c3 = (-5.0 * Am + 5.0 * Jp - Sm) * 0.125;
        const double c4 = (Sp - Jm) * 0.0625;
        const double c5 = (3.0 * Am - 3.0 * Jp + Sm) * 0.0625;
        d3[c] = 6.0 * (c3 + 4.0 * c4 + 10.0 * c5) * ihh3;
        d4[c] = 24.0 * (c4 + 5.0 * c5) * (ihh3 * ihh);
        d5[c] = 120.0 * c5 * (ihh3 * ihh * ihh);
    }
    s.st0[i] = make_double4(x1[0], x1[1], x1[2], p.w);
    s.st1[i] = make_double4(v1[0], v1[1], v1[2], t_new);
    s.st2[i] = make_double4(a1[0], a1[1], a1[2], j1[0]);
    s.st3[i] = make_double4(j1[1], j1[2], s1[0], s1[1]);
    s.st4[i] = make_double4(s1[2], d3[0], d3[1], d3[2]);

    if (dt_shared > 0.0) { s.dt[i] = dt_shared; s.tn[i] = t_new + dt_shared; return; }

    // dt_crit = eta (A1/A4)^(1/3); level = floor(log2 dt_crit) = floor(ilogb(dt_crit^3) / 3), no cube root needed
    const double n0 = norm3(a1[0], a1[1], a1[2]), n1 = norm3(j1[0], j1[1], j1[2]), n2 = norm3(s1[0], s1[1], s1[2]);
    const double n3 = norm3(d3[0], d3[1], d3[2]), n4 = norm3(d4[0], d4[1], d4[2]), n5 = norm3(d5[0], d5[1], d5[2]);
    const double A1 = sqrt(fma(n0, n2, n1 * n1)), A4 = sqrt(fma(n3, n5, n4 * n4));
    const double r3 = eta3 * (A1 / A4);
    int k_crit;
    if (!(r3 < INFINITY)) k_crit = k_max;
    else if (!(r3 > 0.0)) k_crit = k_min;
    else k_crit = clampi(floordiv3(ilog2_pos(r3)), k_min, k_max);
    const int k_old = ilog2_pos(dt_old);
    int k_new = k_old;
    if (k_crit < k_old) k_new = k_crit;
    else if (k_crit > k_old && k_old < k_max) {
        const double m = scalbn(t_new, -(k_old + 1));       // exact: t_new / 2^(k_old+1)
        if (m == rint(m)) k_new = k_old + 1;                // grow only on the doubled grid
    }
    s.dt[i] = scalbn(1.0, k_new); s.tn[i] = t_new + s.dt[i];
}

__global__ void __launch_bounds__(TPB) corrector_kernel(StateArrays s, const int32_t* idx, int64_t n_act, double dt_shared,
                                                        double t_new, const double* fa, const double* fj, const double* fs,
                                                        double eta3, int k_min, int k_max)
{
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n_act; k += (int64_t)gridDim.x * blockDim.x)
        corrector_one(s, idx, k, dt_shared, t_new, fa, fj, fs, eta3, k_min, k_max);
}

// Device-planned block step (nb_run_blocks): the partial-sum reduction of row a3 and the corrector in ONE kernel.  The
// sums are those of reduce_partials_kernel (nb_force.cu), both call nb_reduce_pass (nb_reduce.h) - the same order, so the
// same bits - and the thread that holds a particle's total stores it and corrects the particle.  S = 1: the force kernel stored the results itself.
template <int NC>
__global__ void __launch_bounds__(RED_THREADS) reduce_correct_kernel(StateArrays s, const int32_t* idx, ForceArgs A, double eta3,
                                                                     int k_min, int k_max, DevPlan* dp, unsigned long long* steplog)
{
    __shared__ double sm[NC][RED_THREADS];
    if (dp->stop) return;
    const int n_act = dp->n_act, S = dp->n_split, T = dp->red_T, ld = dp->ld;
    const double t_new = dp->t_next;
    if (blockIdx.x == 0 && threadIdx.x == 0) {             // last kernel of the step: book-keeping nobody else reads now
        dp->steps_done += 1; dp->steps_left -= 1; dp->sum_act += n_act; dp->t_last = t_new;
        // step log (nb_step_log): n_act and the device clock, in a ring of NB_STEP_LOG entries after the running count
        unsigned long long now;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(now));
        const unsigned long long pos = steplog[0]++;
        steplog[1 + 2 * (pos % NB_STEP_LOG)] = (unsigned long long)n_act;
        steplog[2 + 2 * (pos % NB_STEP_LOG)] = now;
    }
    if (S <= 1) {
        for (int k = blockIdx.x * blockDim.x + threadIdx.x; k < n_act; k += gridDim.x * blockDim.x)
            corrector_one(s, idx, k, 0.0, t_new, A.out_a, A.out_j, A.out_s, eta3, k_min, k_max);
        return;
    }
    const int R = RED_THREADS / T;                         // active particles per block and pass
    for (int k0 = blockIdx.x * R; k0 < n_act; k0 += gridDim.x * R) {        // uniform over the block
        double r[NC];
        int k;
        if (!nb_reduce_pass<NC>(A.partial, ld, S, T, n_act, k0, sm, r, &k)) continue;
        nb_store_totals<NC>(A, k, r);
        corrector_one(s, idx, k, 0.0, t_new, A.out_a, A.out_j, A.out_s, eta3, k_min, k_max);   // reads back what this thread stored
    }
}

// ------------------------------------------------------------------ state I/O
__device__ __forceinline__ int field_width(int f) { return (f == NB_M || f == NB_T || f == NB_DT) ? 1 : 3; }

__global__ void get_kernel(StateArrays s, int field, const int32_t* idx, int64_t n, double* out)
{
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    const int64_t i = idx ? (int64_t)idx[k] : k;
    double a = 0, b = 0, c = 0;
    switch (field) {
        case NB_M: a = s.st0[i].w; break;
        case NB_T: a = s.st1[i].w; break;
        case NB_DT: a = s.dt[i]; break;
        case NB_X: { double4 p = s.st0[i]; a = p.x; b = p.y; c = p.z; } break;
        case NB_V: { double4 p = s.st1[i]; a = p.x; b = p.y; c = p.z; } break;
        case NB_A: { double4 p = s.st2[i]; a = p.x; b = p.y; c = p.z; } break;
        case NB_J: { double4 p = s.st2[i], q = s.st3[i]; a = p.w; b = q.x; c = q.y; } break;
        case NB_S: { double4 p = s.st3[i], q = s.st4[i]; a = p.z; b = p.w; c = q.x; } break;
        case NB_C: { double4 p = s.st4[i]; a = p.y; b = p.z; c = p.w; } break;
        case NB_XP: { const double2* r = s.rec + i * nb_rec_q(s.order); a = r[0].x; b = r[0].y; c = r[1].x; } break;
        case NB_VP: { const double2* r = s.rec + i * nb_rec_q(s.order); a = r[2].x; b = r[2].y; c = r[3].x; } break;
        case NB_AP: { const double2* r = s.rec + i * nb_rec_q(s.order); a = r[3].y; b = r[4].x; c = r[4].y; } break;
        case NB_A4: { double4 p = s.st5[i]; a = p.x; b = p.y; c = p.z; } break;
        case NB_A5: { double4 p = s.st5[i], q = s.st6[i]; a = p.w; b = q.x; c = q.y; } break;
        case NB_JP: if (s.order == 8) { const double2* r = s.rec + i * 7; a = r[5].x; b = r[5].y; c = r[6].x; } break;
    }
    if (field_width(field) == 1) out[k] = a;
    else { out[3 * k] = a; out[3 * k + 1] = b; out[3 * k + 2] = c; }
}

__global__ void set_kernel(StateArrays s, int field, const int32_t* idx, int64_t n, const double* in)
{
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    const int64_t i = idx ? (int64_t)idx[k] : k;
    const bool one = field_width(field) == 1;
    const double a = one ? in[k] : in[3 * k], b = one ? 0.0 : in[3 * k + 1], c = one ? 0.0 : in[3 * k + 2];
    switch (field) {
        case NB_M: s.st0[i].w = a; break;
        case NB_T: s.st1[i].w = a; s.tn[i] = a + s.dt[i]; break;
        case NB_DT: s.dt[i] = a; s.tn[i] = s.st1[i].w + a; break;
        case NB_X: s.st0[i].x = a; s.st0[i].y = b; s.st0[i].z = c; break;
        case NB_V: s.st1[i].x = a; s.st1[i].y = b; s.st1[i].z = c; break;
        case NB_A: s.st2[i].x = a; s.st2[i].y = b; s.st2[i].z = c; break;
        case NB_J: s.st2[i].w = a; s.st3[i].x = b; s.st3[i].y = c; break;
        case NB_S: s.st3[i].z = a; s.st3[i].w = b; s.st4[i].x = c; break;
        case NB_C: s.st4[i].y = a; s.st4[i].z = b; s.st4[i].w = c; break;
        case NB_A4: s.st5[i].x = a; s.st5[i].y = b; s.st5[i].z = c; break;
        case NB_A5: s.st5[i].w = a; s.st6[i].x = b; s.st6[i].y = c; break;
    }
}

// ------------------------------------------------------------------ a6: block scheduler, ONE kernel
// t_next = min_i tn_i (tn = t + dt, kept by the corrector) and the list { i : tn_i == t_next } in increasing index order.
// Every block takes 2048 consecutive particles: it finds ITS minimum and compacts the particles that attain it, in order,
// into its own stretch of `cand`.  The block that finishes last (atomic ticket) takes the minimum over the block minima,
// scans the counts of the blocks that attain it and copies their candidate lists, in block order, into the active list;
// in a device-planned block step it then decides whether the step is taken and plans the force launch (nb_plan.h).
// One pass over 8 B per particle instead of three passes over 16 B.
// scratch layout (bytes): [0] double t_next  [8] i64 n_act  [16] u32 blocks-done counter
//                         [64 ...] double bmin[B]; then u32 cnt[B]; then u32 off[B]       (B = blocks)
constexpr int SCHED_TPB = 1024;
constexpr int SCHED_CHUNK = 2 * SCHED_TPB;

// exclusive prefix sum of v over the block's 1024 threads in thread order; *total = the block's sum.  wt: 33 words of smem.
__device__ __forceinline__ unsigned int block_excl_scan(unsigned int v, unsigned int* wt, unsigned int* total)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    unsigned int inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const unsigned int n = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += n; }
    __syncthreads();                                        // wt may still be read from a previous call
    if (lane == 31) wt[warp] = inc;
    __syncthreads();
    if (warp == 0) {
        const unsigned int w = wt[lane];
        unsigned int wi = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const unsigned int n = __shfl_up_sync(0xffffffffu, wi, o); if (lane >= o) wi += n; }
        wt[lane] = wi - w;                                  // exclusive offset of each warp
        if (lane == 31) wt[32] = wi;
    }
    __syncthreads();
    *total = wt[32];
    return wt[warp] + inc - v;
}

__global__ void __launch_bounds__(SCHED_TPB) sched_kernel(StateArrays s, int64_t N, int32_t* cand, int32_t* active, char* scratch,
                                                         DevPlan* dp, int64_t Npad, int n_sm)
{
    __shared__ double red[32];
    __shared__ unsigned int warp_tot[33];
    __shared__ bool last;
    __shared__ double best_c[SCHED_TPB];
    __shared__ int best_s[SCHED_TPB];
    if (dp && dp->stop) return;
    const int B = gridDim.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    double* bmin_arr = (double*)(scratch + 64);
    unsigned int* cnt_arr = (unsigned int*)(bmin_arr + B);
    unsigned int* off_arr = cnt_arr + B;
    unsigned int* done = (unsigned int*)(scratch + 16);

    // ---- this block's minimum and its candidates
    const int64_t i0 = (int64_t)blockIdx.x * SCHED_CHUNK + 2 * tid;
    double v0 = INFINITY, v1 = INFINITY;
    if (i0 + 1 < N) { const double2 t2 = *(const double2*)(s.tn + i0); v0 = t2.x; v1 = t2.y; }
    else if (i0 < N) v0 = s.tn[i0];
    double m = fmin(v0, v1);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmin(m, __shfl_xor_sync(0xffffffffu, m, o));
    if (lane == 0) red[warp] = m;
    __syncthreads();
    m = red[lane];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmin(m, __shfl_xor_sync(0xffffffffu, m, o));
    const double bmin = m;                                  // every thread has it
    const bool f0 = v0 == bmin && i0 < N, f1 = v1 == bmin && i0 + 1 < N;
    const unsigned int c = (unsigned)f0 + (unsigned)f1;
    unsigned int total;
    unsigned int o_ = block_excl_scan(c, warp_tot, &total);   // in thread (= index) order
    int32_t* my = cand + (int64_t)blockIdx.x * SCHED_CHUNK;
    if (f0) my[o_++] = (int32_t)i0;
    if (f1) my[o_] = (int32_t)(i0 + 1);
    if (tid == 0) {
        bmin_arr[blockIdx.x] = bmin; cnt_arr[blockIdx.x] = total;
        __threadfence();
        last = atomicAdd(done, 1u) == (unsigned)(B - 1);
    }
    __syncthreads();
    if (!last) return;
    __threadfence();

    // ---- the last block: global minimum, offsets of the blocks that attain it, ordered copy
    // thread t looks after blocks t * per .. t * per + per - 1 (per = 1 up to 2^21 particles)
    const int per = (B + SCHED_TPB - 1) / SCHED_TPB;
    double g = INFINITY;
    double bm0 = INFINITY;                                  // per == 1: this thread's block, kept in registers
    unsigned int cn0 = 0;
    if (per == 1) {
        if (tid < B) { bm0 = __ldcg(bmin_arr + tid); cn0 = __ldcg(cnt_arr + tid); }
        g = bm0;
    } else {
        for (int b = tid; b < B; b += SCHED_TPB) g = fmin(g, __ldcg(bmin_arr + b));
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) g = fmin(g, __shfl_xor_sync(0xffffffffu, g, o));
    __syncthreads();                                        // red[] is free again
    if (lane == 0) red[warp] = g;
    __syncthreads();
    g = red[lane];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) g = fmin(g, __shfl_xor_sync(0xffffffffu, g, o));
    const double tn = g;
    unsigned int sum = 0;
    if (per == 1) sum = bm0 == tn ? cn0 : 0;
    else
        for (int q = 0; q < per; ++q) {
            const int b = tid * per + q;
            if (b < B && __ldcg(bmin_arr + b) == tn) sum += __ldcg(cnt_arr + b);
        }
    unsigned int n_tot;
    unsigned int run = block_excl_scan(sum, warp_tot, &n_tot);
    const long long n_act = n_tot;
    if (tid == 0) {
        ((double*)scratch)[0] = tn;
        ((long long*)scratch)[1] = n_act;
        *done = 0;
    }
    if (per == 1) {
        // offsets and counts of the blocks that attain the minimum go through shared memory (best_s / best_c are free)
        unsigned int* s_off = (unsigned int*)best_s;
        unsigned int* s_cnt = (unsigned int*)best_c;
        s_off[tid] = run; s_cnt[tid] = sum;                 // sum = 0: nothing to copy
        __syncthreads();
        for (int b = warp; b < B; b += SCHED_TPB / 32) {
            const unsigned int n = s_cnt[b], off = s_off[b];
            const int32_t* src = cand + (int64_t)b * SCHED_CHUNK;
            for (unsigned int i = lane; i < n; i += 32) active[off + i] = __ldcg(src + i);
        }
        __syncthreads();                                    // best_s / best_c are reused by the plan below
    } else {
        for (int q = 0; q < per; ++q) {
            const int b = tid * per + q;
            if (b < B) {
                const bool hit = __ldcg(bmin_arr + b) == tn;
                off_arr[b] = hit ? run : 0xffffffffu;
                if (hit) run += __ldcg(cnt_arr + b);
            }
        }
        __syncthreads();                                    // off_arr (global) written by this block: visible after the barrier
        for (int b = warp; b < B; b += SCHED_TPB / 32) {
            const unsigned int off = __ldcg(off_arr + b);
            if (off == 0xffffffffu) continue;
            const unsigned int n = __ldcg(cnt_arr + b);
            const int32_t* src = cand + (int64_t)b * SCHED_CHUNK;
            for (unsigned int i = lane; i < n; i += 32) active[off + i] = __ldcg(src + i);
        }
    }
    if (!dp) return;
    // device-planned block step (nb_run_blocks): decide whether the step is taken, and plan the force launch for its
    // n_act with the functions the host uses (nb_plan.h); the candidates S are spread over one warp.
    const bool stop = tn > dp->t_end || dp->steps_left <= 0 || n_act <= 0;
    if (stop) {
        if (tid == 0) { dp->stop = 1; dp->n_act = 0; }
        return;
    }
    if (warp != 0) return;
    const PlanShape sh = nb_plan_shape(Npad, n_act, n_sm, dp->max_split);
    double cst;
    long long S = nb_best_split(sh, lane, 32, &cst);          // S = 0: this lane had no candidate (cost 1e300)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const double c2 = __shfl_xor_sync(0xffffffffu, cst, o);
        const long long s2 = __shfl_xor_sync(0xffffffffu, S, o);
        // least cost; on ties the smaller S (as the host's scan)
        if (s2 != 0 && (S == 0 || c2 < cst || (c2 == cst && s2 < S))) { cst = c2; S = s2; }
    }
    if (lane == 0) {
        nb_fill_devplan(dp, sh, S, n_act);
        dp->t_next = tn;
    }
}

// ------------------------------------------------------------------ energy (fixed-order reduction)
__global__ void __launch_bounds__(TPB) energy_partial_kernel(StateArrays s, int64_t N, const double* pot, double* part)
{
    __shared__ double sk[TPB], sw[TPB];
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    double k = 0, w = 0;
    if (i < N) {
        const double4 p = s.st0[i], v = s.st1[i];
        k = 0.5 * p.w * fma(v.x, v.x, fma(v.y, v.y, v.z * v.z));
        w = 0.5 * p.w * pot[i];
    }
    sk[threadIdx.x] = k; sw[threadIdx.x] = w;
    __syncthreads();
    for (int o = TPB / 2; o > 0; o >>= 1) {
        if (threadIdx.x < o) { sk[threadIdx.x] += sk[threadIdx.x + o]; sw[threadIdx.x] += sw[threadIdx.x + o]; }
        __syncthreads();
    }
    if (threadIdx.x == 0) { part[2 * blockIdx.x] = sk[0]; part[2 * blockIdx.x + 1] = sw[0]; }
}

__global__ void __launch_bounds__(TPB) energy_final_kernel(const double* part, int nb, double* out)
{
    __shared__ double sk[TPB], sw[TPB];
    double k = 0, w = 0;
    for (int b = threadIdx.x; b < nb; b += TPB) { k += part[2 * b]; w += part[2 * b + 1]; }
    sk[threadIdx.x] = k; sw[threadIdx.x] = w;
    __syncthreads();
    for (int o = TPB / 2; o > 0; o >>= 1) {
        if (threadIdx.x < o) { sk[threadIdx.x] += sk[threadIdx.x + o]; sw[threadIdx.x] += sw[threadIdx.x + o]; }
        __syncthreads();
    }
    if (threadIdx.x == 0) { out[0] = sk[0]; out[1] = sw[0]; }
}

// ------------------------------------------------------------------ index-list verification (nb_config.check_indices)
// flag bit 0: an index outside [0, N); bit 1: a duplicate (bitmap: one bit per particle, zeroed by the caller).
__global__ void __launch_bounds__(TPB) check_idx_kernel(const int32_t* idx, int64_t n, int64_t N, uint32_t* bitmap, uint32_t* flag, bool unique)
{
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    const int32_t i = idx[k];
    if (i < 0 || (int64_t)i >= N) { atomicOr(flag, 1u); return; }
    if (!unique) return;
    const uint32_t bit = 1u << (i & 31);
    if (atomicOr(bitmap + (i >> 5), bit) & bit) atomicOr(flag, 2u);
}

}  // namespace

cudaError_t nb_launch_check_idx(const int32_t* idx, int64_t n, int64_t N, uint32_t* bitmap, uint32_t* flag, bool unique, cudaStream_t st)
{
    check_idx_kernel<<<nblocks(n), TPB, 0, st>>>(idx, n, N, bitmap, flag, unique);
    return cudaGetLastError();
}

cudaError_t nb_launch_init_state(const StateArrays& s, int64_t N, int64_t Npad, const double* m, const double* x, const double* v, cudaStream_t st)
{
    init_state_kernel<<<nblocks(Npad), TPB, 0, st>>>(s, N, Npad, m, x, v);
    return cudaGetLastError();
}

cudaError_t nb_launch_predict(const StateArrays& s, int64_t N, double t, bool own_time, cudaStream_t st)
{
    launch_predict(s, N, t, own_time, nullptr, st);
    return cudaGetLastError();
}

cudaError_t nb_launch_startup(const StateArrays& s, int64_t N, const double* fa, const double* fj, const double* fs, int pass,
                              double eta_s, int k_min, int k_max, cudaStream_t st)
{
    startup_kernel<<<nblocks(N), TPB, 0, st>>>(s, N, fa, fj, fs, pass, eta_s, k_min, k_max);
    return cudaGetLastError();
}

static double eta_power(int order, double eta) { return order == 4 ? eta : order == 8 ? eta * eta * eta * eta * eta : eta * eta * eta; }

cudaError_t nb_launch_corrector(const StateArrays& s, const int32_t* idx, int64_t n_act, double dt_shared, double t_new,
                                const double* fa, const double* fj, const double* fs, double eta, int k_min, int k_max,
                                cudaStream_t st)
{
    corrector_kernel<<<nblocks(n_act), TPB, 0, st>>>(s, idx, n_act, dt_shared, t_new, fa, fj, fs, eta_power(s.order, eta), k_min, k_max);
    return cudaGetLastError();
}

cudaError_t nb_launch_get(const StateArrays& s, int field, const int32_t* idx, int64_t n, double* out, cudaStream_t st)
{
    get_kernel<<<nblocks(n), TPB, 0, st>>>(s, field, idx, n, out);
    return cudaGetLastError();
}

cudaError_t nb_launch_set(const StateArrays& s, int field, const int32_t* idx, int64_t n, const double* in, cudaStream_t st)
{
    set_kernel<<<nblocks(n), TPB, 0, st>>>(s, field, idx, n, in);
    return cudaGetLastError();
}

cudaError_t nb_launch_next_block(const StateArrays& s, int64_t N, int32_t* active, int32_t* cand, void* scratch, cudaStream_t st, int* launches)
{
    sched_kernel<<<nblocks(N, SCHED_CHUNK), SCHED_TPB, 0, st>>>(s, N, cand, active, (char*)scratch, nullptr, 0, 0);
    *launches += 1;
    return cudaGetLastError();
}

cudaError_t nb_launch_devstep_head(const StateArrays& s, int64_t N, int64_t Npad, int n_sm, int32_t* active, int32_t* cand, void* scratch,
                                   DevPlan* dp, cudaStream_t st, int* launches)
{
    sched_kernel<<<nblocks(N, SCHED_CHUNK), SCHED_TPB, 0, st>>>(s, N, cand, active, (char*)scratch, dp, Npad, n_sm);
    launch_predict(s, N, 0.0, false, dp, st);
    *launches += 2;
    return cudaGetLastError();
}

cudaError_t nb_launch_devstep_tail(const StateArrays& s, int n_sm, const int32_t* active, const ForceArgs& fargs, DevPlan* dp,
                                   unsigned long long* steplog, double eta, int k_min, int k_max, cudaStream_t st, int* launches)
{
    if (s.order == 8) reduce_correct_kernel<13><<<n_sm * 4, RED_THREADS, 0, st>>>(s, active, fargs, eta_power(s.order, eta), k_min, k_max, dp, steplog);
    else reduce_correct_kernel<10><<<n_sm * 4, RED_THREADS, 0, st>>>(s, active, fargs, eta_power(s.order, eta), k_min, k_max, dp, steplog);
    *launches += 1;
    return cudaGetLastError();
}

cudaError_t nb_launch_energy(const StateArrays& s, int64_t N, const double* pot, double* scratch, cudaStream_t st, int* launches)
{
    const int nb = nblocks(N);
    energy_partial_kernel<<<nb, TPB, 0, st>>>(s, N, pot, scratch + 2);
    energy_final_kernel<<<1, TPB, 0, st>>>(scratch + 2, nb, scratch);
    *launches += 2;
    return cudaGetLastError();
}
