/*
 * oracle/nb_oracle.c — TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU brute force of the hot path of the direct-summation
 * Hermite-6 block-time-step method of arXiv:1411.5234.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call it.
 * It shares no code, header, table or helper with the CUDA path.
 *
 * What the paper fixes: eq. (1) and the softened pair force eq. (2)
 * (PAPER.md:35-36).  What it names but does not print (Hermite 6th order, PAPER.md:49,57;
 * Taylor-series predictor and block time steps) is taken in the readings
 * listed in DESIGN.md ("Readings"), cited below as R1..R12.
 *
 * Arithmetic type: REAL (default long double = x87 80-bit here) for every floating-point
 * operation of the method; inputs/outputs are fp64.  -DREAL=double gives the all-fp64
 * variant that bench.py times as the CPU baseline.  No blocking, no reordering: the
 * sums run j = 0..N-1 in index order, exactly as eq. (1) is written.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): circular-binary closed form, 50-digit
 * mpmath brute force + differentiation on N = 2, 3, Newton's third law, finite differences
 * along the Taylor trajectory, polynomial exactness of predictor/corrector, Kepler orbit
 * 6th-order convergence, time-step criterion on the circular binary, energy conservation,
 * Plummer mean field; for the 4th- and 8th-order variants (R21, R22) their own polynomial-exactness,
 * Kepler-convergence, criterion and (8th) 50-digit crackle pins.  Unpinned: the VALUES of eta, eta_s
 * (parameters).
 */
#include <math.h>
#include <stdint.h>
#include <stddef.h>

#ifndef REAL
#define REAL long double
#define R_SQRT sqrtl
#define R_CBRT cbrtl
#define R_LOG2 log2l
#define R_FLOOR floorl
#define R_POW powl
#else
#define R_SQRT sqrt
#define R_CBRT cbrt
#define R_LOG2 log2
#define R_FLOOR floor
#define R_POW pow
#endif
typedef REAL real;

/* Size in bytes of the arithmetic type this build computes in (16 = x87 long double). */
int oracle_real_bytes(void) { return (int)sizeof(real); }

/*
 * O1 — pairwise evaluation.  eq. (1) with the softening of eq. (2),
 * G = 1, per unit mass (R2), and its first and second time derivatives (R3):
 *   dx = x_j - x_i, dv = v_j - v_i, da = a_j - a_i   (predicted quantities, R7)
 *   s = dx.dx + eps^2
 *   a_i    = sum_{j != i} m_j dx / s^(3/2)
 *   jerk_i = d/dt a_i  = sum m_j s^(-3/2) (dv - 3 alpha dx),          alpha = (dx.dv)/s
 *   snap_i = d2/dt2 a_i = sum m_j s^(-3/2) (da - 6 alpha (dv - 3 alpha dx) - 3 beta dx),
 *                                                     beta = (dv.dv + dx.da)/s + alpha^2
 *   pot_i  = - sum_{j != i} m_j s^(-1/2)                                             (R5)
 * xp, vp, ap: [N][3] row-major.  idx == NULL means i = k.  Output row k <-> idx[k].
 */
void oracle_force(int64_t N, const double* m, const double* xp, const double* vp, const double* ap,
                  double eps, const int32_t* idx, int64_t n_act,
                  double* acc, double* jerk, double* snap, double* pot)
{
    const real eps2 = (real)eps * (real)eps;
#pragma omp parallel for schedule(dynamic, 8)
    for (int64_t k = 0; k < n_act; ++k) {
        const int64_t i = idx ? (int64_t)idx[k] : k;
        real A[3] = {0, 0, 0}, J[3] = {0, 0, 0}, S[3] = {0, 0, 0}, P = 0;
        for (int64_t j = 0; j < N; ++j) {
            if (j == i) continue;                                 /* j != i, eq. (1) */
            real dx[3], dv[3], da[3];
            for (int c = 0; c < 3; ++c) {
                dx[c] = (real)xp[3 * j + c] - (real)xp[3 * i + c];
                dv[c] = (real)vp[3 * j + c] - (real)vp[3 * i + c];
                da[c] = (real)ap[3 * j + c] - (real)ap[3 * i + c];
            }
            const real s = dx[0] * dx[0] + dx[1] * dx[1] + dx[2] * dx[2] + eps2;
            const real rho2 = 1 / s;
            const real rho = R_SQRT(rho2);
            const real q = (real)m[j] * rho * rho2;               /* m_j s^(-3/2) */
            const real alpha = (dx[0] * dv[0] + dx[1] * dv[1] + dx[2] * dv[2]) * rho2;
            const real beta = (dv[0] * dv[0] + dv[1] * dv[1] + dv[2] * dv[2]
                             + dx[0] * da[0] + dx[1] * da[1] + dx[2] * da[2]) * rho2 + alpha * alpha;
            for (int c = 0; c < 3; ++c) {
                const real Ac = q * dx[c];
                const real Jc = q * dv[c] - 3 * alpha * Ac;
                const real Sc = q * da[c] - 6 * alpha * Jc - 3 * beta * Ac;
                A[c] += Ac; J[c] += Jc; S[c] += Sc;
            }
            P -= (real)m[j] * rho;
        }
        for (int c = 0; c < 3; ++c) {
            if (acc)  acc[3 * k + c]  = (double)A[c];
            if (jerk) jerk[3 * k + c] = (double)J[c];
            if (snap) snap[3 * k + c] = (double)S[c];
        }
        if (pot) pot[k] = (double)P;
    }
}

/*
 * O2 — predictor ("estimated using Taylor expansions"; order per R6):
 * for ALL N particles, D = t - t_i,
 *   x_p = x + D v + D^2/2 a + D^3/6 j + D^4/24 s + D^5/120 c
 *   v_p = v + D a + D^2/2 j + D^3/6 s + D^4/24 c
 *   a_p = a + D j + D^2/2 s + D^3/6 c          (c = third derivative of a, "crackle")
 */
void oracle_predict(int64_t N, double t, const double* ti,
                    const double* x, const double* v, const double* a,
                    const double* j, const double* s, const double* c,
                    double* xp, double* vp, double* ap)
{
    for (int64_t i = 0; i < N; ++i) {
        const real D = (real)t - (real)ti[i];
        const real D2 = D * D, D3 = D2 * D, D4 = D3 * D, D5 = D4 * D;
        for (int k = 0; k < 3; ++k) {
            const int64_t e = 3 * i + k;
            xp[e] = (double)((real)x[e] + D * v[e] + D2 / 2 * a[e] + D3 / 6 * j[e] + D4 / 24 * s[e] + D5 / 120 * c[e]);
            vp[e] = (double)((real)v[e] + D * a[e] + D2 / 2 * j[e] + D3 / 6 * s[e] + D4 / 24 * c[e]);
            ap[e] = (double)((real)a[e] + D * j[e] + D2 / 2 * s[e] + D3 / 6 * c[e]);
        }
    }
}

/*
 * O4 — time-step level.  R11: generalised Aarseth criterion for a 6th-order scheme,
 *   dt_crit = eta (A1/A4)^(1/3),  Ak = sqrt(|a^(k-1)| |a^(k+1)| + |a^(k)|^2),
 * level = floor(log2 dt_crit) clamped to [k_min, k_max] ("forced to be a power of two",
 * PAPER.md:58).  d[0..5] are a, a', a'', a''', a'''', a''''' (3-vectors) at the new time.
 */
static int level_clamp(real dt_crit, int k_min, int k_max)
{
    if (!(dt_crit < (real)INFINITY)) return k_max;          /* A4 == 0 or NaN: largest step */
    if (!(dt_crit > 0)) return k_min;
    real k = R_FLOOR(R_LOG2(dt_crit));
    if (k < k_min) k = k_min;
    if (k > k_max) k = k_max;
    return (int)k;
}

static real norm3(const real* u) { return R_SQRT(u[0] * u[0] + u[1] * u[1] + u[2] * u[2]); }

static int aarseth6_level(real d[6][3], double eta, int k_min, int k_max)
{
    const real n0 = norm3(d[0]), n1 = norm3(d[1]), n2 = norm3(d[2]);
    const real n3 = norm3(d[3]), n4 = norm3(d[4]), n5 = norm3(d[5]);
    const real A1 = R_SQRT(n0 * n2 + n1 * n1);
    const real A4 = R_SQRT(n3 * n5 + n4 * n4);
    return level_clamp((real)eta * R_CBRT(A1 / A4), k_min, k_max);
}

/* Startup step (R11): dt = eta_s |a| / |jerk|, floored to a power of two. */
void oracle_startup_levels(int64_t N, const double* a, const double* j, double eta_s,
                           int k_min, int k_max, double* dt)
{
    for (int64_t i = 0; i < N; ++i) {
        real av[3] = {a[3 * i], a[3 * i + 1], a[3 * i + 2]};
        real jv[3] = {j[3 * i], j[3 * i + 1], j[3 * i + 2]};
        int k = level_clamp((real)eta_s * norm3(av) / norm3(jv), k_min, k_max);
        dt[i] = ldexp(1.0, k);
    }
}

/*
 * O3 — corrector (R10) for the active particles, with h = step length:
 *   v1 = v0 + h/2 (a1 + a0) - h^2/10 (j1 - j0) + h^3/120 (s1 + s0)
 *   x1 = x0 + h/2 (v1 + v0) - h^2/10 (a1 - a0) + h^3/120 (j1 + j0)
 * and the derivatives of the quintic Hermite interpolant of a(t) at the END of the step:
 * with hh = h/2, Am = a1 - a0, Jp = hh (j1 + j0), Jm = hh (j1 - j0), Sp = hh^2 (s1 + s0),
 * Sm = hh^2 (s1 - s0):  c3 = (-5Am + 5Jp - Sm)/8, c4 = (-Jm + Sp)/16, c5 = (3Am - 3Jp + Sm)/16,
 *   a'''(t1) = 6 (c3 + 4 c4 + 10 c5)/hh^3, a''''(t1) = 24 (c4 + 5 c5)/hh^4, a'''''(t1) = 120 c5/hh^5.
 * Stored afterwards (R9): x1, v1, a1, j1, s1 (the values evaluated at the predicted state),
 * c := a'''(t1), t_i := t_new.
 * dt_shared > 0: every active particle steps h = dt_shared and dt_i := dt_shared.
 * dt_shared <= 0: h = dt_i, then the new level by O4 and the block rule R12: shrink freely;
 * grow one level only if t_new is a multiple of the doubled step.
 * a1, j1, s1: [n_act][3], row k <-> idx[k] (idx NULL: i = k).
 */
void oracle_correct(int64_t N, const int32_t* idx, int64_t n_act, double dt_shared, double t_new,
                    const double* a1, const double* j1, const double* s1,
                    double* x, double* v, double* a, double* j, double* s, double* c,
                    double* ti, double* dt, double eta, int k_min, int k_max)
{
    (void)N;
    for (int64_t k = 0; k < n_act; ++k) {
        const int64_t i = idx ? (int64_t)idx[k] : k;
        const real h = dt_shared > 0 ? (real)dt_shared : (real)dt[i];
        const real hh = h / 2;
        real d[6][3];
        for (int q = 0; q < 3; ++q) {
            const int64_t e = 3 * i + q, f = 3 * k + q;
            const real A0 = a[e], J0 = j[e], S0 = s[e], A1 = a1[f], J1 = j1[f], S1 = s1[f];
            const real v0 = v[e], x0 = x[e];
            const real v1 = v0 + h / 2 * (A1 + A0) - h * h / 10 * (J1 - J0) + h * h * h / 120 * (S1 + S0);
            const real x1 = x0 + h / 2 * (v1 + v0) - h * h / 10 * (A1 - A0) + h * h * h / 120 * (J1 + J0);
            const real Am = A1 - A0;
            const real Jp = hh * (J1 + J0), Jm = hh * (J1 - J0);
            const real Sp = hh * hh * (S1 + S0), Sm = hh * hh * (S1 - S0);
            const real c3 = (-5 * Am + 5 * Jp - Sm) / 8;
            const real c4 = (-Jm + Sp) / 16;
            const real c5 = (3 * Am - 3 * Jp + Sm) / 16;
            d[0][q] = A1; d[1][q] = J1; d[2][q] = S1;
            d[3][q] = 6 * (c3 + 4 * c4 + 10 * c5) / (hh * hh * hh);
            d[4][q] = 24 * (c4 + 5 * c5) / (hh * hh * hh * hh);
            d[5][q] = 120 * c5 / (hh * hh * hh * hh * hh);
            x[e] = (double)x1; v[e] = (double)v1;
            a[e] = (double)A1; j[e] = (double)J1; s[e] = (double)S1; c[e] = (double)d[3][q];
        }
        ti[i] = t_new;
        if (dt_shared > 0) {
            dt[i] = dt_shared;
        } else {
            int k_old = (int)lrint(log2(dt[i]));                    /* dt_i is an exact power of two */
            int k_crit = aarseth6_level(d, eta, k_min, k_max);
            int k_new = k_old;
            if (k_crit < k_old) k_new = k_crit;
            else if (k_crit > k_old && k_old < k_max && fmod(t_new, ldexp(1.0, k_old + 1)) == 0.0) k_new = k_old + 1;
            dt[i] = ldexp(1.0, k_new);
        }
    }
}

/* Exposes O4 alone for the pins: level from the six derivatives of one particle. */
int oracle_aarseth6_level(const double* d18, double eta, int k_min, int k_max)
{
    real d[6][3];
    for (int r = 0; r < 6; ++r) for (int q = 0; q < 3; ++q) d[r][q] = d18[3 * r + q];
    return aarseth6_level(d, eta, k_min, k_max);
}

/* The un-quantised criterion dt_crit = eta (A1/A4)^(1/3), for the pins. */
double oracle_aarseth6_dt(const double* d18, double eta)
{
    real d[6][3];
    for (int r = 0; r < 6; ++r) for (int q = 0; q < 3; ++q) d[r][q] = d18[3 * r + q];
    const real n0 = norm3(d[0]), n1 = norm3(d[1]), n2 = norm3(d[2]);
    const real n3 = norm3(d[3]), n4 = norm3(d[4]), n5 = norm3(d[5]);
    return (double)((real)eta * R_CBRT(R_SQRT(n0 * n2 + n1 * n1) / R_SQRT(n3 * n5 + n4 * n4)));
}

/* Same interpolant as O3, returning a''', a'''', a''''' at the end of the step (pins only). */
void oracle_hermite_derivs(double h, const double* a0, const double* j0, const double* s0,
                           const double* a1, const double* j1, const double* s1, double* d345)
{
    const real hh = (real)h / 2;
    for (int q = 0; q < 3; ++q) {
        const real Am = (real)a1[q] - a0[q];
        const real Jp = hh * ((real)j1[q] + j0[q]), Jm = hh * ((real)j1[q] - j0[q]);
        const real Sp = hh * hh * ((real)s1[q] + s0[q]), Sm = hh * hh * ((real)s1[q] - s0[q]);
        const real c3 = (-5 * Am + 5 * Jp - Sm) / 8;
        const real c4 = (-Jm + Sp) / 16;
        const real c5 = (3 * Am - 3 * Jp + Sm) / 16;
        d345[q]     = (double)(6 * (c3 + 4 * c4 + 10 * c5) / (hh * hh * hh));
        d345[3 + q] = (double)(24 * (c4 + 5 * c5) / (hh * hh * hh * hh));
        d345[6 + q] = (double)(120 * c5 / (hh * hh * hh * hh * hh));
    }
}

/*
 * ---- 4th-order variant ("Hermite time integrators (4th, 6th and 8th order)"; formulas: DESIGN.md R21) ----
 * The pairwise evaluation is O1 restricted to a and jerk (neither depends on the predicted accelerations).
 *
 * O2/4 - predictor:  x_p = x + D v + D^2/2 a + D^3/6 j,   v_p = v + D a + D^2/2 j.
 */
void oracle_predict4(int64_t N, double t, const double* ti, const double* x, const double* v,
                     const double* a, const double* j, double* xp, double* vp)
{
    for (int64_t i = 0; i < N; ++i) {
        const real D = (real)t - (real)ti[i];
        const real D2 = D * D, D3 = D2 * D;
        for (int k = 0; k < 3; ++k) {
            const int64_t e = 3 * i + k;
            xp[e] = (double)((real)x[e] + D * v[e] + D2 / 2 * a[e] + D3 / 6 * j[e]);
            vp[e] = (double)((real)v[e] + D * a[e] + D2 / 2 * j[e]);
        }
    }
}

/* O4/4 - generalised Aarseth criterion for a 4th-order scheme: dt_crit = eta A1/A2,
 * Ak = sqrt(|a^(k-1)| |a^(k+1)| + |a^(k)|^2); d[0..3] = a, a', a'', a''' at the new time. */
static real aarseth4_dt(real d[4][3], double eta)
{
    const real n0 = norm3(d[0]), n1 = norm3(d[1]), n2 = norm3(d[2]), n3 = norm3(d[3]);
    return (real)eta * R_SQRT(n0 * n2 + n1 * n1) / R_SQRT(n1 * n3 + n2 * n2);
}

double oracle_aarseth4_dt(const double* d12, double eta)
{
    real d[4][3];
    for (int r = 0; r < 4; ++r) for (int q = 0; q < 3; ++q) d[r][q] = d12[3 * r + q];
    return (double)aarseth4_dt(d, eta);
}

/*
 * O3/4 - corrector: the two-point cubic Hermite quadrature
 *   v1 = v0 + h/2 (a1 + a0) - h^2/12 (j1 - j0),   x1 = x0 + h/2 (v1 + v0) - h^2/12 (a1 - a0)
 * and the cubic Hermite interpolant of a(t) through (a0, j0) and (a1, j1):
 *   d3a/dt3     = (12 (a0 - a1) + 6 h (j0 + j1)) / h^3        (constant over the step)
 *   d2a/dt2(t1) = (6 (a0 - a1) + h (2 j0 + 4 j1)) / h^2
 * Stored afterwards: x1, v1, a1, j1, s := d2a/dt2(t1), c := d3a/dt3, t_i := t_new; dt_i as in O3.
 */
void oracle_correct4(int64_t N, const int32_t* idx, int64_t n_act, double dt_shared, double t_new,
                     const double* a1, const double* j1,
                     double* x, double* v, double* a, double* j, double* s, double* c,
                     double* ti, double* dt, double eta, int k_min, int k_max)
{
    (void)N;
    for (int64_t k = 0; k < n_act; ++k) {
        const int64_t i = idx ? (int64_t)idx[k] : k;
        const real h = dt_shared > 0 ? (real)dt_shared : (real)dt[i];
        real d[4][3];
        for (int q = 0; q < 3; ++q) {
            const int64_t e = 3 * i + q, f = 3 * k + q;
            const real A0 = a[e], J0 = j[e], A1 = a1[f], J1 = j1[f];
            const real v0 = v[e], x0 = x[e];
            const real v1 = v0 + h / 2 * (A1 + A0) - h * h / 12 * (J1 - J0);
            const real x1 = x0 + h / 2 * (v1 + v0) - h * h / 12 * (A1 - A0);
            d[0][q] = A1; d[1][q] = J1;
            d[2][q] = (6 * (A0 - A1) + h * (2 * J0 + 4 * J1)) / (h * h);
            d[3][q] = (12 * (A0 - A1) + 6 * h * (J0 + J1)) / (h * h * h);
            x[e] = (double)x1; v[e] = (double)v1;
            a[e] = (double)A1; j[e] = (double)J1; s[e] = (double)d[2][q]; c[e] = (double)d[3][q];
        }
        ti[i] = t_new;
        if (dt_shared > 0) {
            dt[i] = dt_shared;
        } else {
            int k_old = (int)lrint(log2(dt[i]));
            int k_crit = level_clamp(aarseth4_dt(d, eta), k_min, k_max);
            int k_new = k_old;
            if (k_crit < k_old) k_new = k_crit;
            else if (k_crit > k_old && k_old < k_max && fmod(t_new, ldexp(1.0, k_old + 1)) == 0.0) k_new = k_old + 1;
            dt[i] = ldexp(1.0, k_new);
        }
    }
}

/*
 * ---- 8th-order variant ("Hermite time integrators (4th, 6th and 8th order)"; formulas: DESIGN.md R22) ----
 *
 * O1/8 - pairwise evaluation with the third time derivative ("crackle") added.  With dj = j_j - j_i (predicted
 * jerks), alpha and beta as in O1 and
 *   gamma = (3 dv.da + dx.dj)/s + alpha (3 beta - 4 alpha^2),
 *   u = dv - 3 alpha dx,  w = da - 6 alpha u - 3 beta dx   (jerk and snap terms per unit q = m_j s^(-3/2)),
 *   crackle_i = d3/dt3 a_i = sum q (dj - 9 alpha w - 9 beta u - 3 gamma dx).
 */
void oracle_force8(int64_t N, const double* m, const double* xp, const double* vp, const double* ap, const double* jp,
                   double eps, const int32_t* idx, int64_t n_act,
                   double* acc, double* jerk, double* snap, double* crackle, double* pot)
{
    const real e2 = (real)eps * (real)eps;
#pragma omp parallel for schedule(dynamic, 8)
    for (int64_t k = 0; k < n_act; ++k) {
        const int64_t i = idx ? (int64_t)idx[k] : k;
        real A[3] = {0, 0, 0}, J[3] = {0, 0, 0}, S[3] = {0, 0, 0}, C[3] = {0, 0, 0}, P = 0;
        for (int64_t j = 0; j < N; ++j) {
            if (j == i) continue;
            real dx[3], dv[3], da[3], dj[3];
            for (int q = 0; q < 3; ++q) {
                dx[q] = (real)xp[3 * j + q] - (real)xp[3 * i + q];
                dv[q] = (real)vp[3 * j + q] - (real)vp[3 * i + q];
                da[q] = (real)ap[3 * j + q] - (real)ap[3 * i + q];
                dj[q] = (real)jp[3 * j + q] - (real)jp[3 * i + q];
            }
            const real s = dx[0] * dx[0] + dx[1] * dx[1] + dx[2] * dx[2] + e2;
            const real rho2 = 1 / s, rho = R_SQRT(rho2);
            const real q_ = (real)m[j] * rho * rho2;
            const real xv = dx[0] * dv[0] + dx[1] * dv[1] + dx[2] * dv[2];
            const real vv = dv[0] * dv[0] + dv[1] * dv[1] + dv[2] * dv[2];
            const real xa = dx[0] * da[0] + dx[1] * da[1] + dx[2] * da[2];
            const real va = dv[0] * da[0] + dv[1] * da[1] + dv[2] * da[2];
            const real xj = dx[0] * dj[0] + dx[1] * dj[1] + dx[2] * dj[2];
            const real alpha = xv * rho2;
            const real beta = (vv + xa) * rho2 + alpha * alpha;
            const real gamma = (3 * va + xj) * rho2 + alpha * (3 * beta - 4 * alpha * alpha);
            for (int c = 0; c < 3; ++c) {
                const real u = dv[c] - 3 * alpha * dx[c];
                const real w = da[c] - 6 * alpha * u - 3 * beta * dx[c];
                A[c] += q_ * dx[c];
                J[c] += q_ * u;
                S[c] += q_ * w;
                C[c] += q_ * (dj[c] - 9 * alpha * w - 9 * beta * u - 3 * gamma * dx[c]);
            }
            P -= (real)m[j] * rho;
        }
        for (int c = 0; c < 3; ++c) {
            if (acc) acc[3 * k + c] = (double)A[c];
            if (jerk) jerk[3 * k + c] = (double)J[c];
            if (snap) snap[3 * k + c] = (double)S[c];
            if (crackle) crackle[3 * k + c] = (double)C[c];
        }
        if (pot) pot[k] = (double)P;
    }
}

/*
 * O2/8 - predictor: x_p to D^7/5040 a5, v_p to D^6/720 a5, a_p to D^5/120 a5, j_p to D^4/24 a5, where
 * a4 = d4a/dt4 and a5 = d5a/dt5 come from the previous corrector's interpolant (0 before the first step).
 */
void oracle_predict8(int64_t N, double t, const double* ti, const double* x, const double* v, const double* a,
                     const double* j, const double* s, const double* c, const double* a4, const double* a5,
                     double* xp, double* vp, double* ap, double* jp)
{
    for (int64_t i = 0; i < N; ++i) {
        const real D = (real)t - (real)ti[i];
        const real D2 = D * D, D3 = D2 * D, D4 = D3 * D, D5 = D4 * D, D6 = D5 * D, D7 = D6 * D;
        for (int k = 0; k < 3; ++k) {
            const int64_t e = 3 * i + k;
            xp[e] = (double)((real)x[e] + D * v[e] + D2 / 2 * a[e] + D3 / 6 * j[e] + D4 / 24 * s[e] + D5 / 120 * c[e]
                             + D6 / 720 * a4[e] + D7 / 5040 * a5[e]);
            vp[e] = (double)((real)v[e] + D * a[e] + D2 / 2 * j[e] + D3 / 6 * s[e] + D4 / 24 * c[e] + D5 / 120 * a4[e]
                             + D6 / 720 * a5[e]);
            ap[e] = (double)((real)a[e] + D * j[e] + D2 / 2 * s[e] + D3 / 6 * c[e] + D4 / 24 * a4[e] + D5 / 120 * a5[e]);
            jp[e] = (double)((real)j[e] + D * s[e] + D2 / 2 * c[e] + D3 / 6 * a4[e] + D4 / 24 * a5[e]);
        }
    }
}

/*
 * The septic Hermite interpolant of a(t) through (a, j, s, c) at both ends of a step of length h, about the mid-point in
 * tau = (t - t_mid)/hh, hh = h/2.  With Am = a1 - a0, Jp = hh (j1 + j0), Jm = hh (j1 - j0), Sp = hh^2 (s1 + s0),
 * Sm = hh^2 (s1 - s0), Cp = hh^3 (c1 + c0), Cm = hh^3 (c1 - c0), its derivatives at the END of the step are
 *   hh^4 a4 = (-105 Am + 105 Jp + 15 Jm - 45 Sm - 15 Sp)/2 + 5 Cp + 3 Cm
 *   hh^5 a5 = -315 Am + 315 Jp + (45 Jm - 255 Sm - 45 Sp + 45 Cp + 15 Cm)/2
 *   hh^6 a6 = (-1575 Am + 1575 Jp + 45 Jm - 45 Sp + 105 Cp + 15 Cm)/2 - 315 Sm
 *   hh^7 a7 = (-1575 Am + 1575 Jp + 105 Cp)/2 - 315 Sm
 * (solved from the eight end-point conditions; checked by the polynomial-exactness pin).
 */
static void hermite8_end_derivs(real hh, real A0, real J0, real S0, real C0, real A1, real J1, real S1, real C1, real out[4])
{
    const real Am = A1 - A0;
    const real Jp = hh * (J1 + J0), Jm = hh * (J1 - J0);
    const real Sp = hh * hh * (S1 + S0), Sm = hh * hh * (S1 - S0);
    const real Cp = hh * hh * hh * (C1 + C0), Cm = hh * hh * hh * (C1 - C0);
    const real h4 = hh * hh * hh * hh;
    out[0] = ((-105 * Am + 105 * Jp + 15 * Jm - 45 * Sm - 15 * Sp) / 2 + 5 * Cp + 3 * Cm) / h4;
    out[1] = (-315 * Am + 315 * Jp + (45 * Jm - 255 * Sm - 45 * Sp + 45 * Cp + 15 * Cm) / 2) / (h4 * hh);
    out[2] = ((-1575 * Am + 1575 * Jp + 45 * Jm - 45 * Sp + 105 * Cp + 15 * Cm) / 2 - 315 * Sm) / (h4 * hh * hh);
    out[3] = ((-1575 * Am + 1575 * Jp + 105 * Cp) / 2 - 315 * Sm) / (h4 * hh * hh * hh);
}

void oracle_hermite8_derivs(double h, const double* a0, const double* j0, const double* s0, const double* c0,
                            const double* a1, const double* j1, const double* s1, const double* c1, double* d4567)
{
    for (int q = 0; q < 3; ++q) {
        real o[4];
        hermite8_end_derivs((real)h / 2, a0[q], j0[q], s0[q], c0[q], a1[q], j1[q], s1[q], c1[q], o);
        for (int r = 0; r < 4; ++r) d4567[3 * r + q] = (double)o[r];
    }
}

/* O4/8 - generalised Aarseth criterion for an 8th-order scheme: dt_crit = eta (A1/A6)^(1/5);
 * d[0..7] = a, a', ..., a^(7) at the new time. */
static real aarseth8_dt(real d[8][3], double eta)
{
    const real n0 = norm3(d[0]), n1 = norm3(d[1]), n2 = norm3(d[2]);
    const real n5 = norm3(d[5]), n6 = norm3(d[6]), n7 = norm3(d[7]);
    const real r = R_SQRT(n0 * n2 + n1 * n1) / R_SQRT(n5 * n7 + n6 * n6);
    return (real)eta * R_POW(r, (real)1 / 5);
}

double oracle_aarseth8_dt(const double* d24, double eta)
{
    real d[8][3];
    for (int r = 0; r < 8; ++r) for (int q = 0; q < 3; ++q) d[r][q] = d24[3 * r + q];
    return (double)aarseth8_dt(d, eta);
}

/*
 * O3/8 - corrector: the two-point septic Hermite quadrature
 *   v1 = v0 + h/2 (a1 + a0) - 3 h^2/28 (j1 - j0) + h^3/84 (s1 + s0) - h^4/1680 (c1 - c0)
 *   x1 = x0 + h/2 (v1 + v0) - 3 h^2/28 (a1 - a0) + h^3/84 (j1 + j0) - h^4/1680 (s1 - s0)
 * Stored afterwards: x1, v1, a1, j1, s1, c1 (evaluated at the predicted state), a4, a5 := the interpolant's at t1.
 */
void oracle_correct8(int64_t N, const int32_t* idx, int64_t n_act, double dt_shared, double t_new,
                     const double* a1, const double* j1, const double* s1, const double* c1,
                     double* x, double* v, double* a, double* j, double* s, double* c, double* a4, double* a5,
                     double* ti, double* dt, double eta, int k_min, int k_max)
{
    (void)N;
    for (int64_t k = 0; k < n_act; ++k) {
        const int64_t i = idx ? (int64_t)idx[k] : k;
        const real h = dt_shared > 0 ? (real)dt_shared : (real)dt[i];
        real d[8][3];
        for (int q = 0; q < 3; ++q) {
            const int64_t e = 3 * i + q, f = 3 * k + q;
            const real A0 = a[e], J0 = j[e], S0 = s[e], C0 = c[e], A1 = a1[f], J1 = j1[f], S1 = s1[f], C1 = c1[f];
            const real v0 = v[e], x0 = x[e];
            const real h2 = h * h, h3 = h2 * h, h4 = h3 * h;
            const real v1 = v0 + h / 2 * (A1 + A0) - 3 * h2 / 28 * (J1 - J0) + h3 / 84 * (S1 + S0) - h4 / 1680 * (C1 - C0);
            const real x1 = x0 + h / 2 * (v1 + v0) - 3 * h2 / 28 * (A1 - A0) + h3 / 84 * (J1 + J0) - h4 / 1680 * (S1 - S0);
            real o[4];
            hermite8_end_derivs(h / 2, A0, J0, S0, C0, A1, J1, S1, C1, o);
            d[0][q] = A1; d[1][q] = J1; d[2][q] = S1; d[3][q] = C1;
            d[4][q] = o[0]; d[5][q] = o[1]; d[6][q] = o[2]; d[7][q] = o[3];
            x[e] = (double)x1; v[e] = (double)v1;
            a[e] = (double)A1; j[e] = (double)J1; s[e] = (double)S1; c[e] = (double)C1;
            a4[e] = (double)o[0]; a5[e] = (double)o[1];
        }
        ti[i] = t_new;
        if (dt_shared > 0) {
            dt[i] = dt_shared;
        } else {
            int k_old = (int)lrint(log2(dt[i]));
            int k_crit = level_clamp(aarseth8_dt(d, eta), k_min, k_max);
            int k_new = k_old;
            if (k_crit < k_old) k_new = k_crit;
            else if (k_crit > k_old && k_old < k_max && fmod(t_new, ldexp(1.0, k_old + 1)) == 0.0) k_new = k_old + 1;
            dt[i] = ldexp(1.0, k_new);
        }
    }
}

/*
 * O6 — block scheduler ("blocks that share the same time step"):
 * t_next = min_i (t_i + dt_i); active = { i : t_i + dt_i == t_next } in index order.
 * All times are dyadic rationals, so the fp64 sums and the equality are exact.
 */
int64_t oracle_next_block(int64_t N, const double* ti, const double* dt, double* t_next, int32_t* active)
{
    double tn = INFINITY;
    for (int64_t i = 0; i < N; ++i) { double u = ti[i] + dt[i]; if (u < tn) tn = u; }
    int64_t n = 0;
    for (int64_t i = 0; i < N; ++i) if (ti[i] + dt[i] == tn) active[n++] = (int32_t)i;
    *t_next = tn;
    return n;
}

/* O7 — energy: E = 1/2 sum m |v|^2 + 1/2 sum m pot  (pot from O1 at the same instant). */
void oracle_energy(int64_t N, const double* m, const double* v, const double* pot,
                   double* kinetic, double* potential)
{
    real K = 0, W = 0;
    for (int64_t i = 0; i < N; ++i) {
        const real v2 = (real)v[3 * i] * v[3 * i] + (real)v[3 * i + 1] * v[3 * i + 1] + (real)v[3 * i + 2] * v[3 * i + 2];
        K += (real)m[i] * v2 / 2;
        W += (real)m[i] * pot[i] / 2;
    }
    *kinetic = (double)K; *potential = (double)W;
}
