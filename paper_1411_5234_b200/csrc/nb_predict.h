// nb_predict.h — the predictor of one particle (row a1; "estimated using Taylor expansions"; readings R6,
// R21, R22), as ONE device function: predict_kernel (nb_step.cu) calls it for all N, and the force kernel calls it when
// it predicts the j-records of a block step itself (nb_force.cu, ForceArgs.predict).  Same fma chain in both places, so
// the records are bit-identical and nb_run_blocks stays bitwise equal to the separate calls.
#pragma once
#include "nb_internal.h"

// state of particle i as the predictor reads it (160 B; 224 B at the 8th order)
struct PState { double4 p, q, r, u, w, g, h; };

template <int ORDER>
__device__ __forceinline__ PState nb_load_pstate(const double4* st0, const double4* st1, const double4* st2, const double4* st3,
                                                 const double4* st4, const double4* st5, const double4* st6, int64_t i)
{
    PState s;
    s.p = st0[i]; s.q = st1[i]; s.r = st2[i]; s.u = st3[i]; s.w = st4[i];
    if (ORDER == 8) { s.g = st5[i]; s.h = st6[i]; }
    return s;
}

// D = t - t_i (0 if own_time).  6th order: x to the crackle term, v one order less, a two less.  Record layout: nb_internal.h.
template <int ORDER>
__device__ __forceinline__ void nb_predict_record(const PState& s, double t, bool own_time, double2 (&out)[ORDER == 8 ? 7 : 5])
{
    const double D = own_time ? 0.0 : t - s.q.w;
    const double D2 = D * 0.5, D3 = D * (1.0 / 3.0), D4 = D * 0.25, D5 = D * 0.2;
    const double x[3] = {s.p.x, s.p.y, s.p.z}, v[3] = {s.q.x, s.q.y, s.q.z}, a[3] = {s.r.x, s.r.y, s.r.z};
    const double j[3] = {s.r.w, s.u.x, s.u.y}, sn[3] = {s.u.z, s.u.w, s.w.x}, c[3] = {s.w.y, s.w.z, s.w.w};
    double xp[3], vp[3], ap[3];
    if (ORDER == 8) {                                      // 8th-order variant (R22): two more terms, and the predicted jerk
        const double a4[3] = {s.g.x, s.g.y, s.g.z}, a5[3] = {s.g.w, s.h.x, s.h.y};
        const double D6 = D * (1.0 / 6.0), D7 = D * (1.0 / 7.0);
        double jp[3];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            xp[k] = fma(D, fma(D2, fma(D3, fma(D4, fma(D5, fma(D6, fma(D7, a5[k], a4[k]), c[k]), sn[k]), j[k]), a[k]), v[k]), x[k]);
            vp[k] = fma(D, fma(D2, fma(D3, fma(D4, fma(D5, fma(D6, a5[k], a4[k]), c[k]), sn[k]), j[k]), a[k]), v[k]);
            ap[k] = fma(D, fma(D2, fma(D3, fma(D4, fma(D5, a5[k], a4[k]), c[k]), sn[k]), j[k]), a[k]);
            jp[k] = fma(D, fma(D2, fma(D3, fma(D4, a5[k], a4[k]), c[k]), sn[k]), j[k]);
        }
        out[ORDER == 8 ? 5 : 0] = make_double2(jp[0], jp[1]);
        out[ORDER == 8 ? 6 : 0] = make_double2(jp[2], 0.0);
    } else if (ORDER == 4) {                               // 4th-order variant (R21): x to the jerk term, v to D^2/2 jerk
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            xp[k] = fma(D, fma(D2, fma(D3, j[k], a[k]), v[k]), x[k]);
            vp[k] = fma(D, fma(D2, j[k], a[k]), v[k]);
            ap[k] = 0.0;                                   // a and jerk do not read it
        }
    } else {
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            xp[k] = fma(D, fma(D2, fma(D3, fma(D4, fma(D5, c[k], sn[k]), j[k]), a[k]), v[k]), x[k]);
            vp[k] = fma(D, fma(D2, fma(D3, fma(D4, c[k], sn[k]), j[k]), a[k]), v[k]);
            ap[k] = fma(D, fma(D2, fma(D3, c[k], sn[k]), j[k]), a[k]);
        }
    }
    out[0] = make_double2(xp[0], xp[1]);
    out[1] = make_double2(xp[2], s.p.w);
    out[2] = make_double2(vp[0], vp[1]);
    out[3] = make_double2(vp[2], ap[0]);
    out[4] = make_double2(ap[1], ap[2]);
}
