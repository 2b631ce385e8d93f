// kernel_source_host.cpp — TEST INFRASTRUCTURE (tests/test_kernel_source_cpu.py): the arithmetic of the CUDA sources, compiled
// for the host with g++ so that it can be compared with the oracle where there is no GPU.
//
// What is compiled here is the TEXT of the product's device functions, not a restatement of it: nb_predict.h is included as
// it is; the pair evaluation of nb_force.cu (everything between NB_SCHED_BEGIN and NB_SCHED_END: pair2, pair2_o4, pair_o8),
// pair_mixed, and the corrector with its time-step criterion (nb_step.cu: corrector_one and its helpers) are cut out of the
// .cu files by the test (extracted_*.inc) and included below.  This file supplies only what the GPU supplies: the device
// intrinsics, and the PTX-pinned operations of nb_force.cu (VSUB, VFMA, ...: "one FP64 instruction per line") as the C++
// operation each of them is.  The reciprocal-square-root seed is the exact value cut to 20 bits (MUFU.RSQ64H gives about
// that; the cubic step of the kernel takes it to 2^-60 either way).  Compiled with -ffp-contract=off: the only fused
// operations are the ones the source spells fma().  (nvcc contracts a * b + c in nb_step.cu where g++ here does not: the
// corrector's results differ from the GPU's by rounding, which the comparison's tolerances cover.)
//
// It is NOT a product path: nothing in paper_1411_5234_b200/ refers to it, and it says nothing about the machine code, the
// launch logic, the TMA staging or the reductions - the GPU parity tests do.
#include <cmath>
#include <cstdint>
#include <cstring>

#include <cuda_runtime.h>
#include "nb_internal.h"

static inline int __double2hiint(double x) { int64_t b; std::memcpy(&b, &x, 8); return (int)(b >> 32); }
static inline int __double2loint(double x) { int64_t b; std::memcpy(&b, &x, 8); return (int)(b & 0xffffffff); }
static inline double __hiloint2double(int hi, int lo)
{
    const uint64_t b = ((uint64_t)(uint32_t)hi << 32) | (uint32_t)lo;
    double x; std::memcpy(&x, &b, 8); return x;
}
static inline int __float_as_int(float f) { int b; std::memcpy(&b, &f, 4); return b; }

// ---- nb_force.cu's helpers that are inline PTX there
static inline double F(double a, double b, double c) { return std::fma(a, b, c); }
static inline double M(double a, double b) { return a * b; }
static inline double rsqrt_seed(double s)
{
    const double y = 1.0 / std::sqrt(s);
    int64_t b; std::memcpy(&b, &y, 8);
    b &= ~((int64_t(1) << 32) - 1);                    // keep the high word only: 20 mantissa bits
    double r; std::memcpy(&r, &b, 8); return r;
}
static inline double twice(double c) { return __hiloint2double(__double2hiint(c) + 0x00100000, __double2loint(c)); }
static inline float rsqrt_f32(float s) { return 1.0f / std::sqrt(s); }
#define VSUB(d, a, b) d = (a) - (b)
#define VADD(d, a, b) d = (a) + (b)
#define VMUL(d, a, b) d = (a) * (b)
#define VFMA(d, a, b, c) d = std::fma((a), (b), (c))
#define VFNMA(d, a, b, c) d = std::fma(-(a), (b), (c))
#define VRSQ(d, a) d = rsqrt_seed(a)
#define VTWICE(d, a) d = twice(a)
#undef __device__
#undef __forceinline__
#define __device__
#define __forceinline__ inline

#include "nb_predict.h"                  // the predictor, as it is

namespace {
#include "extracted_force_structs.inc"   // struct Sums, IPart, JRec
#include "extracted_pair_region.inc"     // NB_SCHED_BEGIN .. NB_SCHED_END: pair2, pair2_o4, pair_o8
#include "extracted_pair_mixed.inc"      // struct IPartM, SumsF, JRecM; pair_mixed
#include "extracted_corrector.inc"       // clampi .. norm3, corrector_one
}

// One active particle against all records, as li_body walks them: tiles of `tile` records, two records per call, the masked
// copy of the loop only in the tile that holds the particle itself.  rec: N_even records of Q double2 (nb_internal.h layout).
template <bool EPS0, int ORDER>
static void force_one(const double2* rec, int n_even, int tile, int i, double eps2, Sums& S)
{
    constexpr int Q = ORDER == 8 ? 7 : 5;
    auto load = [&](int j) {
        const double2* r = rec + (size_t)j * Q;
        JRec J{r[0].x, r[0].y, r[1].x, r[1].y, r[2].x, r[2].y, r[3].x, r[3].y, r[4].x, r[4].y, 0.0, 0.0, 0.0};
        if (ORDER == 8) { J.jx = r[5].x; J.jy = r[5].y; J.jz = r[6].x; }
        return J;
    };
    const JRec me = load(i);
    const IPart pi{me.x, me.y, me.z, me.vx, me.vy, me.vz, me.ax, me.ay, me.az, me.jx, me.jy, me.jz};
    for (int jbase = 0; jbase < n_even; jbase += tile) {
        const int jend = jbase + tile < n_even ? jbase + tile : n_even;
        const bool own = i >= jbase && i < jend;
        for (int jj = jbase; jj < jend; jj += 2) {
            if (ORDER == 8) {
                for (int h = 0; h < 2; ++h) {
                    if (own) pair_o8<EPS0, true>(pi, load(jj + h), eps2, jj + h == i, S);
                    else pair_o8<EPS0, false>(pi, load(jj + h), eps2, false, S);
                }
                continue;
            }
            const JRec J[2] = {load(jj), load(jj + 1)};
            const bool self[2] = {own && jj == i, own && jj + 1 == i};
            if (ORDER == 4) { if (own) pair2_o4<EPS0, true>(pi, J, eps2, self, S); else pair2_o4<EPS0, false>(pi, J, eps2, self, S); }
            else if (own) pair2<EPS0, true, true>(pi, J, eps2, self, S);      // PINNED: the copy the warp-unit kernels use
            else pair2<EPS0, false, false>(pi, J, eps2, self, S);             // ... and the one the CTA tiles use
        }
    }
}

extern "C" {

// rec: n_even x Q double2; out: a, j, s, c [n_act][3], pot [n_act] (c only at order 8).  0 = ok.
int host_force(int order, int eps_is_zero, const double* rec, int n_even, int tile, double eps2, const int32_t* idx, int n_act,
               double* oa, double* oj, double* os, double* oc, double* op)
{
    if (n_even % 2 || tile % 2) return -1;
    for (int k = 0; k < n_act; ++k) {
        Sums S{0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
        const double2* r = (const double2*)rec;
        const int i = idx ? idx[k] : k;
        if (order == 6) { if (eps_is_zero) force_one<true, 6>(r, n_even, tile, i, eps2, S); else force_one<false, 6>(r, n_even, tile, i, eps2, S); }
        else if (order == 4) { if (eps_is_zero) force_one<true, 4>(r, n_even, tile, i, eps2, S); else force_one<false, 4>(r, n_even, tile, i, eps2, S); }
        else if (order == 8) { if (eps_is_zero) force_one<true, 8>(r, n_even, tile, i, eps2, S); else force_one<false, 8>(r, n_even, tile, i, eps2, S); }
        else return -1;
        oa[3 * k] = S.ax; oa[3 * k + 1] = S.ay; oa[3 * k + 2] = S.az;
        oj[3 * k] = S.jx; oj[3 * k + 1] = S.jy; oj[3 * k + 2] = S.jz;
        os[3 * k] = S.sx; os[3 * k + 1] = S.sy; os[3 * k + 2] = S.sz;
        if (oc) { oc[3 * k] = S.cx; oc[3 * k + 1] = S.cy; oc[3 * k + 2] = S.cz; }
        op[k] = -S.p;
    }
    return 0;
}

// mixed precision: x fp64, the rest fp32; fp32 sums of `tile` pairs are added into fp64 accumulators (li_mixed_body)
int host_force_mixed(int eps_is_zero, int n, const double* x, const float* m, const float* v, const float* a, int tile, float eps2,
                     const int32_t* idx, int n_act, double* oa, double* oj, double* os, double* op)
{
    for (int k = 0; k < n_act; ++k) {
        const int i = idx ? idx[k] : k;
        const IPartM pi{x[3 * i], x[3 * i + 1], x[3 * i + 2], v[3 * i], v[3 * i + 1], v[3 * i + 2], a[3 * i], a[3 * i + 1], a[3 * i + 2]};
        double acc[10] = {0};
        for (int jbase = 0; jbase < n; jbase += tile) {
            SumsF f{0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
            for (int j = jbase; j < n && j < jbase + tile; ++j) {
                const JRecM J{x[3 * j], x[3 * j + 1], x[3 * j + 2], m[j], v[3 * j], v[3 * j + 1], v[3 * j + 2], a[3 * j], a[3 * j + 1], a[3 * j + 2]};
                if (eps_is_zero) pair_mixed<true, true>(pi, J, eps2, j == i, f);
                else pair_mixed<false, true>(pi, J, eps2, j == i, f);
            }
            const float fs[10] = {f.ax, f.ay, f.az, f.jx, f.jy, f.jz, f.sx, f.sy, f.sz, f.p};
            for (int c = 0; c < 10; ++c) acc[c] += (double)fs[c];
        }
        for (int c = 0; c < 3; ++c) { oa[3 * k + c] = acc[c]; oj[3 * k + c] = acc[3 + c]; os[3 * k + c] = acc[6 + c]; }
        op[k] = -acc[9];
    }
    return 0;
}

// st: 7 arrays of n double4 (nb_internal.h state layout); out: n x Q double2 records
int host_predict(int order, int n, const double* st0, const double* st1, const double* st2, const double* st3, const double* st4,
                 const double* st5, const double* st6, double t, int own_time, double* out)
{
    const double4 *p0 = (const double4*)st0, *p1 = (const double4*)st1, *p2 = (const double4*)st2, *p3 = (const double4*)st3,
                  *p4 = (const double4*)st4, *p5 = (const double4*)st5, *p6 = (const double4*)st6;
    for (int i = 0; i < n; ++i) {
        if (order == 6) { double2 r[5]; nb_predict_record<6>(nb_load_pstate<6>(p0, p1, p2, p3, p4, p5, p6, i), t, own_time != 0, r); std::memcpy(out + (size_t)i * 10, r, sizeof r); }
        else if (order == 4) { double2 r[5]; nb_predict_record<4>(nb_load_pstate<4>(p0, p1, p2, p3, p4, p5, p6, i), t, own_time != 0, r); std::memcpy(out + (size_t)i * 10, r, sizeof r); }
        else if (order == 8) { double2 r[7]; nb_predict_record<8>(nb_load_pstate<8>(p0, p1, p2, p3, p4, p5, p6, i), t, own_time != 0, r); std::memcpy(out + (size_t)i * 14, r, sizeof r); }
        else return -1;
    }
    return 0;
}

// the corrector + criterion on host arrays in the state layout (st0 .. st6, dt, tn are updated in place); eta_p = eta^p as
// nb_launch_corrector passes it (p = 1, 3, 5 at order 4, 6, 8)
int host_correct(int order, double* st0, double* st1, double* st2, double* st3, double* st4, double* st5, double* st6, double* dt,
                 double* tn, const int32_t* idx, int n_act, double dt_shared, double t_new, const double* fa, const double* fj,
                 const double* fs, const double* fc, double eta_p, int k_min, int k_max)
{
    StateArrays s{};
    s.st0 = (double4*)st0; s.st1 = (double4*)st1; s.st2 = (double4*)st2; s.st3 = (double4*)st3; s.st4 = (double4*)st4;
    s.st5 = (double4*)st5; s.st6 = (double4*)st6; s.dt = dt; s.tn = tn; s.fc = fc; s.order = order;
    for (int k = 0; k < n_act; ++k) corrector_one(s, idx, k, dt_shared, t_new, fa, fj, fs, eta_p, k_min, k_max);
    return 0;
}

}  // extern "C"
