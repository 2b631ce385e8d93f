// nb_internal.h — declarations shared by the translation units of libnb.so (CUDA path only).
// Data layout in HBM:
//   state, 5 arrays of double4 (one 32-B sector each per particle, so gathers by active index use
//   whole sectors and the predictor reads exactly the 160 B it needs):
//     st0 = (x, y, z, m)   st1 = (vx, vy, vz, t)   st2 = (ax, ay, az, jx)
//     st3 = (jy, jz, sx, sy)   st4 = (sz, cx, cy, cz)           + dt[N]
//   predicted j-records, 80 B per particle, three contiguous arrays so a j-tile is three bulk copies:
//     pj0 = (xp, yp, zp, m)   pj1 = (vxp, vyp, vzp, axp)   pj2 = (ayp, azp)
//   padded to a multiple of NB_PAD particles with massless records far away (contribute exactly 0).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "nb.h"

constexpr int NB_PAD = 256;          // particle arrays are padded to a multiple of this

// The force kernels keep one active particle per thread (lanes-over-i) or two per warp (lanes-over-j: every j-record
// loaded serves both).  The lanes-over-i kernel evaluates two j-records at a time with a fixed instruction order (pair2,
// nb_force.cu): 114 registers, 16 warps (4 per scheduler) per SM as 4 CTAs of 128 threads; CTA shapes that leave the four
// schedulers with unequal warp counts (5 x 96, 3 x 160) measured 15-27 % slower.
// lanes-over-i kernel: each thread owns one active particle, a CTA streams j-tiles through smem
constexpr int LI_THREADS = 128;
constexpr int LI_I = 1;
constexpr int LI_UNIT = LI_THREADS * LI_I;   // active particles per i-tile
constexpr int LI_TJ = 128;                   // j-records per smem stage (80 B each), even
constexpr int LI_STAGES = 2;
constexpr int LI_CTAS_PER_SM = 4;
constexpr int LI_W = LI_THREADS / 32;        // small active sets: the CTA's warps share 32 particles and split each j-tile
// lanes-over-j kernel: each warp owns LJ_I active particles, lanes take different j
constexpr int LJ_THREADS = 256;
constexpr int LJ_WARPS = LJ_THREADS / 32;
constexpr int LJ_I = 2;
constexpr int LJ_TJ = 32;                    // j-records per warp iteration
constexpr int LJ_CTAS_PER_SM = 2;
constexpr int64_t LJ_MAX_ACT = 16;           // n_act <= this -> lanes-over-j
constexpr int RED_THREADS = 256;             // threads per block of the partial-sum reduction
constexpr int64_t LIW_MAX_ACT = 96;          // n_act <= this -> lanes-over-i with 32-particle units (above, a 128-lane i-tile is >= 75 % full)

struct DevPlan;   // nb_plan.h

struct ForceArgs {
    const double4* pj0; const double4* pj1; const double2* pj2;   // predicted records (padded)
    const double4* pj3;      // predicted jerk (8th order only)
    const int32_t* idx;      // active indices or nullptr (i = k)
    int n_act;
    int n_units;             // i-tiles (LI) or warp i-groups (LJ)
    int n_split;             // S: j-slices per unit
    int n_planes;            // partial planes per unit = S x sub-slices (1: results are written directly)
    int slice_tiles;         // j-tiles per slice
    int n_tiles;             // total j-tiles (Npad / TJ)
    int n_items;             // n_units * n_split
    int ld;                  // rows of the partial buffer per (slice, component) plane
    double eps2;
    double* partial;         // [planes][NC][ld] when planes > 1; NC = 10 components (a, jerk, snap, pot), 13 at the 8th order
    const DevPlan* dp;       // non-null: the launch was planned on the device (nb_run_blocks); overrides the plan fields above
    int* queue;              // work queue: [0] next item, [1] finished CTAs (both 0 between launches)
    double* out_a; double* out_j; double* out_s; double* out_p;   // [n_act][3] x3, [n_act]
    double* out_c;           // crackle [n_act][3] (8th order only)
};

// nb_force.cu
cudaError_t nb_launch_force(const nb_plan& plan, const ForceArgs& args, bool eps_is_zero, int order, cudaStream_t st, int* launches);
// device-planned: all three kernel shapes and the reduction at their largest grids; the ones the plan does not name return at once
cudaError_t nb_launch_force_devplan(const ForceArgs& args, bool eps_is_zero, int order, int n_sm, int Npad, cudaStream_t st, int* launches);
void nb_force_occupancy(int* li_ctas_per_sm, int* lj_ctas_per_sm);

// nb_step.cu
struct StateArrays {
    double4 *st0, *st1, *st2, *st3, *st4; double* dt; double4 *pj0, *pj1; double2* pj2;
    double4 *st5, *st6;   // 8th order: st5 = (a4x, a4y, a4z, a5x), st6 = (a5y, a5z, -, -), a4 = d4a/dt4, a5 = d5a/dt5
    double4* pj3;         // 8th order: predicted jerk (jxp, jyp, jzp, -)
    const double* fc;     // 8th order: crackle of the last evaluation, row k <-> active_idx[k]
    int order;            // 4, 6 or 8
};
cudaError_t nb_launch_init_state(const StateArrays& s, int64_t N, int64_t Npad, const double* m, const double* x, const double* v, cudaStream_t st);
cudaError_t nb_launch_predict(const StateArrays& s, int64_t N, double t, bool own_time, cudaStream_t st);
cudaError_t nb_launch_startup(const StateArrays& s, int64_t N, const double* fa, const double* fj, const double* fs, int pass,
                              double eta_s, int k_min, int k_max, cudaStream_t st);
cudaError_t nb_launch_corrector(const StateArrays& s, const int32_t* idx, int64_t n_act, double dt_shared, double t_new,
                                const double* fa, const double* fj, const double* fs,
                                double eta, int k_min, int k_max, cudaStream_t st);
cudaError_t nb_launch_get(const StateArrays& s, int field, const int32_t* idx, int64_t n, double* out, cudaStream_t st);
cudaError_t nb_launch_set(const StateArrays& s, int field, const int32_t* idx, int64_t n, const double* in, cudaStream_t st);
// scheduler: scratch = >= 64 KiB; result: scratch_out[0] = t_next (double), ((int64*)scratch_out)[1] = n_act
cudaError_t nb_launch_next_block(const StateArrays& s, int64_t N, int32_t* active, void* scratch, cudaStream_t st, int* launches);
// the O(N) / O(n_act) kernels of one device-planned block step (nb_run_blocks): scheduler + plan, predictor; corrector
cudaError_t nb_launch_devstep_head(const StateArrays& s, int64_t N, int64_t Npad, int n_sm, int32_t* active, void* scratch, DevPlan* dp,
                                   cudaStream_t st, int* launches);
cudaError_t nb_launch_devstep_tail(const StateArrays& s, int n_sm, const int32_t* active, void* scratch, DevPlan* dp, const double* fa,
                                   const double* fj, const double* fs, double eta, int k_min, int k_max, cudaStream_t st, int* launches);
cudaError_t nb_launch_energy(const StateArrays& s, int64_t N, const double* pot, double* scratch, cudaStream_t st, int* launches);
cudaError_t nb_launch_check_idx(const int32_t* idx, int64_t n, int64_t N, uint32_t* bitmap, uint32_t* flag, bool unique, cudaStream_t st);
