// nb_internal.h — declarations shared by the translation units of libnb.so (CUDA path only).
// Data layout in HBM:
//   state, 5 arrays of double4 (one 32-B sector each per particle, so gathers by active index use
//   whole sectors and the predictor reads exactly the 160 B it needs):
//     st0 = (x, y, z, m)   st1 = (vx, vy, vz, t)   st2 = (ax, ay, az, jx)
//     st3 = (jy, jz, sx, sy)   st4 = (sz, cx, cy, cz)           + dt[N], tn[N] = t + dt (what the scheduler reads)
//   predicted j-records, ONE array of 80-B records (five double2; seven = 112 B at the 8th order):
//     (xp, yp) (zp, m) (vxp, vyp) (vzp, axp) (ayp, azp) [(jxp, jyp) (jzp, -)]
//   so a j-tile is one contiguous bulk copy, and in shared memory both access patterns of the force kernel are free of
//   bank conflicts: all lanes reading one record (broadcast) and every lane reading its own record (16-B pieces at an
//   80-B / 112-B stride fall into eight different 16-B bank groups per quarter warp).
//   Padded to a multiple of NB_PAD particles with massless records far away (they contribute exactly 0).
//   Mixed precision (nb_config.precision) adds a second record array of 64 B per particle, four 16-B pieces:
//     (x, y) fp64 | z fp64, (m, vx) fp32 | (vy, vz, ax, ay) fp32 | (az, -, -, -) fp32
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "nb.h"

constexpr int NB_PAD = 256;          // particle arrays are padded to a multiple of this
constexpr int REC_Q_MAX = 7;         // double2 per predicted record the workspace is laid out for
__host__ __device__ constexpr int nb_rec_q(int order) { return order == 8 ? 7 : 5; }

// Force kernel shapes (nb.h: nb_plan.kernel).
// 0  "CTA tiles": a CTA of 128 threads owns 128 active particles (one per thread) and streams j-tiles of 128 records
//    through shared memory, double-buffered (one bulk copy per tile, mbarrier); all lanes read the same record.
//    pair2 (nb_force.cu) needs 106 registers as ptxas orders it, up to 126 in source order (sass_sched.py): 16 warps (4 per
//    scheduler) per SM as 4 CTAs, 128 registers each at most; CTA shapes that leave the
//    four schedulers with unequal warp counts (5 x 96, 3 x 160) measured 15-27 % slower.
// 1  "warp units": every WARP is its own worker with a private double-buffered ring of 64-record tiles.  A unit is
//    p = 32, 16, ... 1 active particles; the warp's lanes are split p ways over particles and 32/p ways over the records
//    of a step (p = 32: lanes over i, broadcast reads; p = 1: lanes over j), partial sums of a unit's 32/p lanes per
//    particle are combined by a shuffle butterfly.  n_act is decomposed into full units, so no lane idles (nb_plan.h).
constexpr int LI_THREADS = 128;
constexpr int LI_UNIT = LI_THREADS;          // active particles per i-tile
constexpr int LI_TJ = 128;                   // j-records per smem stage, even
constexpr int LI_STAGES = 2;
constexpr int LI_CTAS_PER_SM = 4;
constexpr int WU_THREADS = 128;
constexpr int WU_WARPS = WU_THREADS / 32;
constexpr int WU_CTAS_PER_SM = 4;
constexpr int WU_TJ = 64;                    // j-records per stage of a warp's ring
constexpr int WU_STAGES = 2;
constexpr int RED_THREADS = 256;             // threads per block of the partial-sum reduction
// partial sums are laid out [c][k][s] when a whole reduction block works on one particle (T = RED_THREADS), else [s][c][k]
__host__ __device__ constexpr bool nb_slice_minor(int T) { return T == RED_THREADS; }
constexpr int NB_STEP_LOG = 8192;            // block steps the device-side step log of nb_run_blocks remembers

struct DevPlan;   // nb_plan.h

struct ForceArgs {
    const double2* rec;      // predicted records (padded), nb_rec_q(order) double2 each
    const double4 *st0, *st1, *st2, *st3, *st4, *st5, *st6;   // state: read when the kernel predicts the records itself
    const float4* recm;      // mixed-precision records (64 B: x, y, z fp64; m, vx, vy, vz, ax, ay, az fp32), or nullptr
    const int32_t* idx;      // active indices or nullptr (i = k)
    int n_act;
    int n_units;             // i-tiles (kernel 0) or warp units (kernel 1)
    int n_split;             // S: j-slices per unit = partial planes per particle (1: results are written directly)
    int slice_tiles;         // j-tiles per slice
    int n_tiles;             // total j-tiles (Npad / tile)
    int n_items;             // n_units * n_split
    int ld;                  // rows of a partial plane
    int slice_minor;         // layout of the partial sums (nb_reduce.h: PartialLayout, nb_slice_minor)
    int predict;             // 1: the kernel predicts every j-record it reads from the state, to time t_pred (device-planned
                             //    block steps with few units: saves the predictor's pass over all N)
    double t_pred;
    double eps2;
    double* partial;         // S x NC x ld partial sums when S > 1; NC = 10 components (a, jerk, snap, pot), 13 at the 8th order
    const DevPlan* dp;       // non-null: the launch was planned on the device (nb_run_blocks); overrides the plan fields above
    int* queue;              // work queue: [0] next item, [1] finished workers (both 0 between launches)
    double* out_a; double* out_j; double* out_s; double* out_p;   // [n_act][3] x3, [n_act]
    double* out_c;           // crackle [n_act][3] (8th order only)
};

// nb_force.cu
cudaError_t nb_force_setup();   // once per process and device: shared-memory attributes of the kernels
cudaError_t nb_launch_force(const nb_plan& plan, const ForceArgs& args, bool eps_is_zero, int order, cudaStream_t st, int* launches);
// device-planned (nb_run_blocks): ONE launch at the full grid; the kernel takes shape and sizes from the DevPlan
cudaError_t nb_launch_force_devplan(const ForceArgs& args, bool eps_is_zero, int order, int n_sm, int Npad, cudaStream_t st, int* launches);
void nb_force_occupancy(int order, int* li_ctas_per_sm, int* wu_ctas_per_sm);

// nb_step.cu
struct StateArrays {
    double4 *st0, *st1, *st2, *st3, *st4; double* dt; double* tn; double2* rec;
    double4 *st5, *st6;   // 8th order: st5 = (a4x, a4y, a4z, a5x), st6 = (a5y, a5z, -, -), a4 = d4a/dt4, a5 = d5a/dt5
    float4* recm;         // mixed precision (nb_config.precision): 64-B records written beside rec, else nullptr
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
// scheduler (one kernel): scratch = >= 64 KiB + 16 B per 2048 particles; cand = Npad int32 of candidate lists.
// Result: ((double*)scratch)[0] = t_next, ((int64*)scratch)[1] = n_act, `active` = the ordered list.
cudaError_t nb_launch_next_block(const StateArrays& s, int64_t N, int32_t* active, int32_t* cand, void* scratch, cudaStream_t st, int* launches);
// the O(N) / O(n_act) kernels of one device-planned block step (nb_run_blocks): scheduler + plan, predictor (returns at
// once when the plan lets the force kernel predict); partial-sum reduction + corrector in one kernel
cudaError_t nb_launch_devstep_head(const StateArrays& s, int64_t N, int64_t Npad, int n_sm, int32_t* active, int32_t* cand, void* scratch,
                                   DevPlan* dp, cudaStream_t st, int* launches);
cudaError_t nb_launch_devstep_tail(const StateArrays& s, int n_sm, const int32_t* active, const ForceArgs& fargs, DevPlan* dp,
                                   unsigned long long* steplog, double eta, int k_min, int k_max, cudaStream_t st, int* launches);
cudaError_t nb_launch_energy(const StateArrays& s, int64_t N, const double* pot, double* scratch, cudaStream_t st, int* launches);
cudaError_t nb_launch_check_idx(const int32_t* idx, int64_t n, int64_t N, uint32_t* bitmap, uint32_t* flag, bool unique, cudaStream_t st);
