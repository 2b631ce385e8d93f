/*
 * nb.h — C ABI of libnb.so: the data-parallel hot path of the direct-summation Hermite-6
 * block-time-step N-body method of arXiv:1411.5234 (Spera 2014, "HiGPUs" as template),
 * implemented as hand-written CUDA for NVIDIA B200 (sm_100a).  One GPU per context.
 *
 * The method (citations are PAPER.md lines):
 *   eq. (1)  r''_i = -G sum_{j != i} m_j r_ij / r_ij^3
 *   eq. (2)  softened pair force  F = -G m_i m_j r_ij / (r_ij^2 + eps^2)^(3/2)
 *   Hermite 6th-order integrator: Taylor-series predictor for all N, one pairwise evaluation
 *   per step, corrector for the active particles
 *   Block time steps: power-of-two steps, m <= N active particles per step,
 *   cost O(mN) per step
 * G = 1.  Everything the paper names without printing is fixed in DESIGN.md ("Readings").
 *
 * Conventions common to all calls
 *   - fp64 throughout; indices are int32; sizes are int64.
 *   - Vector arguments x, v, a, jerk, snap are row-major [n][3]; m, pot, t, dt are [n].
 *   - Every pointer argument marked "(h/d)" is a HOST pointer if cfg->ptrs_on_device == 0 and a
 *     DEVICE pointer (on cfg->device) if cfg->ptrs_on_device == 1.  The caller owns every buffer it
 *     passes; the library neither frees nor retains them after the call returns, EXCEPT the
 *     workspace, which the context uses until nb_free.
 *   - All device memory lives in the caller-provided workspace (PyTorch is the allocator).
 *   - Work is enqueued on cfg->stream.  With host pointers a call returns after its outputs have
 *     arrived (it synchronises the stream); with device pointers calls are asynchronous.
 *   - Return value: NB_OK (0) or a negative nb_status.  No exceptions, no exit(), nothing is
 *     printed.  A context is not thread-safe.
 */
#ifndef NB_H
#define NB_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct nb_ctx nb_ctx; /* opaque: one particle system on one GPU */

typedef enum {
    NB_OK = 0,
    NB_EINVAL = -1, /* bad argument: N < 1, eps < 0, NULL where not allowed, n_act out of range, bad level range; with index
                       checking on (nb_config.check_indices): an index outside [0, N) or a duplicate in an index list */
    NB_ENOMEM = -2, /* workspace missing, misaligned (< 256 B) or smaller than nb_workspace_bytes(N) */
    NB_ESTATE = -3, /* call order: nb_force without nb_predict since the last state change, nb_corrector without nb_force */
    NB_ECUDA = -4   /* a CUDA runtime call or kernel failed; nb_last_error(ctx) holds the CUDA message */
} nb_status;

typedef struct {
    int device;             /* CUDA device ordinal */
    void* stream;           /* cudaStream_t to enqueue on; NULL = the legacy default stream */
    void* workspace;        /* DEVICE memory, 256-B aligned, >= nb_workspace_bytes(N) bytes, owned by the caller */
    size_t workspace_bytes;
    int ptrs_on_device;     /* 0: (h/d) pointers are host pointers; 1: device pointers */
    double eta;             /* accuracy parameter of the time-step criterion (reading R11); 0 -> 0.45 (order 6), 0.14 (order 4) */
    double eta_s;           /* same, for the startup step dt = eta_s |a|/|jerk|;             0 -> 0.01 */
    int k_min, k_max;       /* allowed levels: dt = 2^k, k_min <= k <= k_max; both 0 -> -20, -3 */
    int order;              /* Hermite order ("4th, 6th and 8th order"): 0 or 6 = the 6th-order scheme of the
                               north star; 4 = the 4th-order variant (reading R21): nb_force evaluates a, jerk and pot (snap
                               is returned as 0), the predictor stops at the jerk term, nb_corrector is the cubic Hermite
                               quadrature and the criterion dt = eta A1/A2;
                               8 = the 8th-order variant (reading R22): nb_force also evaluates crackle = d3a/dt3 (read it with
                               nb_force_crackle), the predictor runs to d5a/dt5 and predicts the jerk, nb_corrector is the
                               septic Hermite quadrature, criterion dt = eta (A1/A6)^(1/5), eta -> 0.75, two startup passes. */
    int check_indices;      /* index lists passed to nb_force / nb_corrector / nb_get_state / nb_set_state (the
                               m <= N active particles) are verified on the device before use: every index in [0, N), and no
                               duplicates (nb_get_state allows duplicates).  A bad list returns NB_EINVAL and nothing is
                               launched on it.  The check reads one flag back, so it synchronises the stream.
                               0 = default: on for host-pointer contexts (those calls synchronise anyway), off for
                               device-pointer contexts (calls stay asynchronous; indices are then the caller's contract);
                               1 = always on; -1 = always off. */
    int precision;          /* nb_precision: 0 = NB_PREC_FP64 (default: everything fp64, the north star's 1e-11);
                               1 = NB_PREC_MIXED, the throughput mode of the paper's template ("DP ... to
                               calculate reciprocal distances and to cumulate accelerations", SP elsewhere): position
                               differences in fp64, the rest of the pair in fp32, fp32 sums flushed into fp64 accumulators
                               every 128 j-particles.  Applies to 6th-order evaluations that run as CTA tiles (nb_plan.kernel
                               == 0: large active sets); smaller active sets and all O(N) steps stay fp64.  Accuracy about
                               1e-6 per particle (measured against the oracle: DESIGN.md 11), so the time-step criterion and
                               the energy error are those of a single-precision force.  NB_EINVAL with order 4 or 8. */
} nb_config;

typedef enum { NB_PREC_FP64 = 0, NB_PREC_MIXED = 1 } nb_precision;

/* Selectors of nb_get_state / nb_set_state.  Width = doubles per particle. */
typedef enum {
    NB_M = 0,   /* mass, 1 */
    NB_X = 1,   /* position at t_i, 3 */
    NB_V = 2,   /* velocity at t_i, 3 */
    NB_A = 3,   /* acceleration at t_i, 3 */
    NB_J = 4,   /* jerk  (da/dt), 3 */
    NB_S = 5,   /* snap  (d2a/dt2), 3 */
    NB_C = 6,   /* crackle (d3a/dt3, from the corrector's interpolant; 0 before the first step), 3 */
    NB_T = 7,   /* particle time t_i, 1 */
    NB_DT = 8,  /* particle step dt_i (a power of two), 1 */
    NB_XP = 9,  /* predicted position at the time of the last nb_predict, 3 (get only) */
    NB_VP = 10, /* predicted velocity, 3 (get only) */
    NB_AP = 11, /* predicted acceleration, 3 (get only) */
    NB_A4 = 12, /* d4a/dt4 from the corrector's interpolant, 3 (8th order only) */
    NB_A5 = 13, /* d5a/dt5, 3 (8th order only) */
    NB_JP = 14  /* predicted jerk, 3 (get only; 8th order only) */
} nb_field;

/* How nb_force maps an evaluation onto the GPU (reading R15; "Bfactor"). */
typedef struct {
    int kernel;       /* 0 = CTA tiles: a CTA of 128 threads owns 128 active particles, j-tiles broadcast from shared memory
                         1 = warp units: every warp owns a unit of p = 32, 16, ... 1 active particles and streams its own
                             j-slice; its lanes are split p ways over particles and 32/p ways over j-records (p = 32:
                             lanes over i; p = 1: lanes over j).  n_act = 32 a + r is decomposed into a units of 32 and
                             the binary digits of r, so no lane idles */
    int n_units;      /* i-tiles (kernel 0) or warp units (kernel 1) */
    int n_split;      /* S: number of j-slices each unit is split into ("Bfactor") = partial sums per particle */
    int slice_tiles;  /* j-tiles per slice (the last slice may hold fewer) */
    int grid;         /* CTAs launched */
    int unit;         /* active particles per full unit (kernel 0: 128; kernel 1: 32) */
    int tile;         /* j-records per j-tile (kernel 0: one shared-memory stage of the CTA, 128; kernel 1: of a warp, 64) */
    int ctas_per_sm;  /* resident CTAs per multiprocessor the plan assumes */
    int predict_in_force; /* 1: in a device-planned block step (nb_run_blocks) with this n_act the force kernel predicts the
                         j-records it reads from the state itself and the predictor's pass over all N is skipped */
    double waves;     /* work items / resident workers (CTAs or warps) on the device */
} nb_plan;

/* Bytes of device workspace a context for N particles needs.  Pure; 0 if N < 1. */
size_t nb_workspace_bytes(int64_t N);

/* Pure host logic: the launch plan nb_force would use for n_act active particles out of N on a device
 * with n_sm multiprocessors.  NB_EINVAL on bad sizes. */
int nb_plan_force(int64_t N, int64_t n_act, int n_sm, nb_plan* plan);

/* Cap the j-split S of this context's nb_force / nb_run_blocks launches: 0 (default) = the cost model decides,
 * 1 = no split (the "Bfactor off" arm of the paper's Fig. 1), k = at most k slices. */
int nb_set_max_split(nb_ctx* ctx, int64_t max_split);

/*
 * nb_init — create a system from the initial conditions of eq. (1): masses m[N],
 * positions x[N][3], velocities v[N][3] (h/d), softening eps >= 0 of eq. (2).
 * Copies the inputs, sets t_i = 0 and performs the startup (reading R8): one evaluation with a_j = 0
 * to get a and jerk, a second with those a to get snap; crackle = 0; dt_i = eta_s |a|/|jerk| floored
 * to a power of two in [2^k_min, 2^k_max].  eps = 0 is legal (eq. 1): coincident particles then give
 * inf/NaN.  On success *ctx is a new context (host bookkeeping only); release with nb_free.
 */
int nb_init(nb_ctx** ctx, int64_t N, const double* m, const double* x, const double* v, double eps,
            const nb_config* cfg);

/*
 * nb_predict — Taylor-extrapolate ALL N particles from their own t_i to time t (PAPER.md:58:
 * "the kinematic state will be estimated using Taylor expansions"; orders per reading R6):
 * x_p to 5th order, v_p to 4th, a_p to 3rd.  Fills the internal predicted j-records that
 * nb_force streams.  t may be any time (also < t_i).
 */
int nb_predict(nb_ctx* ctx, double t);

/*
 * nb_force — the O(N n_act) pairwise evaluation (eq. 1-2 and their first two time
 * derivatives, reading R3): for each active particle i = active_idx[k], over all j != i of the
 * predicted records,
 *   a = sum m_j dx / s^(3/2), jerk = da/dt, snap = d2a/dt2, pot = -sum m_j / s^(1/2),
 *   s = |x_j - x_i|^2 + eps^2.
 * active_idx (h/d): n_act unique int32 in [0, N), any order; NULL = all N in index order (then
 * n_act must equal N).  Outputs (h/d), row k <-> active_idx[k]: a, jerk, snap [n_act][3], pot
 * [n_act]; any may be NULL.  The results are also kept inside the context for nb_corrector.
 * Small active sets are split over j-slices so that the whole GPU is used, and the
 * partial sums are added in a fixed order: results are bitwise reproducible run to run.
 * n_act == 0 is a no-op.  NB_ESTATE if no nb_predict since the last change of state.
 */
int nb_force(nb_ctx* ctx, const int32_t* active_idx, int64_t n_act,
             double* a, double* jerk, double* snap, double* pot);

/* 8th order only: crackle [n_act][3] (h/d) of the last nb_force, row k <-> active_idx[k].  NB_ESTATE otherwise. */
int nb_force_crackle(nb_ctx* ctx, double* crackle);

/*
 * nb_corrector — finish the Hermite-6 step (formulas: reading R10) for the active
 * particles of the preceding nb_force (same active_idx, same n_act): corrects x and v with the
 * two-point quintic Hermite quadrature, stores the new a, jerk, snap and the interpolant's crackle,
 * sets t_i to the time of the last nb_predict.
 *   dt > 0 : shared time step — every active particle steps h = dt; dt_i := dt.
 *   dt <= 0: block time steps — h = dt_i; then the new power-of-two dt_i from the
 *            6th-order Aarseth criterion (reading R11) under the block rule (reading R12).
 * Invalidates the predicted records.
 */
int nb_corrector(nb_ctx* ctx, const int32_t* active_idx, int64_t n_act, double dt);

/*
 * nb_next_block — block scheduler: t_next = min_i (t_i + dt_i) and the active list
 * { i : t_i + dt_i == t_next } in increasing index order.  t_next, n_act: HOST pointers always.
 * active_idx (h/d): capacity N int32; may be NULL (then the list stays inside the context and
 * nb_force / nb_corrector accept NB_ACTIVE_INTERNAL in its place).
 */
int nb_next_block(nb_ctx* ctx, double* t_next, int32_t* active_idx, int64_t* n_act);

/* Pass as active_idx to use the list the last nb_next_block left inside the context. */
#define NB_ACTIVE_INTERNAL ((const int32_t*)(uintptr_t)1)

/*
 * nb_run_blocks — advance the system by whole block steps without the host in the loop:
 * repeats { nb_next_block; stop if t_next > t_end; nb_predict(t_next); nb_force(internal list);
 * nb_corrector(internal list, per-particle dt) } at most max_steps times.  Every decision of a step -
 * t_next, the active list, n_act, the j-split of the force launch (reading R15; "determined
 * step by step") - is taken on the device, and a step is four kernels (scheduler, predictor, force, reduction +
 * corrector) inside a CUDA graph that holds eight steps; for small active sets the force kernel predicts the
 * j-records it reads and the predictor's pass is skipped.  The host enqueues batches of replays and reads
 * the counters after each batch.  The arithmetic and its order are those of the separate calls: states
 * agree bit for bit.  The predicted records (NB_XP ...) are not defined afterwards.
 * steps_done, t_last (time of the last completed step; -1 if none), sum_n_act (sum of n_act over the
 * steps: interactions = sum_n_act * (N - 1)): HOST pointers, any may be NULL.  Synchronises the stream.
 */
int nb_run_blocks(nb_ctx* ctx, double t_end, int64_t max_steps, int64_t* steps_done, double* t_last,
                  int64_t* sum_n_act);

/*
 * nb_step_log — the device's own record of the most recent block steps nb_run_blocks took (up to 8192): for each, the
 * number of active particles and the device clock (%globaltimer) read by the step's last kernel, in microseconds relative
 * to the first returned step.  Differences of consecutive stamps are the full cost of a block step on the device, launch
 * gaps included - the per-step figures of profiles/ come from here.  n_act, t_us: HOST arrays of `capacity` entries.
 * Returns the number of entries written (oldest first), or a negative nb_status.  Synchronises the stream.
 */
int64_t nb_step_log(nb_ctx* ctx, int64_t capacity, int64_t* n_act, double* t_us);

/* Read / write one field for the particles idx[0..n) (h/d; NULL = the first n in index order). */
int nb_get_state(nb_ctx* ctx, int field, const int32_t* idx, int64_t n, double* out);
int nb_set_state(nb_ctx* ctx, int field, const int32_t* idx, int64_t n, const double* in);

/*
 * nb_energy — kinetic and potential energy of the STORED state (x, v at t_i; meaningful when all
 * t_i are equal): K = 1/2 sum m |v|^2, W = 1/2 sum m_i pot_i with pot from a full evaluation.
 * kinetic, potential: HOST pointers always.  Invalidates the predicted records.
 */
int nb_energy(nb_ctx* ctx, double* kinetic, double* potential);

/*
 * nb_check_indices — verify an index list (h/d) the way nb_config.check_indices does, on demand: NB_OK if all n
 * indices are in [0, N) and (unique != 0) pairwise different, NB_EINVAL otherwise (also for n > N: no call takes a
 * longer list).  Synchronises the stream.  n == 0 is NB_OK.  (the active subset, m <= N.)
 */
int nb_check_indices(nb_ctx* ctx, const int32_t* idx, int64_t n, int unique);

/* CTAs of force kernel shape `kernel` (nb_plan.kernel: 0 or 1) that the device keeps resident per multiprocessor for this
 * context's order, as the occupancy calculator reports it; the launch plan assumes nb_plan.ctas_per_sm.  NB_EINVAL (< 0)
 * on a bad argument. */
int nb_resident_ctas(const nb_ctx* ctx, int kernel);

/* Kernel launches issued by this context so far (what bench.py reports as gpu_launches). */
int64_t nb_launch_count(const nb_ctx* ctx);

/* Device time in ms of the force kernel(s) of the last nb_force (CUDA events on cfg->stream,
 * excludes index upload and output copies); synchronises the stream.  < 0 on error. */
double nb_last_force_ms(nb_ctx* ctx);

const char* nb_strerror(int status);
const char* nb_last_error(const nb_ctx* ctx); /* detail of the last NB_ECUDA of this context, "" if none */
void nb_free(nb_ctx* ctx);                    /* host bookkeeping only; NULL is allowed */

#ifdef __cplusplus
}
#endif
#endif /* NB_H */
