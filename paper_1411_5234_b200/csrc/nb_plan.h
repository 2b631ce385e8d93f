// nb_plan.h — how an evaluation for n_act active particles is mapped onto the GPU (reading R15; the "Bfactor" of
// PAPER.md:59-65, "determined step by step").  Pure integer / double logic compiled for the host (nb_plan_force,
// nb_force) AND for the device (nb_run_blocks plans every block step on the GPU, so the host never has to learn
// n_act).  Both sides run the same functions, so they produce the same plan.
#pragma once
#include <stdint.h>
#include "nb_internal.h"

#ifdef __CUDACC__
#define NB_HD __host__ __device__ __forceinline__
#else
#define NB_HD inline
#endif

NB_HD int64_t nb_pad_n(int64_t N) { return (N + NB_PAD - 1) / NB_PAD * NB_PAD; }
NB_HD int64_t nb_partial_rows(int64_t Npad) { return 8 * Npad + (int64_t(1) << 19); }   // rows of each partial-sum plane
NB_HD int64_t nb_min64(int64_t a, int64_t b) { return a < b ? a : b; }
NB_HD int64_t nb_max64(int64_t a, int64_t b) { return a > b ? a : b; }

// Everything about a plan except the split S.
struct PlanShape {
    int kernel;        // 0 lanes-over-i, 1 lanes-over-j, 2 lanes-over-i with 32-particle units (nb.h: nb_plan.kernel)
    int unit, tile, sub, ctas_per_sm, fixed;
    int64_t n_units, n_tiles, resident, s_max;
};

// max_split > 0 caps S (1 = no j-split: the "Bfactor off" arm of the paper's Fig. 1); 0 = no cap.
NB_HD PlanShape nb_plan_shape(int64_t Npad, int64_t n_act, int n_sm, int64_t max_split = 0)
{
    PlanShape p;
    const int64_t rows = nb_partial_rows(Npad);
    if (n_act <= LJ_MAX_ACT) {
        // lanes-over-j: a work item is (warp i-group, j-slice); resident = warps on the device
        p.kernel = 1; p.unit = LJ_I; p.tile = LJ_TJ; p.sub = 1; p.ctas_per_sm = LJ_CTAS_PER_SM; p.fixed = 6;
        p.n_units = (n_act + LJ_I - 1) / LJ_I;
        p.n_tiles = Npad / LJ_TJ;
        p.resident = (int64_t)n_sm * LJ_CTAS_PER_SM * LJ_WARPS;
        p.s_max = nb_min64(rows / (p.n_units * LJ_I), p.n_tiles / 4);
    } else {
        // lanes-over-i: a work item is (i-tile, j-slice); resident = CTAs on the device.  Up to LIW_MAX_ACT active
        // particles the i-tile is 32 particles and the CTA's warps each take a part of every j-tile (sub > 1).
        const bool small = n_act <= LIW_MAX_ACT;
        p.kernel = small ? 2 : 0; p.sub = small ? LI_W : 1;
        p.unit = LI_UNIT / p.sub; p.tile = LI_TJ; p.ctas_per_sm = LI_CTAS_PER_SM; p.fixed = 2;
        p.n_units = (n_act + p.unit - 1) / p.unit;
        p.n_tiles = Npad / LI_TJ;
        p.resident = (int64_t)n_sm * LI_CTAS_PER_SM;
        p.s_max = nb_min64(nb_min64(rows / (p.n_units * p.unit * p.sub), 2048), p.n_tiles / 2);
    }
    p.s_max = nb_max64(1, nb_min64(p.s_max, p.n_tiles));
    if (max_split > 0) p.s_max = nb_min64(p.s_max, max_split);
    return p;
}

// Cost of splitting into S slices, in units of one j-tile of work on one work slot (a negative value: S leaves a
// slice empty and is not a candidate).  Work items (unit, slice) are pulled from a queue by `resident` workers (CTAs
// or warps); an item costs slice_tiles + fixed.
// Lanes-over-i with 128-particle tiles (kernel 0): co-resident CTAs do not get equal shares of the FP64 pipe, so a
// single round of equal items ends with the slow CTA of every SM running alone (measured 0.78 of the issue bound
// against 0.86 with ten rounds): one round counts 1.5, more rounds items / resident + 0.9 for the tail.
// The other shapes (tiny active sets, latency-bound): up to four rounds the last round is counted whole; beyond that
// the queue balances the workers up to a tail of about 0.7 items.
NB_HD double nb_split_cost(const PlanShape& p, int64_t S, int64_t* slice_tiles)
{
    const int64_t st = (p.n_tiles + S - 1) / S;
    *slice_tiles = st;
    if ((p.n_tiles + st - 1) / st != S) return -1.0;
    const int64_t items = p.n_units * S;
    double rounds;
    if (p.kernel == 0)
        rounds = items <= p.resident ? 1.5 : (double)items / (double)p.resident + 0.9;
    else
        rounds = items <= 4 * p.resident ? (double)((items + p.resident - 1) / p.resident)
                                         : (double)items / (double)p.resident + 0.7;
    return rounds * (double)(st + p.fixed);
}

// The split is the S in [1, s_max] of least cost, the smallest such S on ties (S = 1 is always a candidate).
NB_HD int64_t nb_best_split(const PlanShape& p, int64_t s_begin, int64_t s_stride, double* best_cost)
{
    int64_t best = 0;
    double bc = 1e300;
    for (int64_t S = s_begin; S <= p.s_max; S += s_stride) {
        int64_t st;
        const double c = nb_split_cost(p, S, &st);
        if (c >= 0.0 && c < bc) { bc = c; best = S; }
    }
    *best_cost = bc;
    return best;
}

// threads per active particle of the partial-sum reduction: enough to spread the planes, few enough that large active
// sets keep coalesced rows
NB_HD int nb_reduce_threads(int64_t n_act, int n_planes)
{
    int T = 1;
    while (T < RED_THREADS && T * 4 <= n_planes && n_act * T < (int64_t(1) << 18)) T <<= 1;
    return T;
}

// The launch parameters the force, reduction and corrector kernels read from device memory when a block step is
// planned on the GPU (nb_run_blocks); the host path passes the same numbers as kernel arguments.
struct DevPlan {
    int stop;                  // 1: t_next > t_end (or the step budget is used up) - every kernel of the step returns at once
    int kernel;
    int n_act, n_units, n_split, slice_tiles, n_items, ld, n_planes, red_T;
    double t_next;
    double t_end;
    long long max_split;       // cap on S (0: none), see nb_plan_shape
    long long steps_left;      // block steps this call may still take
    long long steps_done;
    long long sum_act;         // sum of n_act over the steps done (interactions = sum_act * (N - 1))
    double t_last;             // time of the last completed block step
};

NB_HD void nb_fill_devplan(DevPlan* d, const PlanShape& p, int64_t S, int64_t n_act)
{
    int64_t st;
    nb_split_cost(p, S, &st);
    d->kernel = p.kernel;
    d->n_act = (int)n_act;
    d->n_units = (int)p.n_units;
    d->n_split = (int)S;
    d->slice_tiles = (int)st;
    d->n_items = (int)(p.n_units * S);
    d->ld = (int)(p.n_units * p.unit);
    d->n_planes = (int)(S * p.sub);
    d->red_T = nb_reduce_threads(n_act, d->n_planes);
}
