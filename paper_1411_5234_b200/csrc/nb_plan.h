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
NB_HD int nb_pow2ceil(int v) { int p = 1; while (p < v) p <<= 1; return p; }
NB_HD int nb_pow2floor(int v) { int p = 1; while (2 * p <= v) p <<= 1; return p; }

// Which shape: CTA tiles of 128 particles run the pipe 6-12 % better than warp units (shared j-tiles, longer items;
// measured) but leave the lanes of a ragged last tile idle; warp units waste nothing.  CTA tiles are taken
// from 256 active particles on when at least 93 % of their lanes hold a particle.
constexpr int64_t LI_MIN_ACT = 256;
NB_HD bool nb_use_cta_tiles(int64_t n_act)
{
    const int64_t lanes = (n_act + LI_UNIT - 1) / LI_UNIT * LI_UNIT;
    return n_act >= LI_MIN_ACT && n_act * 100 >= lanes * 93;
}
// block steps whose evaluation has at most this many warp units let the force kernel predict the j-records itself
constexpr int PIF_MAX_UNITS = 2;

// ---------------------------------------------------------------------------------------------------------------
// Warp units (kernel 1).  n_act = 32 n_full + rem.  The first n_full units hold 32 particles each.  The remainder is
// decomposed from its highest bit down into units of p = 16, 8, ... 1 particles, every one full, EXCEPT that a rest
// which nearly fills the next power of two (at most an eighth of it, or one particle, missing) becomes one padded unit:
// 31 -> one unit of 32 with 31 valid lanes rather than 16 + 8 + 4 + 2 + 1 (five units, each streaming all j-records).
// unit u -> first row k0, width p (lanes are split p ways over particles, 32/p ways over the records of a step) and
// the number of valid particles.
// ---------------------------------------------------------------------------------------------------------------
NB_HD void nb_wu_rest_step(int rem, int* p, int* valid)
{
    const int pc = nb_pow2ceil(rem);
    if (pc - rem <= (pc >= 16 ? pc / 8 : 1)) { *p = pc; *valid = rem; }
    else { *p = nb_pow2floor(rem); *valid = *p; }
}

NB_HD void nb_wu_unit(int n_act, int u, int* k0, int* p, int* valid)
{
    const int n_full = n_act >> 5;
    if (u < n_full) { *k0 = u << 5; *p = 32; *valid = 32; return; }
    int rem = n_act & 31, k = n_full << 5;
    for (int idx = u - n_full;; --idx) {
        nb_wu_rest_step(rem, p, valid);
        if (idx == 0) { *k0 = k; return; }
        k += *valid; rem -= *valid;
    }
}

// number of units; *work = sum of p / 32 (units weighted by the time a slice costs them), *w_max = the largest weight
NB_HD int nb_wu_count(int64_t n_act, double* work, double* w_max)
{
    const int n_full = (int)(n_act >> 5);
    int n = n_full, rem = (int)(n_act & 31);
    double w = (double)n_full, wm = n_full ? 1.0 : 0.0;
    while (rem > 0) {
        int p, valid;
        nb_wu_rest_step(rem, &p, &valid);
        w += p / 32.0;
        if (p / 32.0 > wm) wm = p / 32.0;
        rem -= valid; ++n;
    }
    *work = w; *w_max = wm;
    return n;
}

// Everything about a plan except the split S.
struct PlanShape {
    int kernel;        // 0 CTA tiles of 128 particles, 1 warp units (nb.h: nb_plan.kernel)
    int unit, tile, ctas_per_sm;
    double fixed;      // cost of starting a work item, in j-tiles of a full unit
    double work, w_max;   // kernel 1: sum and maximum of the unit weights p / 32; kernel 0: n_units, 1
    int64_t n_units, n_tiles, resident, s_max;
};

// max_split > 0 caps S (1 = no j-split: the "Bfactor off" arm of the paper's Fig. 1); 0 = no cap.
NB_HD PlanShape nb_plan_shape(int64_t Npad, int64_t n_act, int n_sm, int64_t max_split = 0)
{
    PlanShape p;
    const int64_t rows = nb_partial_rows(Npad);
    if (nb_use_cta_tiles(n_act)) {
        // CTA tiles: a work item is (i-tile of 128 particles, j-slice); resident = CTAs on the device
        p.kernel = 0; p.unit = LI_UNIT; p.tile = LI_TJ; p.ctas_per_sm = LI_CTAS_PER_SM; p.fixed = 4.0;
        p.n_units = (n_act + LI_UNIT - 1) / LI_UNIT;
        p.work = (double)p.n_units; p.w_max = 1.0;
        p.n_tiles = Npad / LI_TJ;
        p.resident = (int64_t)n_sm * LI_CTAS_PER_SM;
        p.s_max = nb_min64(nb_min64(rows / (p.n_units * LI_UNIT), 2048), p.n_tiles / 2);
    } else {
        // warp units: a work item is (unit, j-slice); resident = warps on the device
        p.kernel = 1; p.unit = 32; p.tile = WU_TJ; p.ctas_per_sm = WU_CTAS_PER_SM; p.fixed = 1.0;
        p.n_units = nb_wu_count(n_act, &p.work, &p.w_max);
        p.n_tiles = Npad / WU_TJ;
        p.resident = (int64_t)n_sm * WU_CTAS_PER_SM * WU_WARPS;
        p.s_max = nb_min64(nb_min64(rows / n_act, 16384), p.n_tiles / 2);
    }
    p.s_max = nb_max64(1, nb_min64(p.s_max, p.n_tiles));
    if (max_split > 0) p.s_max = nb_min64(p.s_max, max_split);
    return p;
}

// Cost of splitting into S slices, in units of one j-tile of work on one work slot (a negative value: S leaves a
// slice empty and is not a candidate).  Work items (unit, slice) are pulled from a queue by `resident` workers (CTAs
// or warps); an item of a unit of weight w costs w * slice_tiles + fixed.
// CTA tiles (kernel 0): co-resident CTAs do not get equal shares of the FP64 pipe, so a single round of equal items
// ends with the slow CTA of every SM running alone (measured 0.78 of the issue bound against 0.86 with ten rounds):
// up to eight rounds the rounds are counted whole plus half a round (745 slices x 4 tiles = 5.03 rounds measured 0.814,
// 592 x 4 = 4.00 rounds 0.833), more rounds items / resident + 0.9 for the tail.
// Warp units (kernel 1): up to one round the largest item decides; up to four rounds the last round is counted whole;
// beyond that the queue balances the workers up to a tail of about 0.7 of the largest item.  (For nb_force alone half a
// round of twice as long slices measured up to 15 % faster at N = 2^18 - 8 particles: 24.2 against 28.8 us - but the same
// plan serves the device-planned block steps, where the force kernel predicts its j-records and more, shorter slices win:
// 41.5 against 48.2 us per step for 5-16 active particles.  One plan for both keeps nb_run_blocks bitwise equal to the
// separate calls, and the block step is the case the j-split exists for.)
NB_HD double nb_split_cost(const PlanShape& p, int64_t S, int64_t* slice_tiles)
{
    const int64_t st = (p.n_tiles + S - 1) / S;
    *slice_tiles = st;
    if ((p.n_tiles + st - 1) / st != S) return -1.0;
    const int64_t items = p.n_units * S;
    if (p.kernel == 0) {
        const double rounds = items <= 8 * p.resident ? (double)((items + p.resident - 1) / p.resident) + 0.5
                                                      : (double)items / (double)p.resident + 0.9;
        return rounds * ((double)st + p.fixed);
    }
    const double c_max = p.w_max * (double)st + p.fixed;
    const double c_avg = p.work / (double)p.n_units * (double)st + p.fixed;
    if (items <= p.resident) return c_max;
    if (items <= 4 * p.resident) return (double)((items + p.resident - 1) / p.resident) * c_max;   // a round lasts as long as its heaviest item
    return (double)items * c_avg / (double)p.resident + 0.7 * c_max;
}

// The candidates for S.  The cost above is piecewise: flat or falling up to a whole number of rounds (items = k x
// resident), and beyond a few rounds smooth with a minimum near S* = sqrt(tail x n_tiles x resident / (n_units x
// fixed)).  So instead of all S in [1, s_max] (tens of thousands of 64-bit divisions - microseconds of every block step
// when the plan is made on the device) only these are examined: S = 1, S = s_max, the largest S with items <= k x
// resident for k = 1 .. 4, and S*; each with the neighbouring slice lengths.  Candidate c -> a valid S (one that leaves
// no slice empty) or 0.
constexpr int NB_SPLIT_CANDIDATES = 24;

NB_HD int64_t nb_isqrt_floor(double x)
{
    int64_t r = 1;
    while ((double)(r * 2) * (double)(r * 2) <= x) r *= 2;            // no libm: identical on host and device
    for (int64_t b = r / 2; b > 0; b /= 2)
        if ((double)(r + b) * (double)(r + b) <= x) r += b;
    return r;
}

NB_HD int64_t nb_split_candidate(const PlanShape& p, int c)
{
    int64_t target;                                         // an S to aim for; snapped to a valid one below
    const int group = c / 3, var = c % 3;                   // var: slice length st, st + 1, st - 1
    if (group == 0) target = 1;
    else if (group == 1) target = p.s_max;
    else if (group <= 5) target = (int64_t)(group - 1) * p.resident / p.n_units;
    else if (group == 6) {
        const double tail = p.kernel == 0 ? 0.9 : 0.7 * p.w_max;
        target = nb_isqrt_floor(tail * (double)p.n_tiles * (double)p.resident / ((double)p.n_units * p.fixed));
    } else target = 2 * p.n_units <= p.resident ? p.resident / (2 * p.n_units) : 0;  // group 7: half a round
    if (target < 1) return 0;
    target = nb_min64(target, p.s_max);
    int64_t st = (p.n_tiles + target - 1) / target + (var == 1 ? 1 : var == 2 ? -1 : 0);
    if (st < 1 || st > p.n_tiles) return 0;
    const int64_t S = (p.n_tiles + st - 1) / st;
    return S >= 1 && S <= p.s_max ? S : 0;
}

// The split is the candidate S of least cost, the smallest such S on ties.  Candidates c_begin, c_begin + c_stride, ...
// (the host takes all of them, the device spreads them over a warp).
NB_HD int64_t nb_best_split(const PlanShape& p, int c_begin, int c_stride, double* best_cost)
{
    int64_t best = 0;
    double bc = 1e300;
    for (int c = c_begin; c < NB_SPLIT_CANDIDATES; c += c_stride) {
        const int64_t S = nb_split_candidate(p, c);
        if (S == 0) continue;
        int64_t st;
        const double cost = nb_split_cost(p, S, &st);
        if (cost >= 0.0 && (cost < bc || (cost == bc && S < best))) { bc = cost; best = S; }
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
    int n_act, n_units, n_split, slice_tiles, n_items, ld, red_T;
    int predict;               // 1: the force kernel predicts the j-records it reads; the predictor kernel returns at once
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
    d->ld = p.kernel == 0 ? (int)(p.n_units * p.unit) : (int)n_act;
    d->red_T = nb_reduce_threads(n_act, (int)S);
    d->predict = p.kernel == 1 && p.n_units <= PIF_MAX_UNITS;
}
