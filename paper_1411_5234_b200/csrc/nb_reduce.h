// nb_reduce.h — the fixed-order sum of the per-slice partial sums of one evaluation (row a3; the deterministic form of
// the paper's Bfactor reduction), as ONE device function: reduce_partials_kernel (nb_force.cu, after
// nb_force) and reduce_correct_kernel (nb_step.cu, inside a device-planned block step) both call it, so both add the
// same numbers in the same order and produce the same bits.
// T threads per active particle (T a power of two from nb_reduce_threads): thread `lane` adds slices lane, lane + T, ...
// in increasing order, then the T lane sums are
// combined by a binary tree in shared memory.  The order depends only on (S, T).  T = 1 is the plain loop over slices
// (large active sets, few slices: the loads of neighbouring threads coalesce over k).
#pragma once
#include "nb_internal.h"

// Where the partial sum (slice s, component c, row k) of an evaluation lives.  Two layouts, chosen by T (so by n_act and S):
//   T < RED_THREADS (a block reduces several particles; a warp's threads are neighbouring rows k of 32 / R slices): [s][c][k];
//   T = RED_THREADS (tiny active sets: a whole block per particle, a warp's threads are 32 neighbouring slices): [c][k][s].
// Either way a warp's load touches about 8 sectors, not 32 (the [s][c][k] layout read with lanes over s cost the reduction
// of 8 particles x 2341 slices 17 us of LSU time; profiles/).
struct PartialLayout {
    size_t stride_s, stride_c, stride_k;
    __host__ __device__ PartialLayout(int NC, int ld, int S, bool slice_minor)
        : stride_s(slice_minor ? 1 : (size_t)NC * ld), stride_c(slice_minor ? (size_t)ld * S : (size_t)ld), stride_k(slice_minor ? (size_t)S : 1) {}
};

// One pass of a block of RED_THREADS threads over the particles k0 .. k0 + RED_THREADS / T - 1.  Returns true in the one
// thread per particle that ends up with the total in r[] (and sets *k_out); all threads of the block must call it.
template <int NC>
__device__ __forceinline__ bool nb_reduce_pass(const double* __restrict__ partial, int ld, int S, int T, int n_act, int k0,
                                               double (*sm)[RED_THREADS], double (&r)[NC], int* k_out)
{
    const int R = RED_THREADS / T;                         // active particles per block and pass
    const int kl = threadIdx.x % R, lane = threadIdx.x / R;
    const int k = k0 + kl;
    const PartialLayout L(NC, ld, S, nb_slice_minor(T));
#pragma unroll
    for (int c = 0; c < NC; ++c) r[c] = 0.0;
    if (k < n_act) {
        const double* P = partial + (size_t)lane * L.stride_s + (size_t)k * L.stride_k;
        // one slice at a time: the NC loads of a slice are in flight together, the additions stay in slice order.  (Issuing
        // 2, 4 or 8 slices' loads together measured SLOWER: 26.0 / 29.1 / 32.1 / 34.4 us for force + reduction of 8 particles
        // x 2048 slices - the LSU queue fills, stall_lg_throttle - so the plain loop stays.)
        int s = lane;
        for (; s < S; s += T, P += (size_t)T * L.stride_s) {
            double v[NC];
#pragma unroll
            for (int c = 0; c < NC; ++c) v[c] = __ldcg(P + (size_t)c * L.stride_c);
#pragma unroll
            for (int c = 0; c < NC; ++c) r[c] += v[c];
        }
    }
    for (int off = T >> 1; off > 0; off >>= 1) {
        if (lane >= off && lane < 2 * off) {
#pragma unroll
            for (int c = 0; c < NC; ++c) sm[c][threadIdx.x] = r[c];
        }
        __syncthreads();
        if (lane < off) {
#pragma unroll
            for (int c = 0; c < NC; ++c) r[c] += sm[c][threadIdx.x + off * R];
        }
        __syncthreads();
    }
    *k_out = k;
    return lane == 0 && k < n_act;
}

template <int NC>
__device__ __forceinline__ void nb_store_totals(const ForceArgs& A, int k, const double (&r)[NC])
{
    A.out_a[3 * k] = r[0]; A.out_a[3 * k + 1] = r[1]; A.out_a[3 * k + 2] = r[2];
    A.out_j[3 * k] = r[3]; A.out_j[3 * k + 1] = r[4]; A.out_j[3 * k + 2] = r[5];
    A.out_s[3 * k] = r[6]; A.out_s[3 * k + 1] = r[7]; A.out_s[3 * k + 2] = r[8];
    A.out_p[k] = -r[9];
    if (NC == 13) { A.out_c[3 * k] = r[10]; A.out_c[3 * k + 1] = r[11]; A.out_c[3 * k + 2] = r[12]; }
}
