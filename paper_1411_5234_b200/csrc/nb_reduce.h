// nb_reduce.h — the fixed-order sum of the per-slice partial sums of one evaluation (row a3; the deterministic form of
// the paper's Bfactor reduction), as ONE device function: reduce_partials_kernel (nb_force.cu, after
// nb_force) and reduce_correct_kernel (nb_step.cu, inside a device-planned block step) both call it, so both add the
// same numbers in the same order and produce the same bits.
// T threads per active particle (T a power of two from nb_reduce_threads): thread `lane` adds slices lane, lane + T, ...
// in increasing order (eight slices' loads are issued together, the additions stay in order), then the T lane sums are
// combined by a binary tree in shared memory.  The order depends only on (S, T).  T = 1 is the plain loop over slices
// (large active sets, few slices: the loads of neighbouring threads coalesce over k).
#pragma once
#include "nb_internal.h"

// One pass of a block of RED_THREADS threads over the particles k0 .. k0 + RED_THREADS / T - 1.  Returns true in the one
// thread per particle that ends up with the total in r[] (and sets *k_out); all threads of the block must call it.
template <int NC>
__device__ __forceinline__ bool nb_reduce_pass(const double* __restrict__ partial, int ld, int S, int T, int n_act, int k0,
                                               double (*sm)[RED_THREADS], double (&r)[NC], int* k_out)
{
    const int R = RED_THREADS / T;                         // active particles per block and pass
    const int kl = threadIdx.x % R, lane = threadIdx.x / R;
    const int k = k0 + kl;
#pragma unroll
    for (int c = 0; c < NC; ++c) r[c] = 0.0;
    if (k < n_act) {
        const size_t plane = (size_t)NC * ld;
        const double* P = partial + (size_t)lane * plane + k;
        int s = lane;
        // eight slices at a time: all 8 x NC loads are issued before the first addition (the loads are volatile asm, which
        // ptxas keeps in order and therefore cannot fold into a short register-saving load-add chain), then added in order
        for (; s + 7 * T < S; s += 8 * T, P += (size_t)8 * T * plane) {
            double v[8][NC];
#pragma unroll
            for (int u = 0; u < 8; ++u)
#pragma unroll
                for (int c = 0; c < NC; ++c)
                    asm volatile("ld.global.cg.f64 %0, [%1];" : "=d"(v[u][c]) : "l"(P + (size_t)u * T * plane + (size_t)c * ld));
#pragma unroll
            for (int u = 0; u < 8; ++u)
#pragma unroll
                for (int c = 0; c < NC; ++c) r[c] += v[u][c];
        }
        for (; s < S; s += T, P += (size_t)T * plane) {
            double v[NC];
#pragma unroll
            for (int c = 0; c < NC; ++c) asm volatile("ld.global.cg.f64 %0, [%1];" : "=d"(v[c]) : "l"(P + (size_t)c * ld));
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
