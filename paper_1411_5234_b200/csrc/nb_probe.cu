// nb_probe.cu — libnbprobe.so: measurement aids (nb_probe.h).  Register-resident instruction streams that measure the
// pipe constants DESIGN.md section 6 quotes.  Nothing of the method lives here and libnb.so does not contain this file.
#include <cuda_runtime.h>
#include <algorithm>

#include "nb_probe.h"

namespace {

struct DeviceGuard {
    int prev = -1;
    cudaError_t err;
    explicit DeviceGuard(int device)
    {
        err = cudaGetDevice(&prev);
        if (err == cudaSuccess && prev != device) err = cudaSetDevice(device);
        else prev = -1;
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

// 8 independent FMA chains per thread, 256 threads x 4 CTAs per SM: nothing but DFMA in the loop.
__global__ void __launch_bounds__(256) fp64_peak_kernel(double* out, int iters)
{
    double a0 = threadIdx.x * 1e-9, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
    const double m = 0.999999, c = 1e-7;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 16; ++u) {
            a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
            a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
        }
    }
    const double r = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
    if (r == 12345.678) out[blockIdx.x] = r;     // never true; keeps the chains alive
}

// Operand-source probes: 8 independent chains, 64 DFMAs per loop iteration, in three flavours.
//   0: acc = acc * m + c, m and c loop constants       -> two cycles per DFMA (the pipe's rate)
//   1: acc_k = b_k * d_k + acc_k, three register pairs  -> three cycles
//   2: acc_k = q * d_k + acc_k, q shared by the run     -> two cycles where the operand-reuse cache supplies q
#define P_DFMA(d, a, b, c) asm volatile("fma.rn.f64 %0, %1, %2, %3;" : "=d"(d) : "d"(a), "d"(b), "d"(c))
#define P_FFMA(d, a, b, c) asm volatile("fma.rn.f32 %0, %1, %2, %3;" : "=f"(d) : "f"(a), "f"(b), "f"(c))
#define P_FADD(d, a, b) asm volatile("add.rn.f32 %0, %1, %2;" : "=f"(d) : "f"(a), "f"(b))
#define P_FSUB(d, a, b) asm volatile("sub.rn.f32 %0, %1, %2;" : "=f"(d) : "f"(a), "f"(b))
#define P_DADD(d, a, b) asm volatile("add.rn.f64 %0, %1, %2;" : "=d"(d) : "d"(a), "d"(b))
#define P_D2F(f, d) asm volatile("cvt.rn.f32.f64 %0, %1;" : "=f"(f) : "d"(d))
#define P_F2D(d, f) asm volatile("cvt.f64.f32 %0, %1;" : "=d"(d) : "f"(f))

template <int KIND>
__global__ void __launch_bounds__(256) dfma_source_kernel(double* out, int iters, double seed)
{
    double a[8], b[8], d[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        a[k] = threadIdx.x + k; b[k] = seed * (k + 1) + threadIdx.x * 1e-9; d[k] = seed * 0.1 * (k + 2) + threadIdx.x * 1e-9;
    }
    const double q = seed + threadIdx.x * 1e-9;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                if (KIND == 0) P_DFMA(a[k], a[k], 0.999999, 1e-7);
                if (KIND == 1) P_DFMA(a[k], b[k], d[k], a[k]);
                if (KIND == 2) P_DFMA(a[k], q, d[k], a[k]);
            }
        }
    }
    double r = 0;
#pragma unroll
    for (int k = 0; k < 8; ++k) r += a[k];
    if (r == 12345.678) out[blockIdx.x] = r;
}

// The streams of a mixed-precision pair evaluation (nb_probe.h: nbp_mixed_rates).  64 "elements" per loop iteration.
template <int KIND>
__global__ void __launch_bounds__(256) mixed_rate_kernel(double* out, int iters, float seed)
{
    float fa[8], fb[8], fd[8], lo[8];
    double da[8], db[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        fa[k] = threadIdx.x + k; fb[k] = seed * (k + 1) + threadIdx.x * 1e-6f; fd[k] = seed * 0.1f * (k + 2) + threadIdx.x * 1e-6f;
        lo[k] = 0.f; da[k] = threadIdx.x + 0.5 * k; db[k] = (double)seed * (k + 3) + threadIdx.x * 1e-9;
    }
    unsigned long long pa[8], pb[8], pd[8];                  // packed pairs of floats for the f32x2 streams
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        pa[k] = ((unsigned long long)__float_as_uint(fa[k]) << 32) | __float_as_uint(fa[k] + 0.5f);
        pb[k] = ((unsigned long long)__float_as_uint(fb[k]) << 32) | __float_as_uint(fb[k] * 1.5f);
        pd[k] = ((unsigned long long)__float_as_uint(fd[k]) << 32) | __float_as_uint(fd[k] * 0.5f);
    }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                if (KIND == 0) P_FFMA(fa[k], fb[k], fd[k], fa[k]);                       // FFMA, three register sources
                // ptxas removes conversions whose results are dead, so the conversion streams are dependent chains
                // (8 independent chains per thread, like the FMA streams): double -> float -> double -> ...
                if (KIND == 1) { P_D2F(fa[k], da[k]); P_F2D(da[k], fa[k]); }             // one F2F.F32.F64 + one F2F.F64.F32
                if (KIND == 2) { P_D2F(fa[k], da[k]); P_F2D(da[k], fa[k]); P_DADD(da[k], da[k], db[k]); }   // ... + one DADD
                if (KIND == 3) { double t; P_F2D(t, fb[k]); P_DADD(da[k], da[k], t); P_FADD(fb[k], fb[k], fd[k]); }   // DP accumulation of a changing SP term
                if (KIND == 4) {                                                         // float-float accumulation (two-sum)
                    float s, bb, t1, t2, t3;
                    P_FADD(s, fa[k], fb[k]); P_FSUB(bb, s, fa[k]); P_FSUB(t1, s, bb); P_FSUB(t2, fa[k], t1); P_FSUB(t3, fb[k], bb);
                    P_FADD(t2, t2, t3); P_FADD(lo[k], lo[k], t2); fa[k] = s;
                }
                if (KIND == 5) { P_DFMA(da[k], da[k], 0.999999, 1e-7); P_FFMA(fa[k], fb[k], fd[k], fa[k]); }   // both pipes, 1:1
                if (KIND == 6) P_FFMA(fa[k], fb[0], fd[k], fa[k]);                       // FFMA, one source shared by the run
                if (KIND == 7) P_FFMA(fa[k], fa[k], 0.999999f, 1e-7f);                   // FFMA, one register and two immediates
                if (KIND == 8) asm volatile("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(pa[k]) : "l"(pb[k]), "l"(pd[k]));   // FFMA2: two fp32 FMAs per lane, three register pairs
                if (KIND == 9) asm volatile("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(pa[k]) : "l"(pb[0]), "l"(pd[k]));   // FFMA2, one source shared by the run
            }
        }
    }
    double r = 0;
#pragma unroll
    for (int k = 0; k < 8; ++k) r += (double)fa[k] + da[k] + (double)lo[k] + (double)__uint_as_float((unsigned)pa[k]) + (double)__uint_as_float((unsigned)(pa[k] >> 32));
    if (r == 12345.678) out[blockIdx.x] = r;
}

// time one launch of `launch(iters)` after a warm-up launch; ms of the second
template <class F>
int time_launch(cudaStream_t st, F launch, float* ms)
{
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return -4;
    int rc = 0;
    for (int round = 0; round < 2 && rc == 0; ++round) {
        cudaEventRecord(e0, st);
        launch();
        if (cudaGetLastError() != cudaSuccess) rc = -4;
        cudaEventRecord(e1, st);
        if (cudaEventSynchronize(e1) != cudaSuccess || cudaEventElapsedTime(ms, e0, e1) != cudaSuccess) rc = -4;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    return rc;
}

}  // namespace

extern "C" {

int nbp_fp64_peak(int device, void* stream, void* workspace, size_t workspace_bytes, double seconds, double* tflops, int* n_sm_out)
{
    if (!workspace || workspace_bytes < 65536 || !tflops || !(seconds > 0)) return -1;
    DeviceGuard g(device);
    if (g.err != cudaSuccess) return -4;
    cudaStream_t st = (cudaStream_t)stream;
    int n_sm = 0;
    if (cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, device) != cudaSuccess) return -4;
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return -4;
    const double flop_per_iter = (double)n_sm * 4 * 256 * 16 * 8 * 2;
    int iters = 20000;
    float ms = 0;
    double best = 0;
    int rc = 0;
    // calibrate, then run back-to-back launches of ~0.25 s until `seconds` have elapsed
    for (int round = 0; round < 2 && rc == 0; ++round) {
        double elapsed = 0;
        do {
            cudaEventRecord(e0, st);
            fp64_peak_kernel<<<n_sm * 4, 256, 0, st>>>((double*)workspace, iters);
            if (cudaGetLastError() != cudaSuccess) { rc = -4; break; }
            cudaEventRecord(e1, st);
            if (cudaEventSynchronize(e1) != cudaSuccess || cudaEventElapsedTime(&ms, e0, e1) != cudaSuccess) { rc = -4; break; }
            elapsed += ms * 1e-3;
            if (round == 1) best = flop_per_iter * iters / (ms * 1e-3) * 1e-12;   // the LAST launch: sustained, not burst
        } while (round == 1 && elapsed < seconds);
        if (round == 0 && ms > 0) iters = std::max(1000, (int)(iters * 250.0 / ms));
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    if (rc != 0) return rc;
    *tflops = best;
    if (n_sm_out) *n_sm_out = n_sm;
    return 0;
}

int nbp_dfma_sources(int device, void* stream, void* workspace, size_t workspace_bytes, int kind, double sm_mhz, double* cycles)
{
    if (!workspace || workspace_bytes < 65536 || !cycles || kind < 0 || kind > 2 || !(sm_mhz > 0)) return -1;
    DeviceGuard g(device);
    if (g.err != cudaSuccess) return -4;
    cudaStream_t st = (cudaStream_t)stream;
    int n_sm = 0;
    if (cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, device) != cudaSuccess) return -4;
    const int iters = 40000;
    const double seed = 1e-3;
    double* out = (double*)workspace;
    float ms = 0;
    const int rc = time_launch(st, [&] {
        if (kind == 0) dfma_source_kernel<0><<<n_sm * 3, 256, 0, st>>>(out, iters, seed);
        else if (kind == 1) dfma_source_kernel<1><<<n_sm * 3, 256, 0, st>>>(out, iters, seed);
        else dfma_source_kernel<2><<<n_sm * 3, 256, 0, st>>>(out, iters, seed);
    }, &ms);
    if (rc != 0) return rc;
    // 3 x 8 warps per SM = 6 per sub-partition, 64 DFMAs per iteration each
    *cycles = (double)ms * 1e-3 * sm_mhz * 1e6 / (6.0 * 64.0 * iters);
    return 0;
}

int nbp_mixed_rates(int device, void* stream, void* workspace, size_t workspace_bytes, int kind, double sm_mhz, double* cycles)
{
    if (!workspace || workspace_bytes < 65536 || !cycles || kind < 0 || kind > 9 || !(sm_mhz > 0)) return -1;
    DeviceGuard g(device);
    if (g.err != cudaSuccess) return -4;
    cudaStream_t st = (cudaStream_t)stream;
    int n_sm = 0;
    if (cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, device) != cudaSuccess) return -4;
    const int iters = 20000;
    const float seed = 1e-3f;
    double* out = (double*)workspace;
    float ms = 0;
    const int rc = time_launch(st, [&] {
        switch (kind) {
            case 0: mixed_rate_kernel<0><<<n_sm * 3, 256, 0, st>>>(out, iters, seed); break;
            case 1: mixed_rate_kernel<1><<<n_sm * 3, 256, 0, st>>>(out, iters, seed); break;
            case 2: mixed_rate_kernel<2><<<n_sm * 3, 256, 0, st>>>(out, iters, seed); break;
            case 3: mixed_rate_kernel<3><<<n_sm * 3, 256, 0, st>>>(out, iters, seed); break;
            case 4: mixed_rate_kernel<4><<<n_sm * 3, 256, 0, st>>>(out, iters, seed); break;
            case 5: mixed_rate_kernel<5><<<n_sm * 3, 256, 0, st>>>(out, iters, seed); break;
            case 6: mixed_rate_kernel<6><<<n_sm * 3, 256, 0, st>>>(out, iters, seed); break;
            case 7: mixed_rate_kernel<7><<<n_sm * 3, 256, 0, st>>>(out, iters, seed); break;
            case 8: mixed_rate_kernel<8><<<n_sm * 3, 256, 0, st>>>(out, iters, seed); break;
            default: mixed_rate_kernel<9><<<n_sm * 3, 256, 0, st>>>(out, iters, seed); break;
        }
    }, &ms);
    if (rc != 0) return rc;
    *cycles = (double)ms * 1e-3 * sm_mhz * 1e6 / (6.0 * 64.0 * iters);   // per element (kinds 3-5: per element group)
    return 0;
}

}  // extern "C"
