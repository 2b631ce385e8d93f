/*
 * nb_probe.h — C ABI of libnbprobe.so: MEASUREMENT AIDS, not part of the method and not part of libnb.so.
 * bench.py and the sweep scripts load this library to measure the denominators and the pipe constants that
 * DESIGN.md section 6 quotes (FP64 FMA peak, cycles per DFMA by operand source, and the conversion / FP32 /
 * float-float rates behind the mixed-precision decision).  Every call: device ordinal, a
 * cudaStream_t (NULL = default stream), >= 64 KiB of device workspace; returns 0 or a negative code
 * (-1 bad argument, -4 CUDA error).  The caller's current device is restored on return.
 */
#ifndef NB_PROBE_H
#define NB_PROBE_H
#include <stddef.h>
#ifdef __cplusplus
extern "C" {
#endif

/* Sustained rate of a register-resident chain of independent FP64 FMAs on every SM, run for about `seconds`:
 * TFLOP/s (FMA = 2 flop) of the LAST launch (sustained, not burst) and the SM count. */
int nbp_fp64_peak(int device, void* stream, void* workspace, size_t workspace_bytes, double seconds, double* tflops, int* n_sm);

/* Cycles one warp-wide DFMA holds the FP64 pipe of an SM sub-partition, from a stream of independent DFMAs whose
 * sources are (kind 0) one register and two constants, (kind 1) three different registers, (kind 2) three registers
 * of which one is shared by the whole run (operand-reuse cache).  sm_mhz: the SM clock to convert with. */
int nbp_dfma_sources(int device, void* stream, void* workspace, size_t workspace_bytes, int kind, double sm_mhz, double* cycles);

/* Cycles per warp-wide instruction and SM sub-partition of the streams a mixed-precision pair evaluation would be
 * made of ("DP for reciprocal distances and accumulation, SP elsewhere"):
 *   kind 0  FFMA, three register sources
 *   kind 1  conversion round trip double -> float -> double (one F2F.F32.F64 + one F2F.F64.F32 per element)
 *   kind 2  the same round trip + one DADD per element
 *   kind 3  DP accumulation of an SP term: F2F.F64.F32 + DADD + one FADD (that changes the term) per element
 *   kind 4  float-float accumulation (two-sum, 6 FADD-class ops per element, no conversion)
 *   kind 5  DFMA (2-source) and FFMA interleaved 1:1 - do the FP32 and FP64 pipes issue side by side?
 *   kind 6  FFMA with one source shared by the run (operand-reuse cache)
 *   kind 7  FFMA with one register and two immediates
 *   kind 8  FFMA2 (fma.rn.f32x2: two fp32 FMAs per lane on register pairs, sm_100), three register-pair sources
 *   kind 9  FFMA2 with one source shared by the run
 * `cycles` = sub-partition cycles per warp instruction of the named kind (kinds 1-4: per element;
 * kind 5: per DFMA+FFMA pair). */
int nbp_mixed_rates(int device, void* stream, void* workspace, size_t workspace_bytes, int kind, double sm_mhz, double* cycles);

#ifdef __cplusplus
}
#endif
#endif
