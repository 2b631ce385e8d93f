// tests/host/simt/nb_force_shims.h — TEST INFRASTRUCTURE: what nb_force.cu writes as inline PTX, as the C++ operation each of
// them is (the test removes those definitions from the copy of nb_force.cu it compiles and includes this file instead).
//   F, M, V*: one IEEE operation each (fma / mul / add / sub, round to nearest), as the PTX says.
//   rsqrt_seed: MUFU.RSQ64H gives about 20 good bits; here the exact value cut to the high word (the kernel's cubic step takes
//   either to 2^-60).  rsqrt_f32: MUFU.RSQ (2^-22); here the correctly rounded value.
//   mbarrier + 1-D bulk copy (UBLKCP): the copy happens at once and completes one phase of the barrier; a wait passes when
//   the phase with the given parity has completed.  Shared-memory addresses are 32-bit offsets from a fixed symbol.
#pragma once
#include <cuda_runtime.h>

static inline double F(double a, double b, double c) { return std::fma(a, b, c); }
static inline double M(double a, double b) { return a * b; }
static inline double rsqrt_seed(double s)
{
    const double y = 1.0 / std::sqrt(s);
    int64_t b; memcpy(&b, &y, 8);
    b &= ~((int64_t(1) << 32) - 1);
    double r; memcpy(&r, &b, 8); return r;
}
static inline float rsqrt_f32(float s) { return 1.0f / std::sqrt(s); }
#define VSUB(d, a, b) d = (a) - (b)
#define VADD(d, a, b) d = (a) + (b)
#define VMUL(d, a, b) d = (a) * (b)
#define VFMA(d, a, b, c) d = std::fma((a), (b), (c))
#define VFNMA(d, a, b, c) d = std::fma(-(a), (b), (c))
#define VRSQ(d, a) d = rsqrt_seed(a)
#define VTWICE(d, a) d = __hiloint2double(__double2hiint(a) + 0x00100000, __double2loint(a))

namespace simt {
inline char smem_anchor;                                     // shared memory is static storage of this library: within 2 GiB of here
inline uint32_t to_smem(const void* p) { return (uint32_t)(int32_t)((intptr_t)p - (intptr_t)&smem_anchor); }
inline char* from_smem(uint32_t a) { return (char*)((intptr_t)&smem_anchor + (intptr_t)(int32_t)a); }    // (integer arithmetic: not "inside" the anchor object)
}
static inline uint32_t smem_u32(const void* p) { return simt::to_smem(p); }
static inline void mbar_init(uint32_t bar, uint32_t) { *(unsigned long long*)simt::from_smem(bar) = 0; }      // phases completed so far
static inline void mbar_expect_tx(uint32_t, uint32_t) {}
static inline void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar)
{
    memcpy(simt::from_smem(dst), src, bytes);
    *(unsigned long long*)simt::from_smem(bar) += 1;
    simt::S().progress += 1;
}
static inline void mbar_wait(uint32_t bar, uint32_t parity)
{
    while ((*(volatile unsigned long long*)simt::from_smem(bar) & 1u) == parity) simt::yield();
}
