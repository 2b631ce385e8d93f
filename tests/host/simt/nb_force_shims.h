// tests/host/simt/nb_force_shims.h — TEST INFRASTRUCTURE: what nb_force.cu writes as inline PTX, as the C++ operation each of
// them is (the test removes those definitions from the copy of nb_force.cu it compiles and includes this file instead).
//   F, M, V*: one IEEE operation each (fma / mul / add / sub, round to nearest), as the PTX says.
//   rsqrt_seed: MUFU.RSQ64H gives about 20 good bits; here the exact value cut to the high word (the kernel's cubic step takes
//   either to 2^-60).  rsqrt_f32: MUFU.RSQ (2^-22); here the correctly rounded value.
//   mbarrier + 1-D bulk copy (UBLKCP): the copy happens at once and completes one phase of the barrier; a wait passes when
//   the phase with the given parity has completed.  Shared-memory addresses are 32-bit offsets from a fixed symbol.
//   On the GPU the copy lands at some unknown moment between its issue and the completion of the barrier's phase.  "At once" is
//   the earliest moment (it shows a stage that is overwritten while somebody still reads it); NB_SIMT_BULK_COPY=late is the
//   latest: the destination is filled with 0xFF bytes (NaN) at issue and the data arrives when the first thread waits on the
//   barrier (it shows a read that does not wait).  A copy still pending when the next kernel initialises its barriers aborts.
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
namespace simt {
struct PendingCopy { uint32_t dst; const void* src; uint32_t bytes; uint32_t bar; };
inline std::vector<PendingCopy>& pending_copies() { static std::vector<PendingCopy> v; return v; }
inline long long& late_copies() { static long long n = 0; return n; }      // copies delivered late so far (for the test)
inline bool bulk_copy_late() { const char* e = getenv("NB_SIMT_BULK_COPY"); return e && !strcmp(e, "late"); }
inline void deliver(uint32_t bar)
{
    auto& v = pending_copies();
    for (size_t k = 0; k < v.size();) {
        if (v[k].bar != bar) { ++k; continue; }
        memcpy(from_smem(v[k].dst), v[k].src, v[k].bytes);
        *(unsigned long long*)from_smem(bar) += 1;
        S().progress += 1; late_copies() += 1;
        v.erase(v.begin() + (long)k);
    }
}
}
extern "C" __attribute__((weak, used)) long long nb_simt_late_copies() { return simt::late_copies(); }
static inline void mbar_init(uint32_t bar, uint32_t)
{
    for (const auto& c : simt::pending_copies())
        if (c.bar == bar) { fprintf(stderr, "simt: a bulk copy of %u bytes was still in flight when its CTA exited\n", c.bytes); abort(); }
    *(unsigned long long*)simt::from_smem(bar) = 0;                                                           // phases completed so far
}
static inline void mbar_expect_tx(uint32_t, uint32_t) {}
static inline void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar)
{
    if (simt::bulk_copy_late()) {
        memset(simt::from_smem(dst), 0xFF, bytes);
        simt::pending_copies().push_back({dst, src, bytes, bar});
        return;
    }
    memcpy(simt::from_smem(dst), src, bytes);
    *(unsigned long long*)simt::from_smem(bar) += 1;
    simt::S().progress += 1;
}
static inline void mbar_wait(uint32_t bar, uint32_t parity)
{
    simt::deliver(bar);
    while ((*(volatile unsigned long long*)simt::from_smem(bar) & 1u) == parity) simt::yield();
}
