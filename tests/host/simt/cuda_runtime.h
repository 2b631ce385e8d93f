// tests/host/simt/cuda_runtime.h — TEST INFRASTRUCTURE (tests/test_simt_host_cpu.py): a stand-in for <cuda_runtime.h> with which
// the WHOLE library (nb_api.cu, nb_force.cu, nb_step.cu and their headers) compiles with g++ and runs on the host, one CUDA thread =
// one fibre, so that the kernels' structure - work queue, j-split, tile staging, shuffle reductions, partial-sum layouts, the
// fixed-order reduction, the one-kernel scheduler, the device-planned block step and its graph - can be compared with the oracle
// through the library's real C ABI where there is no GPU (and where compute-sanitizer is closed: profiles/r02_sanitizer.md).
//
// What it is: the SIMT execution model, restated for one OS thread.  A launch runs its CTAs one after the other; inside a CTA
// every thread is a ucontext fibre that runs until it has to wait (__syncthreads, __syncwarp, a shuffle / vote, an mbarrier);
// barriers count the threads that have not exited; shuffles and votes exchange through a per-warp slot array between two warp
// barriers.  Shared memory is `static` storage (CTAs do not overlap).  Global-memory atomics are plain operations.  Streams are
// in order and synchronous; a stream capture records the launches as closures and a graph launch replays them.
// Switches (environment, read at every launch): NB_SIMT_SMS = multiprocessors the device reports; NB_SIMT_CTA_ORDER = reverse |
// shuffle and NB_SIMT_THREAD_ORDER = reverse | shuffle = the order in which CTAs of a grid run and threads of a CTA are resumed
// (undefined on a GPU: results must not depend on it); NB_SIMT_BULK_COPY = late (nb_force_shims.h) = bulk copies land at the
// first mbarrier wait instead of at issue.  Every CTA starts with 0xFF bytes in its dynamic and static shared memory; built with
// -fsanitize=address (NB_SIMT_CXXFLAGS of the test) only the dynamic shared memory a launch asked for is addressable.
// What it is not: a product path (nothing under paper_1411_5234_b200/ refers to it; the library refuses to run without a CUDA
// device), a model of timing, of memory ordering or of races between CTAs, or a check of the machine code.  The GPU parity
// tests (-m gpu) remain the proof for the B200.
#pragma once
#include <ucontext.h>

#include <cmath>
#include <cstddef>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <ctime>
#include <functional>
#include <tuple>
#include <utility>
#include <vector>

#define NB_SIMT_HOST 1

// ---------------------------------------------------------------------------------------------------------------
// qualifiers and vector types
// ---------------------------------------------------------------------------------------------------------------
#define __global__
#define __device__
#define __host__
#define __forceinline__ inline
#define __launch_bounds__(...)
#define __align__(n) alignas(n)
// static shared memory: static storage, collected in one section so that every CTA can be started with garbage in it (on the GPU a
// CTA does not find zeros, nor what the CTA before it left).  Under AddressSanitizer plain statics instead: variables in a named
// section get no red zones, and there the bounds are worth more than the garbage.
#if defined(__SANITIZE_ADDRESS__)
#define __shared__ static
#else
#define NB_SIMT_SMEM_SECTION 1
#define __shared__ __attribute__((section("nb_smem"))) static
extern "C" char __start_nb_smem[] __attribute__((weak, visibility("hidden")));
extern "C" char __stop_nb_smem[] __attribute__((weak, visibility("hidden")));
#endif

struct alignas(16) double2 { double x, y; };
struct alignas(32) double4 { double x, y, z, w; };
struct alignas(16) float4 { float x, y, z, w; };
struct uint3 { unsigned x, y, z; };
static inline double2 make_double2(double x, double y) { return double2{x, y}; }
static inline double4 make_double4(double x, double y, double z, double w) { return double4{x, y, z, w}; }
static inline float4 make_float4(float x, float y, float z, float w) { return float4{x, y, z, w}; }

// ---------------------------------------------------------------------------------------------------------------
// the engine
// ---------------------------------------------------------------------------------------------------------------
namespace simt {

constexpr int MAX_THREADS = 1024;
constexpr size_t STACK_BYTES = 96 * 1024;

struct Warp {
    int alive = 0, arrived = 0;
    unsigned gen = 0;
    unsigned long long slot[32];
};

// Switching fibres: glibc's swapcontext saves and restores the signal mask with a system call on every switch, which dominates
// the run time of kernels that synchronise once per j-tile.  On x86-64 the switch is therefore done by hand (simt_switch.S:
// callee-saved registers and the stack pointer, nothing else - no fibre changes the FP control words or the signal mask);
// elsewhere ucontext is used.
#if defined(__x86_64__) && !defined(NB_SIMT_UCONTEXT)
#define NB_SIMT_FAST_SWITCH 1
extern "C" void nb_simt_switch(void** save_sp, void* load_sp);
#endif

struct Fibre {
    ucontext_t ctx;
    void* sp = nullptr;
    uint3 tid{0, 0, 0};
    int lane = 0, warp = 0;
    bool done = true;
};

struct Cta {
    uint3 bid{0, 0, 0}, bdim{1, 1, 1}, gdim{1, 1, 1};
    int alive = 0, arrived = 0;
    unsigned gen = 0;
    Warp warps[MAX_THREADS / 32];
};

struct State {
    Fibre fib[MAX_THREADS];
    char* stacks = nullptr;
    ucontext_t main_ctx;
    void* main_sp = nullptr;
    Fibre* self = nullptr;
    Cta cta;
    std::function<void()> body;               // the kernel call of the launch that is running
    bool capturing = false;
    std::vector<std::function<void()>>* capture = nullptr;
    long long launches = 0, permuted = 0, reordered = 0, switches = 0, progress = 0;   // permuted: launches run in another CTA order; reordered: CTAs run in another thread order; progress: arrivals, releases, exits, completed copies
    unsigned long long clock = 0;
};

inline State& S() { static State s; return s; }

inline void to_main(Fibre* f)
{
    State& s = S();
#ifdef NB_SIMT_FAST_SWITCH
    nb_simt_switch(&f->sp, s.main_sp);
#else
    swapcontext(&f->ctx, &s.main_ctx);
#endif
}
inline void to_fibre(Fibre* f)
{
    State& s = S();
    s.self = f;
#ifdef NB_SIMT_FAST_SWITCH
    nb_simt_switch(&s.main_sp, f->sp);
#else
    swapcontext(&s.main_ctx, &f->ctx);
#endif
}
inline void yield() { State& s = S(); ++s.switches; to_main(s.self); }

inline void fibre_entry()
{
    State& s = S();
    s.body();
    Fibre* f = s.self;
    f->done = true;
    s.progress += 1;
    s.cta.alive -= 1;
    s.cta.warps[f->warp].alive -= 1;
    to_main(f);                                  // never resumed
    abort();
}

// barrier over the threads of the CTA that have not exited
inline void cta_barrier()
{
    Cta& c = S().cta;
    const unsigned g = c.gen;
    c.arrived += 1; S().progress += 1;
    while (c.gen == g) {
        if (c.arrived >= c.alive) { c.arrived = 0; c.gen += 1; break; }
        yield();
    }
}

inline void warp_barrier()
{
    State& s = S();
    Warp& w = s.cta.warps[s.self->warp];
    const unsigned g = w.gen;
    w.arrived += 1; s.progress += 1;
    while (w.gen == g) {
        if (w.arrived >= w.alive) { w.arrived = 0; w.gen += 1; break; }
        yield();
    }
}

// static shared arrays inside TEMPLATE kernels do not follow the section attribute; the test appends a registration to their
// declarations instead (first execution of the kernel), and run_cta fills what is registered
inline std::vector<std::pair<char*, size_t>>& smem_regions() { static std::vector<std::pair<char*, size_t>> v; return v; }
inline int register_smem(void* p, size_t n) { smem_regions().emplace_back((char*)p, n); return 0; }
struct DynSmem { char* base = nullptr; size_t bytes = 0, asked = 0; };
inline DynSmem& dyn_smem_array() { static DynSmem d; return d; }
inline int register_dyn_smem(void* base, size_t bytes) { dyn_smem_array() = DynSmem{(char*)base, bytes}; return 0; }

// run one CTA to completion: round-robin over its fibres until all have exited
inline void run_cta(unsigned block, unsigned bid, unsigned grid)
{
    State& s = S();
    if (!s.stacks) s.stacks = (char*)aligned_alloc(4096, STACK_BYTES * MAX_THREADS);
    if (block > (unsigned)MAX_THREADS) { fprintf(stderr, "simt: block of %u threads\n", block); abort(); }
    // a CTA finds garbage in its dynamic shared memory, not what the CTA before it left there: NaN bytes here
    for (auto& r : smem_regions()) memset(r.first, 0xFF, r.second);
#ifdef NB_SIMT_SMEM_SECTION
    if (__start_nb_smem && __stop_nb_smem > __start_nb_smem) memset(__start_nb_smem, 0xFF, (size_t)(__stop_nb_smem - __start_nb_smem));
#endif
    if (dyn_smem_array().base && dyn_smem_array().asked) memset(dyn_smem_array().base, 0xFF, dyn_smem_array().asked);
    Cta& c = s.cta;
    c.bid = uint3{bid, 0, 0}; c.bdim = uint3{block, 1, 1}; c.gdim = uint3{grid, 1, 1};
    c.alive = (int)block; c.arrived = 0; c.gen = 0;
    for (unsigned w = 0; w < (block + 31) / 32; ++w) {
        c.warps[w].alive = (int)(block - 32 * w < 32 ? block - 32 * w : 32);
        c.warps[w].arrived = 0; c.warps[w].gen = 0;
    }
    for (unsigned t = 0; t < block; ++t) {
        Fibre& f = s.fib[t];
        f.tid = uint3{t, 0, 0}; f.lane = (int)(t & 31); f.warp = (int)(t >> 5); f.done = false;
#ifdef NB_SIMT_FAST_SWITCH
        // a fresh stack as nb_simt_switch expects to find it: six zeroed callee-saved registers, then the address it returns
        // to; at fibre_entry's first instruction the stack pointer is 8 mod 16, as after a call
        void** top = (void**)(s.stacks + STACK_BYTES * (t + 1));
        top[-2] = (void*)fibre_entry; top[-1] = nullptr;
        for (int r = 3; r <= 8; ++r) top[-r] = nullptr;
        f.sp = (void*)(top - 8);
#else
        getcontext(&f.ctx);
        f.ctx.uc_stack.ss_sp = s.stacks + STACK_BYTES * t;
        f.ctx.uc_stack.ss_size = STACK_BYTES;
        f.ctx.uc_link = nullptr;
        makecontext(&f.ctx, (void (*)())fibre_entry, 0);
#endif
    }
    // Which thread of a CTA runs first between two synchronisation points is not defined either.  NB_SIMT_THREAD_ORDER =
    // reverse | shuffle (a new permutation every round, reproducible) resumes the fibres in another order than 0, 1, 2, ...: a
    // read of shared or global memory that is not ordered after its write by a barrier then sees the old value in one of the
    // orders, and the results differ (a poor man's racecheck: it finds missing barriers, not memory-model subtleties).
    static unsigned ord[MAX_THREADS];
    const char* torder = getenv("NB_SIMT_THREAD_ORDER");
    const int tmode = !torder ? 0 : !strcmp(torder, "reverse") ? 1 : !strcmp(torder, "shuffle") ? 2 : 0;
    for (unsigned t = 0; t < block; ++t) ord[t] = tmode == 1 ? block - 1 - t : t;
    unsigned long long rnd = 0x9E3779B97F4A7C15ull * (unsigned long long)(s.launches * 4099 + bid + 1);
    s.reordered += tmode != 0;
    while (c.alive > 0) {
        const long long before = s.progress;
        if (tmode == 2)
            for (unsigned t = block - 1; t > 0; --t) {
                rnd += 0x9E3779B97F4A7C15ull;
                unsigned long long z = rnd;
                z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull; z = (z ^ (z >> 27)) * 0x94D049BB133111EBull; z ^= z >> 31;
                std::swap(ord[t], ord[z % (t + 1)]);
            }
        for (unsigned k = 0; k < block; ++k) {
            Fibre& f = s.fib[ord[k]];
            if (f.done) continue;
            to_fibre(&f);
        }
        s.self = nullptr;
        // a fibre yields only while it waits for something another fibre of the CTA has to do: a whole round in which nobody
        // arrived anywhere, left, or completed a copy will repeat for ever (a barrier some thread never reaches)
        if (s.progress == before && c.alive > 0) { fprintf(stderr, "simt: deadlock in CTA %u (%d threads waiting)\n", bid, c.alive); abort(); }
    }
}

// Dynamic shared memory is one static array of the translation unit (the test's edit of `extern __shared__`), larger than any
// launch asks for.  Under AddressSanitizer (NB_SIMT_CXXFLAGS=-fsanitize=address) every launch leaves only the bytes it asked
// for addressable: an access to dynamic shared memory beyond the launch's size is then reported like one on the GPU would be by
// compute-sanitizer's memcheck.  Without the sanitizer the two calls below do nothing.
#if defined(__SANITIZE_ADDRESS__)
extern "C" void __asan_poison_memory_region(void const volatile*, size_t);
extern "C" void __asan_unpoison_memory_region(void const volatile*, size_t);
#define NB_SIMT_POISON(p, n) __asan_poison_memory_region((p), (n))
#define NB_SIMT_UNPOISON(p, n) __asan_unpoison_memory_region((p), (n))
#else
#define NB_SIMT_POISON(p, n) ((void)(p), (void)(n))
#define NB_SIMT_UNPOISON(p, n) ((void)(p), (void)(n))
#endif
inline void bound_dyn_smem(size_t asked)
{
    DynSmem& d = dyn_smem_array();
    if (!d.base) return;
    if (asked > d.bytes) { fprintf(stderr, "simt: a launch asks for %zu bytes of dynamic shared memory\n", asked); abort(); }
    const size_t lim = (asked + 7) / 8 * 8;                  // the sanitizer's granule
    d.asked = asked;
    NB_SIMT_UNPOISON(d.base, d.bytes);
    if (lim < d.bytes) NB_SIMT_POISON(d.base + lim, d.bytes - lim);
}

template <class... P, class... A>
inline void launch(void (*kernel)(P...), long long grid, long long block, size_t smem, void* /*stream*/, A&&... args)
{
    State& s = S();
    std::tuple<std::decay_t<P>...> held(std::forward<A>(args)...);      // kernel arguments are passed by value
    auto run = [kernel, grid, block, smem, held]() {
        State& st = S();
        st.launches += 1;
        bound_dyn_smem(smem);
        st.body = [kernel, &held]() { std::apply(kernel, held); };
        // The order in which a GPU starts and finishes the CTAs of a grid is not defined.  NB_SIMT_CTA_ORDER = reverse | shuffle
        // (a different permutation for every launch, reproducible) runs them in another order than 0, 1, 2, ...: work queues,
        // last-block-done patterns and fixed-order reductions must give the same bits in any of them.
        const char* order = getenv("NB_SIMT_CTA_ORDER");
        if (order && (!strcmp(order, "reverse") || !strcmp(order, "shuffle"))) {
            std::vector<unsigned> perm((size_t)grid);
            for (long long b = 0; b < grid; ++b) perm[(size_t)b] = (unsigned)(order[0] == 'r' ? grid - 1 - b : b);
            if (order[0] == 's') {
                unsigned long long x = 0x9E3779B97F4A7C15ull * (unsigned long long)(st.launches + 1);
                for (long long b = grid - 1; b > 0; --b) {                      // Fisher-Yates on a splitmix64 stream
                    x += 0x9E3779B97F4A7C15ull;
                    unsigned long long z = x;
                    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull; z = (z ^ (z >> 27)) * 0x94D049BB133111EBull; z ^= z >> 31;
                    std::swap(perm[(size_t)b], perm[(size_t)(z % (unsigned long long)(b + 1))]);
                }
            }
            st.permuted += grid > 1;
            for (unsigned b : perm) run_cta((unsigned)block, b, (unsigned)grid);
        } else {
            for (long long b = 0; b < grid; ++b) run_cta((unsigned)block, (unsigned)b, (unsigned)grid);
        }
        st.body = nullptr;
    };
    if (s.capturing) s.capture->push_back(run);
    else run();
}

inline unsigned long long clock_ns() { return S().clock += 1000; }

}  // namespace simt

// for the test that permutes the CTAs: how many multi-CTA launches ran in another order than 0, 1, 2, ...
extern "C" __attribute__((weak, used)) long long nb_simt_permuted_launches() { return simt::S().permuted; }
extern "C" __attribute__((weak, used)) long long nb_simt_reordered_ctas() { return simt::S().reordered; }

#define threadIdx (simt::S().self->tid)
#define blockIdx (simt::S().cta.bid)
#define blockDim (simt::S().cta.bdim)
#define gridDim (simt::S().cta.gdim)

// ---------------------------------------------------------------------------------------------------------------
// device intrinsics
// ---------------------------------------------------------------------------------------------------------------
static inline void __syncthreads() { simt::cta_barrier(); }
static inline void __syncwarp(unsigned = 0xffffffffu) { simt::warp_barrier(); }
static inline void __threadfence() {}

namespace simt {
template <class T>
inline T warp_exchange(T v, int src)          // src: lane to read from (own value if it lies outside the warp)
{
    static_assert(sizeof(T) <= 8, "shuffles move at most 64 bits");
    State& s = S();
    Warp& w = s.cta.warps[s.self->warp];
    unsigned long long bits = 0;
    memcpy(&bits, &v, sizeof(T));
    w.slot[s.self->lane] = bits;
    warp_barrier();
    const unsigned long long got = (src >= 0 && src < 32) ? w.slot[src] : bits;
    warp_barrier();                           // nobody overwrites a slot before everybody has read
    T r;
    memcpy(&r, &got, sizeof(T));
    return r;
}
}  // namespace simt

template <class T> static inline T __shfl_xor_sync(unsigned, T v, int o) { return simt::warp_exchange(v, simt::S().self->lane ^ o); }
template <class T> static inline T __shfl_sync(unsigned, T v, int src) { return simt::warp_exchange(v, src & 31); }
template <class T> static inline T __shfl_up_sync(unsigned, T v, unsigned o)
{
    const int lane = simt::S().self->lane;
    return simt::warp_exchange(v, lane - (int)o >= 0 ? lane - (int)o : -1);
}
static inline int __any_sync(unsigned, int pred)
{
    simt::State& s = simt::S();
    simt::Warp& w = s.cta.warps[s.self->warp];
    w.slot[s.self->lane] = pred ? 1 : 0;
    simt::warp_barrier();
    int any = 0;
    const int first = 32 * s.self->warp;
    for (int l = 0; l < 32 && first + l < (int)s.cta.bdim.x; ++l)
        if (!s.fib[first + l].done && w.slot[l]) any = 1;
    simt::warp_barrier();
    return any;
}

template <class T> static inline T __ldcg(const T* p) { return *p; }
static inline int __double2hiint(double x) { int64_t b; memcpy(&b, &x, 8); return (int)(b >> 32); }
static inline int __double2loint(double x) { int64_t b; memcpy(&b, &x, 8); return (int)(b & 0xffffffff); }
static inline double __hiloint2double(int hi, int lo)
{
    const uint64_t b = ((uint64_t)(uint32_t)hi << 32) | (uint32_t)lo;
    double x; memcpy(&x, &b, 8); return x;
}
static inline int __float_as_int(float f) { int b; memcpy(&b, &f, 4); return b; }
static inline float __int_as_float(int b) { float f; memcpy(&f, &b, 4); return f; }
static inline int __ffs(int v) { return __builtin_ffs(v); }
static inline int min(int a, int b) { return a < b ? a : b; }
static inline int max(int a, int b) { return a > b ? a : b; }

// atomics on global memory: one OS thread, so plain read-modify-write
template <class T> static inline T atomicAdd(T* p, T v) { const T old = *p; *p = old + v; return old; }
static inline unsigned atomicAdd(unsigned* p, int v) { const unsigned old = *p; *p = old + (unsigned)v; return old; }
template <class T> static inline T atomicOr(T* p, T v) { const T old = *p; *p = old | v; return old; }

// ---------------------------------------------------------------------------------------------------------------
// the CUDA runtime calls the library makes: one device, in-order synchronous streams, memory = host memory
// ---------------------------------------------------------------------------------------------------------------
enum cudaError_t { cudaSuccess = 0, cudaErrorInvalidValue = 1 };
enum cudaMemcpyKind { cudaMemcpyHostToHost, cudaMemcpyHostToDevice, cudaMemcpyDeviceToHost, cudaMemcpyDeviceToDevice };
enum { cudaStreamNonBlocking = 1, cudaStreamCaptureModeThreadLocal = 1 };
enum { cudaDevAttrMultiProcessorCount = 16 };
enum { cudaFuncAttributeMaxDynamicSharedMemorySize = 8, cudaFuncAttributePreferredSharedMemoryCarveout = 9, cudaSharedmemCarveoutMaxShared = 100 };
typedef struct simt_stream_st* cudaStream_t;
typedef struct simt_event_st* cudaEvent_t;
typedef std::vector<std::function<void()>>* cudaGraph_t;
typedef std::vector<std::function<void()>>* cudaGraphExec_t;

static inline const char* cudaGetErrorString(cudaError_t e) { return e == cudaSuccess ? "no error" : "simt: invalid value"; }
static inline cudaError_t cudaGetLastError() { return cudaSuccess; }
static inline cudaError_t cudaGetDevice(int* d) { *d = 0; return cudaSuccess; }
static inline cudaError_t cudaSetDevice(int d) { return d == 0 ? cudaSuccess : cudaErrorInvalidValue; }
static inline cudaError_t cudaDeviceGetAttribute(int* v, int attr, int)
{
    if (attr != cudaDevAttrMultiProcessorCount) return cudaErrorInvalidValue;
    const char* e = getenv("NB_SIMT_SMS");                  // how many SMs the emulated device reports (the launch plans depend on it)
    *v = e ? atoi(e) : 148;
    return *v >= 1 ? cudaSuccess : cudaErrorInvalidValue;
}
static inline cudaError_t cudaMemcpyAsync(void* dst, const void* src, size_t n, cudaMemcpyKind, cudaStream_t)
{
    if (simt::S().capturing) return cudaErrorInvalidValue;  // the library captures kernel launches only
    memmove(dst, src, n);
    return cudaSuccess;
}
static inline cudaError_t cudaMemsetAsync(void* dst, int v, size_t n, cudaStream_t)
{
    if (simt::S().capturing) return cudaErrorInvalidValue;
    memset(dst, v, n);
    return cudaSuccess;
}
static inline cudaError_t cudaStreamSynchronize(cudaStream_t) { return cudaSuccess; }
static inline cudaError_t cudaStreamCreateWithFlags(cudaStream_t* s, unsigned) { *s = nullptr; return cudaSuccess; }
static inline cudaError_t cudaStreamDestroy(cudaStream_t) { return cudaSuccess; }
static inline cudaError_t cudaEventCreate(cudaEvent_t* e) { *e = nullptr; return cudaSuccess; }
static inline cudaError_t cudaEventDestroy(cudaEvent_t) { return cudaSuccess; }
static inline cudaError_t cudaEventRecord(cudaEvent_t, cudaStream_t) { return cudaSuccess; }
static inline cudaError_t cudaEventSynchronize(cudaEvent_t) { return cudaSuccess; }
static inline cudaError_t cudaEventElapsedTime(float* ms, cudaEvent_t, cudaEvent_t) { *ms = 0.f; return cudaSuccess; }
template <class K> static inline cudaError_t cudaFuncSetAttribute(K, int, int) { return cudaSuccess; }
template <class K> static inline cudaError_t cudaOccupancyMaxActiveBlocksPerMultiprocessor(int* n, K, int, size_t) { *n = 4; return cudaSuccess; }

// stream capture: launches are recorded instead of run; a graph launch replays them in order
static inline cudaError_t cudaStreamBeginCapture(cudaStream_t, int)
{
    simt::State& s = simt::S();
    if (s.capturing) return cudaErrorInvalidValue;
    s.capture = new std::vector<std::function<void()>>();
    s.capturing = true;
    return cudaSuccess;
}
static inline cudaError_t cudaStreamEndCapture(cudaStream_t, cudaGraph_t* g)
{
    simt::State& s = simt::S();
    if (!s.capturing) return cudaErrorInvalidValue;
    s.capturing = false;
    *g = s.capture; s.capture = nullptr;
    return cudaSuccess;
}
static inline cudaError_t cudaGraphInstantiate(cudaGraphExec_t* e, cudaGraph_t g, unsigned long long)
{
    *e = new std::vector<std::function<void()>>(*g);
    return cudaSuccess;
}
static inline cudaError_t cudaGraphDestroy(cudaGraph_t g) { delete g; return cudaSuccess; }
static inline cudaError_t cudaGraphExecDestroy(cudaGraphExec_t e) { delete e; return cudaSuccess; }
static inline cudaError_t cudaGraphLaunch(cudaGraphExec_t e, cudaStream_t)
{
    for (auto& node : *e) node();
    return cudaSuccess;
}
