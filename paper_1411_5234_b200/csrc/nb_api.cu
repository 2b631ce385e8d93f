// nb_api.cu — the C ABI of include/nb.h: context, workspace carving, launch planning, call-order
// checks.  No arithmetic of the method lives here; every step runs in the kernels of nb_force.cu
// and nb_step.cu.
#include <algorithm>
#include <cfloat>
#include <climits>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>

#include "nb_internal.h"
#include "nb_plan.h"

namespace {

constexpr size_t ALIGN = 256;
inline size_t align_up(size_t x, size_t a = ALIGN) { return (x + a - 1) / a * a; }
inline int64_t pad_n(int64_t N) { return nb_pad_n(N); }
inline int64_t partial_rows(int64_t Npad) { return nb_partial_rows(Npad); }
inline size_t scratch_bytes(int64_t Npad) { return 65536 + (size_t)Npad / 8; }

struct Carve {
    size_t off = 0;
    char* base;
    explicit Carve(void* b) : base((char*)b) {}
    template <class T> T* take(size_t count) { T* p = (T*)(base + off); off = align_up(off + count * sizeof(T)); return p; }
};

// one place that defines the workspace layout, used for sizing (base = nullptr) and for carving
struct Layout {
    StateArrays s;
    double *fa, *fj, *fs, *fp, *fc;     // force results (fc: crackle, 8th order), row k <-> active_idx[k]
    double* partial;
    int32_t *idx_user, *idx_sched, *idx_tmp;
    double* stage;                      // staging for host <-> device transfers, 10 doubles per particle
    char* scratch;
    uint32_t* idx_bitmap;               // one bit per particle + one flag word: index-list verification (nb_config.check_indices)
    int* queue;                         // work queue of the force kernels (2 counters)
    DevPlan* devplan;                   // plan and counters of the device-planned block steps (nb_run_blocks)
    unsigned long long* steplog;        // [0] steps logged so far, then NB_STEP_LOG x (n_act, device clock in ns)
    size_t bytes;
    Layout(void* base, int64_t Npad)
    {
        Carve c(base);
        s.st0 = c.take<double4>(Npad); s.st1 = c.take<double4>(Npad); s.st2 = c.take<double4>(Npad);
        s.st3 = c.take<double4>(Npad); s.st4 = c.take<double4>(Npad); s.dt = c.take<double>(Npad);
        s.tn = c.take<double>(Npad);
        s.rec = c.take<double2>(Npad * REC_Q_MAX);          // 80-B records (112 B at the 8th order)
        s.st5 = c.take<double4>(Npad); s.st6 = c.take<double4>(Npad);
        s.recm = c.take<float4>(Npad * 4);                  // mixed-precision records (used only with NB_PREC_MIXED)
        fa = c.take<double>(3 * Npad); fj = c.take<double>(3 * Npad); fs = c.take<double>(3 * Npad); fp = c.take<double>(Npad);
        fc = c.take<double>(3 * Npad); s.fc = fc; s.order = 6;
        partial = c.take<double>(13 * partial_rows(Npad));   // 10 components, 13 at the 8th order
        idx_user = c.take<int32_t>(Npad); idx_sched = c.take<int32_t>(Npad); idx_tmp = c.take<int32_t>(Npad);
        stage = c.take<double>(10 * Npad);
        scratch = c.take<char>(scratch_bytes(Npad));
        idx_bitmap = c.take<uint32_t>(Npad / 32 + 64);      // [Npad/32] bits, then the flag word
        queue = c.take<int>(64);
        devplan = c.take<DevPlan>(1);
        steplog = c.take<unsigned long long>(1 + 2 * NB_STEP_LOG);
        bytes = c.off;
    }
};

}  // namespace

struct nb_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    bool on_device = false;
    bool check_idx = false;        // verify user index lists before use (nb_config.check_indices)
    int64_t N = 0, Npad = 0;
    double eps = 0, eta = 0.45, eta_s = 0.01;
    int k_min = -20, k_max = -3;
    int order = 6;
    int n_sm = 148;
    int64_t max_split = 0;         // cap on the j-split (0: the cost model decides)
    Layout L{nullptr, 0};
    double t_pred = 0;
    bool predicted = false;        // predicted records are valid
    int64_t forced_n = -1;         // n_act of the last nb_force since the last predict (-1: none)
    int64_t sched_n = -1;          // length of the internal active list (-1: none)
    int64_t launches = 0;
    int occ_li = 0, occ_wu = 0;    // CTAs of each force kernel shape that fit one SM (the plan assumes LI/WU_CTAS_PER_SM)
    cudaEvent_t ev0 = nullptr, ev1 = nullptr;
    cudaGraphExec_t step_graph = nullptr;   // one device-planned block step (built on first use)
    bool ev_valid = false;
    char err[256] = {0};
};

namespace {

int fail_cuda(nb_ctx* c, cudaError_t e, const char* where)
{
    snprintf(c->err, sizeof c->err, "%s: %s", where, cudaGetErrorString(e));
    return NB_ECUDA;
}
#define CU(call, where) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return fail_cuda(ctx, e_, where); } while (0)

// Every entry point that touches the device runs with the context's device current and puts the caller's device back
// on return: a process that holds contexts on several GPUs (or whose framework switched devices) stays correct.
struct DeviceGuard {
    int prev = -1;
    cudaError_t err = cudaSuccess;
    explicit DeviceGuard(int device)
    {
        err = cudaGetDevice(&prev);
        if (err == cudaSuccess && prev != device) err = cudaSetDevice(device);
        else if (err == cudaSuccess) prev = -1;             // nothing to restore
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
    DeviceGuard(const DeviceGuard&) = delete;
    DeviceGuard& operator=(const DeviceGuard&) = delete;
};
#define ON_DEVICE(ctx) DeviceGuard guard_((ctx)->device); if (guard_.err != cudaSuccess) return fail_cuda(ctx, guard_.err, "cudaSetDevice")

// The kernels see eps^2 only.  For 0 < eps < ~1.5e-154 it underflows to 0 or a denormal (flushed by the ftz rsqrt seed),
// so such an eps is treated as what it computes as: eps = 0, self pair masked by index.
inline bool eps2_is_zero(double eps) { return !(eps * eps >= DBL_MIN); }

// the fields of ForceArgs that do not depend on the plan
ForceArgs base_force_args(const nb_ctx* ctx)
{
    ForceArgs A{};
    const StateArrays& s = ctx->L.s;
    A.rec = s.rec; A.recm = s.recm;
    A.st0 = s.st0; A.st1 = s.st1; A.st2 = s.st2; A.st3 = s.st3; A.st4 = s.st4; A.st5 = s.st5; A.st6 = s.st6;
    A.eps2 = eps2_is_zero(ctx->eps) ? 0.0 : ctx->eps * ctx->eps;
    A.partial = ctx->L.partial;
    A.queue = ctx->L.queue;                                 // zeroed by nb_init, left at 0 by every launch
    A.out_a = ctx->L.fa; A.out_j = ctx->L.fj; A.out_s = ctx->L.fs; A.out_p = ctx->L.fp; A.out_c = ctx->L.fc;
    return A;
}

// One block step with every decision taken on the device, captured once as a CUDA graph of FOUR kernels: scheduler (+ plan
// of the force launch) -> predictor (returns at once when the force kernel predicts for itself) -> force (either shape,
// from the plan) -> partial-sum reduction + corrector.
constexpr int STEP_GRAPH_KERNELS = 4;
constexpr int STEPS_PER_GRAPH = 8;      // block steps per graph replay: graph-to-graph hand-over costs more than an edge inside one

int build_step_graph(nb_ctx* ctx)
{
    cudaStream_t cs;                                        // capture needs a non-default stream; nothing runs on it
    CU(cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking), "capture stream");
    cudaGraph_t graph = nullptr;
    int launches = 0;
    cudaError_t e = cudaStreamBeginCapture(cs, cudaStreamCaptureModeThreadLocal);
    if (e == cudaSuccess) {
        ForceArgs A = base_force_args(ctx);
        A.idx = ctx->L.idx_sched;
        A.dp = ctx->L.devplan;
        for (int k = 0; k < STEPS_PER_GRAPH && e == cudaSuccess; ++k) {
            e = nb_launch_devstep_head(ctx->L.s, ctx->N, ctx->Npad, ctx->n_sm, ctx->L.idx_sched, ctx->L.idx_tmp, ctx->L.scratch, ctx->L.devplan,
                                       cs, &launches);
            if (e == cudaSuccess) e = nb_launch_force_devplan(A, eps2_is_zero(ctx->eps), ctx->order, ctx->n_sm, (int)ctx->Npad, cs, &launches);
            if (e == cudaSuccess)
                e = nb_launch_devstep_tail(ctx->L.s, ctx->n_sm, ctx->L.idx_sched, A, ctx->L.devplan, ctx->L.steplog, ctx->eta, ctx->k_min,
                                           ctx->k_max, cs, &launches);
        }
        const cudaError_t e2 = cudaStreamEndCapture(cs, &graph);
        if (e == cudaSuccess) e = e2;
    }
    if (e == cudaSuccess) e = cudaGraphInstantiate(&ctx->step_graph, graph, 0);
    if (graph) cudaGraphDestroy(graph);
    cudaStreamDestroy(cs);
    if (e != cudaSuccess) return fail_cuda(ctx, e, "block-step graph");
    return launches == STEP_GRAPH_KERNELS * STEPS_PER_GRAPH ? NB_OK : NB_ECUDA;
}

// Verify a DEVICE index list: all in [0, N) and, if `unique`, pairwise different.  One kernel marks a bitmap and raises
// a flag, the flag is read back (the stream is synchronised).  NB_EINVAL on a bad list.
int verify_idx(nb_ctx* ctx, const int32_t* didx, int64_t n, bool unique)
{
    uint32_t* flag = ctx->L.idx_bitmap + ctx->Npad / 32;
    CU(cudaMemsetAsync(ctx->L.idx_bitmap, 0, (ctx->Npad / 32 + 1) * sizeof(uint32_t), ctx->stream), "index check");
    CU(nb_launch_check_idx(didx, n, ctx->N, ctx->L.idx_bitmap, flag, unique, ctx->stream), "index check");
    ctx->launches += 1;
    uint32_t bad = 0;
    CU(cudaMemcpyAsync(&bad, flag, sizeof bad, cudaMemcpyDeviceToHost, ctx->stream), "index check");
    CU(cudaStreamSynchronize(ctx->stream), "index check");
    return bad ? NB_EINVAL : NB_OK;
}

// device pointer to n_act indices: uploads a host list into `buf`, or passes a device list through; with index checking
// on, a user list is verified before anything reads through it
int resolve_idx(nb_ctx* ctx, const int32_t* idx, int64_t n, int32_t* buf, const int32_t** out, bool unique = true)
{
    if (idx == nullptr) { *out = nullptr; return NB_OK; }
    if (idx == NB_ACTIVE_INTERNAL) {
        if (ctx->sched_n < 0 || n != ctx->sched_n) return NB_ESTATE;
        *out = ctx->L.idx_sched;
        return NB_OK;
    }
    if (ctx->on_device) *out = idx;
    else {
        CU(cudaMemcpyAsync(buf, idx, n * sizeof(int32_t), cudaMemcpyHostToDevice, ctx->stream), "upload active_idx");
        *out = buf;
    }
    return ctx->check_idx && n > 0 ? verify_idx(ctx, *out, n, unique) : NB_OK;
}

int copy_out(nb_ctx* ctx, double* dst, const double* src, size_t count)
{
    if (!dst) return NB_OK;
    CU(cudaMemcpyAsync(dst, src, count * sizeof(double), ctx->on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost,
                       ctx->stream), "copy result");
    return NB_OK;
}

// The evaluation itself: plan, launch, results left in the context (fa, fj, fs, fp, fc).  didx: DEVICE indices or
// nullptr (all N).  No copies, no synchronisation: nb_force, nb_init's startup and nb_energy share it.
int plan_force(int64_t N, int64_t n_act, int n_sm, int64_t max_split, nb_plan* plan)
{
    if (!plan || N < 1 || n_act < 1 || n_act > N || n_sm < 1 || N > (int64_t(1) << 30) || max_split < 0) return NB_EINVAL;
    const PlanShape sh = nb_plan_shape(pad_n(N), n_act, n_sm, max_split);
    double cost;
    const int64_t S = nb_best_split(sh, 0, 1, &cost);
    int64_t st;
    nb_split_cost(sh, S, &st);
    nb_plan p{};
    p.kernel = sh.kernel; p.unit = sh.unit; p.tile = sh.tile; p.ctas_per_sm = sh.ctas_per_sm;
    p.n_units = (int)sh.n_units; p.n_split = (int)S; p.slice_tiles = (int)st;
    p.predict_in_force = sh.kernel == 1 && sh.n_units <= PIF_MAX_UNITS;
    const int64_t items = sh.n_units * S;
    // everything the kernels index with int: work items, rows of a partial plane
    if (items > INT_MAX || sh.n_units * sh.unit > INT_MAX) return NB_EINVAL;
    p.waves = (double)items / (double)sh.resident;
    p.grid = sh.kernel == 1 ? (int)std::min<int64_t>((items + WU_WARPS - 1) / WU_WARPS, (int64_t)n_sm * WU_CTAS_PER_SM)
                            : (int)std::min<int64_t>(items, sh.resident);
    *plan = p;
    return NB_OK;
}

int force_internal(nb_ctx* ctx, const int32_t* didx, int64_t n_act)
{
    nb_plan plan;
    const int rc = plan_force(ctx->N, n_act, ctx->n_sm, ctx->max_split, &plan);
    if (rc != NB_OK) return rc;

    ForceArgs A = base_force_args(ctx);
    A.idx = didx;
    A.n_act = (int)n_act;
    A.n_units = plan.n_units; A.n_split = plan.n_split; A.slice_tiles = plan.slice_tiles;
    A.n_tiles = (int)(ctx->Npad / plan.tile);
    A.n_items = plan.n_units * plan.n_split;
    A.ld = plan.kernel == 0 ? plan.n_units * plan.unit : (int)n_act;
    A.slice_minor = nb_slice_minor(nb_reduce_threads(n_act, plan.n_split));

    int launches = 0;
    CU(cudaEventRecord(ctx->ev0, ctx->stream), "event record");
    CU(nb_launch_force(plan, A, eps2_is_zero(ctx->eps), ctx->order, ctx->stream, &launches), "force kernel");
    CU(cudaEventRecord(ctx->ev1, ctx->stream), "event record");
    ctx->ev_valid = true;
    ctx->launches += launches;
    ctx->forced_n = n_act;
    return NB_OK;
}

}  // namespace

extern "C" {

size_t nb_workspace_bytes(int64_t N)
{
    if (N < 1) return 0;
    return Layout(nullptr, pad_n(N)).bytes;
}

int nb_plan_force(int64_t N, int64_t n_act, int n_sm, nb_plan* plan) { return plan_force(N, n_act, n_sm, 0, plan); }

int nb_set_max_split(nb_ctx* ctx, int64_t max_split)
{
    if (!ctx || max_split < 0) return NB_EINVAL;
    ctx->max_split = max_split;
    return NB_OK;
}

int nb_init(nb_ctx** out, int64_t N, const double* m, const double* x, const double* v, double eps, const nb_config* cfg)
{
    if (!out || !cfg || !m || !x || !v || N < 1 || N > (int64_t(1) << 30) || !(eps >= 0.0)) return NB_EINVAL;
    const int k_min = (cfg->k_min == 0 && cfg->k_max == 0) ? -20 : cfg->k_min;
    const int k_max = (cfg->k_min == 0 && cfg->k_max == 0) ? -3 : cfg->k_max;
    if (k_min > k_max || k_min < -1000 || k_max > 1000 || cfg->eta < 0 || cfg->eta_s < 0) return NB_EINVAL;
    if (cfg->order != 0 && cfg->order != 4 && cfg->order != 6 && cfg->order != 8) return NB_EINVAL;
    if (cfg->precision != NB_PREC_FP64 && cfg->precision != NB_PREC_MIXED) return NB_EINVAL;
    if (cfg->precision == NB_PREC_MIXED && cfg->order != 0 && cfg->order != 6) return NB_EINVAL;
    const int64_t Npad = pad_n(N);
    if (!cfg->workspace || ((uintptr_t)cfg->workspace % ALIGN) != 0 || cfg->workspace_bytes < Layout(nullptr, Npad).bytes)
        return NB_ENOMEM;

    nb_ctx* ctx = new (std::nothrow) nb_ctx();
    if (!ctx) return NB_ENOMEM;
    *out = ctx;                       // returned even on NB_ECUDA so that nb_last_error can be read; free with nb_free
    ctx->device = cfg->device;
    ctx->stream = (cudaStream_t)cfg->stream;
    ctx->on_device = cfg->ptrs_on_device != 0;
    ctx->check_idx = cfg->check_indices > 0 || (cfg->check_indices == 0 && !ctx->on_device);
    ctx->N = N; ctx->Npad = Npad; ctx->eps = eps;
    ctx->order = cfg->order == 0 ? 6 : cfg->order;
    ctx->eta = cfg->eta > 0 ? cfg->eta : (ctx->order == 4 ? 0.14 : ctx->order == 8 ? 0.75 : 0.45);
    ctx->eta_s = cfg->eta_s > 0 ? cfg->eta_s : 0.01;
    ctx->k_min = k_min; ctx->k_max = k_max;
    ctx->L = Layout(cfg->workspace, Npad);
    ctx->L.s.order = ctx->order;
    if (cfg->precision != NB_PREC_MIXED) ctx->L.s.recm = nullptr;

    ON_DEVICE(ctx);
    CU(cudaDeviceGetAttribute(&ctx->n_sm, cudaDevAttrMultiProcessorCount, ctx->device), "device attribute");
    CU(nb_force_setup(), "kernel attributes");
    nb_force_occupancy(ctx->order, &ctx->occ_li, &ctx->occ_wu);
    CU(cudaEventCreate(&ctx->ev0), "event");
    CU(cudaEventCreate(&ctx->ev1), "event");
    CU(cudaMemsetAsync(ctx->L.scratch, 0, scratch_bytes(Npad), ctx->stream), "memset scratch");
    CU(cudaMemsetAsync(ctx->L.queue, 0, 64 * sizeof(int), ctx->stream), "memset queue");
    CU(cudaMemsetAsync(ctx->L.steplog, 0, sizeof(unsigned long long), ctx->stream), "memset step log");

    const double *dm = m, *dx = x, *dv = v;
    if (!ctx->on_device) {
        double* st = ctx->L.stage;
        CU(cudaMemcpyAsync(st, m, N * sizeof(double), cudaMemcpyHostToDevice, ctx->stream), "upload m");
        CU(cudaMemcpyAsync(st + Npad, x, 3 * N * sizeof(double), cudaMemcpyHostToDevice, ctx->stream), "upload x");
        CU(cudaMemcpyAsync(st + 4 * Npad, v, 3 * N * sizeof(double), cudaMemcpyHostToDevice, ctx->stream), "upload v");
        dm = st; dx = st + Npad; dv = st + 4 * Npad;
    }
    CU(nb_launch_init_state(ctx->L.s, N, Npad, dm, dx, dv, ctx->stream), "init_state");
    ctx->launches += 1;

    // startup (reading R8): two all-active evaluations at t = 0 (one at the 4th order).  The 8th order needs no third:
    // a and jerk are complete after pass 1, so pass 2 - whose records carry them - yields snap AND crackle (R22).
    for (int pass = 1; pass <= (ctx->order == 4 ? 1 : 2); ++pass) {
        CU(nb_launch_predict(ctx->L.s, N, 0.0, true, ctx->stream), "predict");
        ctx->launches += 1;
        ctx->predicted = true; ctx->t_pred = 0.0;
        const int rc = force_internal(ctx, nullptr, N);
        if (rc != NB_OK) return rc;
        CU(nb_launch_startup(ctx->L.s, N, ctx->L.fa, ctx->L.fj, ctx->L.fs, pass, ctx->eta_s, k_min, k_max, ctx->stream), "startup");
        ctx->launches += 1;
    }
    ctx->predicted = false; ctx->forced_n = -1;
    if (!ctx->on_device) CU(cudaStreamSynchronize(ctx->stream), "nb_init");
    return NB_OK;
}

int nb_predict(nb_ctx* ctx, double t)
{
    if (!ctx || !std::isfinite(t)) return NB_EINVAL;
    ON_DEVICE(ctx);
    CU(nb_launch_predict(ctx->L.s, ctx->N, t, false, ctx->stream), "predict");
    ctx->launches += 1;
    ctx->t_pred = t; ctx->predicted = true; ctx->forced_n = -1;
    return NB_OK;
}

int nb_force(nb_ctx* ctx, const int32_t* active_idx, int64_t n_act, double* a, double* jerk, double* snap, double* pot)
{
    if (!ctx || n_act < 0 || n_act > ctx->N) return NB_EINVAL;
    if (active_idx == nullptr && n_act != 0 && n_act != ctx->N) return NB_EINVAL;
    if (!ctx->predicted) return NB_ESTATE;
    if (n_act == 0) { ctx->forced_n = 0; return NB_OK; }
    ON_DEVICE(ctx);

    const int32_t* didx = nullptr;
    int rc = resolve_idx(ctx, active_idx, n_act, ctx->L.idx_user, &didx);
    if (rc != NB_OK) return rc;
    if ((rc = force_internal(ctx, didx, n_act)) != NB_OK) return rc;

    if ((rc = copy_out(ctx, a, ctx->L.fa, 3 * n_act)) != NB_OK) return rc;
    if ((rc = copy_out(ctx, jerk, ctx->L.fj, 3 * n_act)) != NB_OK) return rc;
    if ((rc = copy_out(ctx, snap, ctx->L.fs, 3 * n_act)) != NB_OK) return rc;
    if ((rc = copy_out(ctx, pot, ctx->L.fp, n_act)) != NB_OK) return rc;
    if (!ctx->on_device) CU(cudaStreamSynchronize(ctx->stream), "nb_force");
    return NB_OK;
}

int nb_force_crackle(nb_ctx* ctx, double* crackle)
{
    if (!ctx || !crackle) return NB_EINVAL;
    if (ctx->order != 8 || ctx->forced_n < 0) return NB_ESTATE;
    ON_DEVICE(ctx);
    const int rc = copy_out(ctx, crackle, ctx->L.fc, 3 * (size_t)ctx->forced_n);
    if (rc != NB_OK) return rc;
    if (!ctx->on_device) CU(cudaStreamSynchronize(ctx->stream), "nb_force_crackle");
    return NB_OK;
}

int nb_corrector(nb_ctx* ctx, const int32_t* active_idx, int64_t n_act, double dt)
{
    if (!ctx || n_act < 0 || n_act > ctx->N || !(dt == dt)) return NB_EINVAL;
    if (active_idx == nullptr && n_act != 0 && n_act != ctx->N) return NB_EINVAL;
    if (ctx->forced_n < 0 || ctx->forced_n != n_act) return NB_ESTATE;
    ON_DEVICE(ctx);
    if (n_act > 0) {
        const int32_t* didx = nullptr;
        const int rc = resolve_idx(ctx, active_idx, n_act, ctx->L.idx_user, &didx);
        if (rc != NB_OK) return rc;
        CU(nb_launch_corrector(ctx->L.s, didx, n_act, dt, ctx->t_pred, ctx->L.fa, ctx->L.fj, ctx->L.fs, ctx->eta, ctx->k_min,
                               ctx->k_max, ctx->stream), "corrector");
        ctx->launches += 1;
    }
    ctx->predicted = false; ctx->forced_n = -1; ctx->sched_n = -1;
    if (!ctx->on_device) CU(cudaStreamSynchronize(ctx->stream), "nb_corrector");
    return NB_OK;
}

int nb_next_block(nb_ctx* ctx, double* t_next, int32_t* active_idx, int64_t* n_act)
{
    if (!ctx || !t_next || !n_act) return NB_EINVAL;
    ON_DEVICE(ctx);
    int launches = 0;
    CU(nb_launch_next_block(ctx->L.s, ctx->N, ctx->L.idx_sched, ctx->L.idx_tmp, ctx->L.scratch, ctx->stream, &launches), "scheduler");
    ctx->launches += launches;
    struct { double t; long long n; } res;
    CU(cudaMemcpyAsync(&res, ctx->L.scratch, sizeof res, cudaMemcpyDeviceToHost, ctx->stream), "scheduler result");
    CU(cudaStreamSynchronize(ctx->stream), "nb_next_block");
    *t_next = res.t; *n_act = res.n; ctx->sched_n = res.n;
    if (active_idx && res.n > 0) {
        CU(cudaMemcpyAsync(active_idx, ctx->L.idx_sched, res.n * sizeof(int32_t),
                           ctx->on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, ctx->stream), "active list");
        if (!ctx->on_device) CU(cudaStreamSynchronize(ctx->stream), "nb_next_block");
    }
    return NB_OK;
}

int nb_run_blocks(nb_ctx* ctx, double t_end, int64_t max_steps, int64_t* steps_done, double* t_last, int64_t* sum_n_act)
{
    if (!ctx || !(t_end == t_end) || max_steps < 0) return NB_EINVAL;
    ON_DEVICE(ctx);
    if (!ctx->step_graph) {
        const int rc = build_step_graph(ctx);
        if (rc != NB_OK) return rc;
    }
    DevPlan h{};
    h.t_end = t_end; h.steps_left = max_steps; h.t_last = -1.0; h.max_split = ctx->max_split;
    CU(cudaMemcpyAsync(ctx->L.devplan, &h, sizeof h, cudaMemcpyHostToDevice, ctx->stream), "upload step control");
    ctx->predicted = false; ctx->forced_n = -1; ctx->sched_n = -1;
    // The host cannot know when the device stops, so it enqueues batches of steps and looks at the counters after each;
    // steps enqueued after the stop flag is up return at once (every kernel checks it).
    int64_t enqueued = 0;                                   // block steps enqueued so far
    int batch = 1;                                          // graph replays per batch (STEPS_PER_GRAPH block steps each)
    while (max_steps > 0) {
        const int64_t n = std::min<int64_t>(batch, (max_steps - enqueued + STEPS_PER_GRAPH - 1) / STEPS_PER_GRAPH);
        for (int64_t k = 0; k < n; ++k) CU(cudaGraphLaunch(ctx->step_graph, ctx->stream), "block-step graph launch");
        enqueued += n * STEPS_PER_GRAPH;
        ctx->launches += n * STEP_GRAPH_KERNELS * STEPS_PER_GRAPH;
        CU(cudaMemcpyAsync(&h, ctx->L.devplan, sizeof h, cudaMemcpyDeviceToHost, ctx->stream), "read step control");
        CU(cudaStreamSynchronize(ctx->stream), "nb_run_blocks");
        if (h.stop || enqueued >= max_steps) break;
        if (batch < 16) batch *= 2;
    }
    if (steps_done) *steps_done = h.steps_done;
    if (t_last) *t_last = h.t_last;
    if (sum_n_act) *sum_n_act = h.sum_act;
    return NB_OK;
}

static int field_width_host(int f) { return (f == NB_M || f == NB_T || f == NB_DT) ? 1 : 3; }

int nb_get_state(nb_ctx* ctx, int field, const int32_t* idx, int64_t n, double* out)
{
    if (!ctx || !out || n < 0 || n > ctx->N || field < NB_M || field > NB_JP) return NB_EINVAL;
    if (n == 0) return NB_OK;
    ON_DEVICE(ctx);
    const int32_t* didx = nullptr;
    const int rc = resolve_idx(ctx, idx, n, ctx->L.idx_tmp, &didx, /*unique=*/false);
    if (rc != NB_OK) return rc;
    const size_t count = (size_t)n * field_width_host(field);
    double* dst = ctx->on_device ? out : ctx->L.stage;
    CU(nb_launch_get(ctx->L.s, field, didx, n, dst, ctx->stream), "get_state");
    ctx->launches += 1;
    if (!ctx->on_device) {
        CU(cudaMemcpyAsync(out, dst, count * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream), "get_state copy");
        CU(cudaStreamSynchronize(ctx->stream), "nb_get_state");
    }
    return NB_OK;
}

int nb_set_state(nb_ctx* ctx, int field, const int32_t* idx, int64_t n, const double* in)
{
    if (!ctx || !in || n < 0 || n > ctx->N || field < NB_M || (field > NB_DT && field != NB_A4 && field != NB_A5)) return NB_EINVAL;
    if (n == 0) return NB_OK;
    ON_DEVICE(ctx);
    const int32_t* didx = nullptr;
    const int rc = resolve_idx(ctx, idx, n, ctx->L.idx_tmp, &didx);
    if (rc != NB_OK) return rc;
    const size_t count = (size_t)n * field_width_host(field);
    const double* src = in;
    if (!ctx->on_device) {
        CU(cudaMemcpyAsync(ctx->L.stage, in, count * sizeof(double), cudaMemcpyHostToDevice, ctx->stream), "set_state copy");
        src = ctx->L.stage;
    }
    CU(nb_launch_set(ctx->L.s, field, didx, n, src, ctx->stream), "set_state");
    ctx->launches += 1;
    ctx->predicted = false; ctx->forced_n = -1; ctx->sched_n = -1;
    if (!ctx->on_device) CU(cudaStreamSynchronize(ctx->stream), "nb_set_state");
    return NB_OK;
}

int nb_energy(nb_ctx* ctx, double* kinetic, double* potential)
{
    if (!ctx || !kinetic || !potential) return NB_EINVAL;
    ON_DEVICE(ctx);
    CU(nb_launch_predict(ctx->L.s, ctx->N, 0.0, true, ctx->stream), "predict");
    ctx->launches += 1;
    ctx->predicted = true;
    const int rc = force_internal(ctx, nullptr, ctx->N);
    if (rc != NB_OK) return rc;
    int launches = 0;
    CU(nb_launch_energy(ctx->L.s, ctx->N, ctx->L.fp, (double*)ctx->L.scratch + 16, ctx->stream, &launches), "energy");
    ctx->launches += launches;
    double res[2];
    CU(cudaMemcpyAsync(res, (double*)ctx->L.scratch + 16, sizeof res, cudaMemcpyDeviceToHost, ctx->stream), "energy result");
    CU(cudaStreamSynchronize(ctx->stream), "nb_energy");
    *kinetic = res[0]; *potential = res[1];
    ctx->predicted = false; ctx->forced_n = -1;
    return NB_OK;
}

int nb_check_indices(nb_ctx* ctx, const int32_t* idx, int64_t n, int unique)
{
    if (!ctx || n < 0 || (n > 0 && !idx) || idx == NB_ACTIVE_INTERNAL) return NB_EINVAL;
    if (n == 0) return NB_OK;
    if (n > ctx->N) return NB_EINVAL;                       // no call of this library takes a longer list
    ON_DEVICE(ctx);
    const int32_t* didx = idx;
    if (!ctx->on_device) {
        CU(cudaMemcpyAsync(ctx->L.idx_tmp, idx, n * sizeof(int32_t), cudaMemcpyHostToDevice, ctx->stream), "upload indices");
        didx = ctx->L.idx_tmp;
    }
    return verify_idx(ctx, didx, n, unique != 0);
}

int64_t nb_step_log(nb_ctx* ctx, int64_t capacity, int64_t* n_act, double* t_us)
{
    if (!ctx || capacity < 0 || (capacity > 0 && (!n_act || !t_us))) return NB_EINVAL;
    DeviceGuard guard(ctx->device);
    if (guard.err != cudaSuccess) return NB_ECUDA;
    static_assert(sizeof(unsigned long long) == 8, "log entries are 64-bit");
    unsigned long long* h = new (std::nothrow) unsigned long long[1 + 2 * NB_STEP_LOG];
    if (!h) return NB_ENOMEM;
    int64_t n = NB_ECUDA;
    if (cudaMemcpyAsync(h, ctx->L.steplog, (1 + 2 * NB_STEP_LOG) * sizeof(unsigned long long), cudaMemcpyDeviceToHost, ctx->stream) == cudaSuccess &&
        cudaStreamSynchronize(ctx->stream) == cudaSuccess) {
        const unsigned long long total = h[0];
        n = (int64_t)std::min<unsigned long long>(std::min<unsigned long long>(total, NB_STEP_LOG), (unsigned long long)capacity);
        for (int64_t k = 0; k < n; ++k) {                   // the last n steps, oldest first
            const unsigned long long pos = (total - (unsigned long long)n + (unsigned long long)k) % NB_STEP_LOG;
            n_act[k] = (int64_t)h[1 + 2 * pos];
            t_us[k] = (double)(h[2 + 2 * pos] - h[2 + 2 * ((total - (unsigned long long)n) % NB_STEP_LOG)]) * 1e-3;
        }
    }
    delete[] h;
    return n;
}

int nb_resident_ctas(const nb_ctx* ctx, int kernel)
{
    if (!ctx || kernel < 0 || kernel > 1) return NB_EINVAL;
    return kernel == 0 ? ctx->occ_li : ctx->occ_wu;
}

int64_t nb_launch_count(const nb_ctx* ctx) { return ctx ? ctx->launches : 0; }

double nb_last_force_ms(nb_ctx* ctx)
{
    if (!ctx || !ctx->ev_valid) return -1.0;
    DeviceGuard guard(ctx->device);
    float ms = 0;
    if (cudaEventSynchronize(ctx->ev1) != cudaSuccess) return -1.0;
    if (cudaEventElapsedTime(&ms, ctx->ev0, ctx->ev1) != cudaSuccess) return -1.0;
    return (double)ms;
}

const char* nb_strerror(int status)
{
    switch (status) {
        case NB_OK: return "ok";
        case NB_EINVAL: return "invalid argument";
        case NB_ENOMEM: return "workspace missing, misaligned or too small";
        case NB_ESTATE: return "call order: nb_predict -> nb_force -> nb_corrector";
        case NB_ECUDA: return "CUDA error (see nb_last_error)";
        default: return "unknown status";
    }
}

const char* nb_last_error(const nb_ctx* ctx) { return ctx ? ctx->err : ""; }

void nb_free(nb_ctx* ctx)
{
    if (!ctx) return;
    DeviceGuard guard(ctx->device);
    if (ctx->ev0) cudaEventDestroy(ctx->ev0);
    if (ctx->ev1) cudaEventDestroy(ctx->ev1);
    if (ctx->step_graph) cudaGraphExecDestroy(ctx->step_graph);
    delete ctx;
}

}  // extern "C"
