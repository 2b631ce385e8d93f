"""The WHOLE library on the host, without a GPU: nb_api.cu, nb_force.cu and nb_step.cu are compiled with g++ against a stand-in
for the CUDA runtime (tests/host/simt/cuda_runtime.h: one CUDA thread = one fibre, CTAs one after the other, shuffles / votes /
barriers / mbarriers with their CUDA meaning, stream capture and graph replay) and driven through their real C ABI with numpy
buffers.  What is compared with the oracle here is therefore the STRUCTURE of the CUDA path - launch plans, the work queue, the
j-split, tile staging, lanes-over-i to lanes-over-j warp units, the shuffle butterfly, the partial-sum layouts and the
fixed-order reduction, predict-in-force, the one-kernel scheduler, the device-planned block step and its CUDA graph - which
tests/test_kernel_source_cpu.py (the formulas alone) cannot see and which otherwise only the `-m gpu` tests exercise.

The sources are taken as they are, except for what cannot be C++: `K<<<grid, block, smem, stream>>>(args)` becomes
simt::launch(K, grid, block, smem, stream, args); the helpers of nb_force.cu that are inline PTX (fma / mul with fixed operand
order, the rsqrt seeds, mbarrier and bulk-copy wrappers, the register ballast) are removed and tests/host/simt/nb_force_shims.h
supplies their C++ meaning; `extern __shared__` becomes a static array; %globaltimer becomes a counter.  The test asserts that
every one of these edits found its target.

NOT a product path: nothing under paper_1411_5234_b200/ refers to this; binding.System still refuses to run without a CUDA
device.  Not covered: the machine code, timing, the memory model of truly concurrent CTAs.  CTAs run one after the other here,
but in any order the test asks for, threads are resumed in any order, bulk copies land early or late, shared memory and the workspace
start out as garbage (the switches are listed at the top of tests/host/simt/cuda_runtime.h); NB_SIMT_CXXFLAGS builds the library with
a sanitizer (profiles/r02_sanitizer.md).
"""
import ctypes as C
import os
import re
import shlex
import subprocess

import numpy as np
import pytest

from paper_1411_5234_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
CSRC = os.path.join(ROOT, "paper_1411_5234_b200", "csrc")
SIMT = os.path.join(ROOT, "tests", "host", "simt")
TOL = 1e-11


# ---------------------------------------------------------------------------------------------------------------
# the edits
# ---------------------------------------------------------------------------------------------------------------
def strip_function(text, signature, replacement=""):
    """remove the definition that starts with `signature` (up to the brace that closes its body)"""
    assert text.count(signature) == 1, signature
    i = text.index(signature)
    j = text.index("{", i + len(signature))
    depth = 0
    for k in range(j, len(text)):
        depth += text[k] == "{"
        depth -= text[k] == "}"
        if depth == 0:
            return text[:i] + replacement + text[k + 1:]
    raise AssertionError(signature)


LAUNCH = re.compile(r"([A-Za-z_]\w*(?:<[^<>()]*>)?)<<<([^;]*?)>>>\(")


def to_host_source(name, text):
    n_launch = len(re.findall(r"<<<", text))
    text, n = LAUNCH.subn(r"simt::launch(\1, \2, ", text)
    assert n == n_launch, (name, n, n_launch)
    if name == "nb_force.cu":
        for sig in ("__device__ __forceinline__ double F(double a, double b, double c)",
                    "__device__ __forceinline__ double M(double a, double b)",
                    "__device__ __forceinline__ double rsqrt_seed(double s)",
                    "__device__ __forceinline__ float rsqrt_f32(float s)",
                    "__device__ __forceinline__ uint32_t smem_u32(const void* p)",
                    "__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)",
                    "__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)",
                    "__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar)",
                    "__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)"):
            text = strip_function(text, sig)
        text = strip_function(text, "template <int N>\n__device__ __forceinline__ void reg_ballast(const ForceArgs& A)",
                              "template <int N>\ninline void reg_ballast(const ForceArgs&) {}")
        lines, out, skip = text.split("\n"), [], False
        n_macros = 0
        for l in lines:
            if skip:
                skip = l.rstrip().endswith("\\")
                continue
            if re.match(r"#define V(SUB|ADD|MUL|FMA|FNMA|RSQ|TWICE)\(", l):
                n_macros += 1
                skip = l.rstrip().endswith("\\")
                continue
            out.append(l)
        assert n_macros == 7
        text = "\n".join(out)
        fence = '        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");\n'
        assert text.count(fence) == 1
        text = text.replace(fence, "")
        dyn = "extern __shared__ __align__(128) double2 dyn_smem[];"
        assert text.count(dyn) == 1
        text = text.replace(dyn, "alignas(128) static double2 dyn_smem[16384];      // 256 KiB: more than any kernel asks for\n"
                                 "static const int dyn_smem_registered = simt::register_dyn_smem(dyn_smem, sizeof dyn_smem);   // bounds per launch under ASan")
        inc = '#include "nb_internal.h"\n'
        assert text.count(inc) == 1
        text = text.replace(inc, inc + '#include "nb_force_shims.h"\n')
    if name == "nb_api.cu":
        # test-only switch of the HOST COPY: nb_init without its all-active startup evaluations, so that the plans of large N
        # with few active particles (config 5) can be run on the host in seconds; a, jerk, snap are then 0 and dt is not set
        loop = "for (int pass = 1; pass <= (ctx->order == 4 ? 1 : 2); ++pass) {"
        assert text.count(loop) == 1
        text = text.replace(loop, 'for (int pass = 1; pass <= (getenv("NB_SIMT_SKIP_STARTUP") ? 0 : ctx->order == 4 ? 1 : 2); ++pass) {')
    if name == "nb_step.cu":
        timer = 'asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(now));'
        assert text.count(timer) == 1
        text = text.replace(timer, "now = simt::clock_ns();")
    # every static shared array with a single declarator registers itself with the stand-in, which fills it with 0xFF bytes before
    # every CTA (a CTA finds garbage in shared memory on the GPU, not zeros and not its predecessor's values)
    text, n_reg = re.subn(r"^(\s*)__shared__ ((?:alignas\(8\) )?[\w ]+?) (\w+)((?:\[\w+\])*);[ \t]*$",
                          r"\1__shared__ \2 \3\4; static const int \3_registered_ = simt::register_smem(&\3, sizeof \3);", text, flags=re.M)
    assert n_reg == {"nb_force.cu": 7, "nb_step.cu": 6}.get(name, 0), (name, n_reg)
    text = text.replace("__shared__ alignas(8)", "alignas(8) __shared__")      # g++ wants the attribute before `static`
    assert not re.search(r"\basm\b", re.sub(r"//.*", "", text)), name
    return text


@pytest.fixture(scope="module")
def SIM(tmp_path_factory):
    from paper_1411_5234_b200 import binding as B
    out = str(tmp_path_factory.mktemp("simt_host"))
    srcs = []
    for name in ("nb_api.cu", "nb_force.cu", "nb_step.cu"):
        text = to_host_source(name, open(os.path.join(CSRC, name)).read())
        path = os.path.join(out, name.replace(".cu", "_host.cpp"))
        open(path, "w").write(text)
        srcs.append(path)
    so = os.path.join(out, "libnb_simt_host.so")
    cmd = ["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-w", "-U_FORTIFY_SOURCE", "-D_FORTIFY_SOURCE=0", "-shared", "-fPIC", "-I" + SIMT, "-I" + CSRC,
           "-I" + os.path.join(ROOT, "include")] + srcs + [os.path.join(SIMT, "simt_switch.S"), "-o", so]
    # NB_SIMT_CXXFLAGS: extra compiler flags for a one-off run, e.g. "-fsanitize=undefined -fno-sanitize-recover=undefined -g"
    # (UBSan over the kernels' index arithmetic, shifts and alignment; profiles/r02_sanitizer.md)
    cmd[1:1] = shlex.split(os.environ.get("NB_SIMT_CXXFLAGS", ""))
    r = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    assert r.returncode == 0, r.stdout[-6000:]
    L = C.CDLL(so)
    ref = B.lib()                                            # the real library: only its ctypes signatures are taken from it
    for name in B.EXPORTS:
        f, g = getattr(L, name), getattr(ref, name)
        f.argtypes, f.restype = g.argtypes, g.restype

    class HostSimSystem(B.System):
        """binding.System's marshalling over the host build: numpy workspace (between two bands of 0xA5), host pointers"""

        def __init__(self, m, x, v, eps, n_sms=148, eta=0.0, eta_s=0.0, k_min=0, k_max=0, order=0, check_indices=0, precision=0,
                     guard_bytes=1 << 16, skip_startup=False, device_ptrs=False):
            os.environ["NB_SIMT_SMS"] = str(n_sms)
            os.environ.pop("NB_SIMT_SKIP_STARTUP", None)
            if skip_startup: os.environ["NB_SIMT_SKIP_STARTUP"] = "1"
            self.L, self.host, self.device, self.N, self.ctx = L, True, 0, int(m.shape[0]), C.c_void_p()
            nbytes = L.nb_workspace_bytes(self.N)
            self._guard = (int(guard_bytes) + 255) // 256 * 256
            self.workspace = np.full(nbytes + 256 + 2 * self._guard, 0xFF, dtype=np.uint8)      # the library gets NaNs and index -1:
            self.workspace[:self._guard + 256] = 0xA5                                           # whatever it reads before writing shows
            self.workspace[-(self._guard + 256):] = 0xA5
            base = (self.workspace.ctypes.data + self._guard + 255) // 256 * 256
            self._ws_off, self._ws_bytes = base - self.workspace.ctypes.data, nbytes
            # device_ptrs: the context is told that (h/d) pointers are DEVICE pointers (no staging copies, no synchronisation, index
            # lists unverified unless asked for); on the host build device memory is host memory, so numpy arrays serve as both
            self.cfg = B.nb_config(0, None, C.c_void_p(base), nbytes, 1 if device_ptrs else 0, eta, eta_s, k_min, k_max, order, check_indices,
                                   precision)
            m, x, v = self._in(m, (self.N,)), self._in(x, (self.N, 3)), self._in(v, (self.N, 3))
            self._check(L.nb_init(C.byref(self.ctx), self.N, B._ptr(m), B._ptr(x), B._ptr(v), float(eps), C.byref(self.cfg)))

        def guards_intact(self):
            lo, hi = self.workspace[:self._ws_off], self.workspace[self._ws_off + self._ws_bytes:]
            return bool((lo == 0xA5).all()) and bool((hi == 0xA5).all())

    return HostSimSystem


def relvec(g, o):
    return np.linalg.norm(g - o, axis=-1) / np.linalg.norm(o, axis=-1)


def assert_force_parity(g, o, tol=TOL):
    for name, a, b in zip(("acc", "jerk", "snap"), g[:3], o[:3]):
        assert relvec(a, b).max() <= tol, (name, relvec(a, b).max())
    assert np.abs(g[3] / o[3] - 1).max() <= tol, ("pot", np.abs(g[3] / o[3] - 1).max())


# ---------------------------------------------------------------------------------------------------------------
# config 1 through the host build: startup, one evaluation, eight shared steps
# ---------------------------------------------------------------------------------------------------------------
def test_config1_startup_force_and_steps(SIM, oracle):
    c, m, x, v = W.config_inputs(1)
    g = SIM(m, x, v, c.eps)
    o = oracle.OracleSystem(m, x, v, c.eps)
    for f, ref in (("A", o.a), ("J", o.j), ("S", o.s)):
        assert relvec(g.nb_get_state(f), ref).max() <= TOL
    assert np.array_equal(g.nb_get_state("DT"), o.dt)
    g.nb_predict(0.0); o.predict(0.0)
    assert_force_parity(g.nb_force(), o.force())
    for _ in range(8):
        t = o.t[0] + c.dt
        g.nb_predict(t); g.nb_force(outputs=False); g.nb_corrector(None, c.dt)
        o.shared_step(c.dt)
    assert np.abs(g.nb_get_state("X") - o.x).max() <= 1e-13 and np.abs(g.nb_get_state("V") - o.v).max() <= 1e-12
    Kg, Wg = g.nb_energy()
    Ko, Wo = o.energy()
    assert abs((Kg + Wg) - (Ko + Wo)) / abs(Ko + Wo) <= 1e-10
    assert g.guards_intact()
    g.nb_free()


def oracle_on_records(oracle, g, eps, idx):
    """O1 on the predicted records the kernels read (nb_force is a pure function of them)"""
    m, xp, vp, ap = g.nb_get_state("M"), g.nb_get_state("XP"), g.nb_get_state("VP"), g.nb_get_state("AP")
    return oracle.hermite6.force(m, xp, vp, ap, eps, idx)


# ---------------------------------------------------------------------------------------------------------------
# every kernel shape: warp units of every width (lanes over i ... lanes over j), padded and decomposed rests, ragged CTA
# tiles, the j-split with its two partial-sum layouts and the reduction, on a "device" of 148 SMs and on one of 3
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("N,eps,masses,n_sms", [(1500, 1e-3, "equal", 148), (1027, 0.0, "kroupa", 3), (2, 0.0, "equal", 148), (257, 0.0, "kroupa", 148)])
def test_force_shapes_and_active_sets(SIM, oracle, N, eps, masses, n_sms):
    from paper_1411_5234_b200 import binding as B
    m, x, v = W.plummer(N, 1000 + N, masses)
    g = SIM(m, x, v, eps, n_sms=n_sms)
    g.nb_predict(2.0 ** -9); g.nb_force(outputs=False); g.nb_corrector(None, 2.0 ** -9)     # all derivatives non-zero, D != 0 next
    g.nb_predict(2.0 ** -9 + 2.0 ** -11)
    rng = np.random.default_rng(N)
    sizes = sorted({1, 2, 3, 5, 7, 9, 16, 17, 21, 24, 31, 33, 64, 97, 129, 255, 256, 300, 512, 1023, 1024, N} & set(range(1, N + 1)) | {N})
    shapes = set()
    for n_act in sizes:
        idx = None if n_act == N else rng.choice(N, n_act, replace=False).astype(np.int32)
        assert_force_parity(g.nb_force(idx), oracle_on_records(oracle, g, eps, idx))
        p = B.nb_plan_force(N, n_act, n_sms)
        workers = min(p.n_units * p.n_split, n_sms * 4) if p.kernel == 0 else 4 * min((p.n_units * p.n_split + 3) // 4, n_sms * 4)
        shapes.add((p.kernel, p.n_split > 1, p.n_units * p.n_split > workers))
    if N >= 1024:                                             # both kernels, split launches, and (3 SMs) the work queue in both
        assert {k for k, _, _ in shapes} == {0, 1} and True in {sp for _, sp, _ in shapes}
        if n_sms == 3: assert {k for k, _, q in shapes if q} == {0, 1}
    perm = rng.permutation(N).astype(np.int32)                # permuted full list: row k <-> idx[k]
    assert_force_parity(g.nb_force(perm), oracle_on_records(oracle, g, eps, perm))
    # no j-split at all (the paper's "Bfactor off" arm): same results to rounding
    g.nb_set_max_split(1)
    idx = rng.choice(N, min(N, 37), replace=False).astype(np.int32)
    assert_force_parity(g.nb_force(idx), oracle_on_records(oracle, g, eps, idx))
    assert g.guards_intact()
    g.nb_free()


# ---------------------------------------------------------------------------------------------------------------
# block steps: the one-kernel scheduler bit for bit, predictor / corrector / levels after every step
# ---------------------------------------------------------------------------------------------------------------
def test_block_steps_against_oracle(SIM, oracle):
    N, eps = 384, 1e-3
    m, x, v = W.plummer(N, 77, "kroupa")
    g = SIM(m, x, v, eps)
    o = oracle.OracleSystem(m, x, v, eps)
    assert np.array_equal(g.nb_get_state("DT"), o.dt)
    n_steps = 0
    while True:
        tg, ng, actg = g.nb_next_block()
        to, acto = o.next_block()
        assert tg == to and ng == acto.size and np.array_equal(actg, acto)
        if to > 2.0 ** -5: break
        g.nb_predict(tg); o.predict(to)
        for f, ref in (("XP", o.xp), ("VP", o.vp), ("AP", o.ap)):
            assert relvec(g.nb_get_state(f), ref).max() <= 1e-12, f
        assert_force_parity(g.nb_force(actg), o.force(acto), 1e-10)
        g.nb_corrector(actg, 0.0); o.corrector(acto, 0.0)
        assert np.array_equal(g.nb_get_state("T"), o.t) and np.array_equal(g.nb_get_state("DT"), o.dt)
        n_steps += 1
    assert n_steps > 20
    assert relvec(g.nb_get_state("X"), o.x).max() <= 1e-12 and relvec(g.nb_get_state("V"), o.v).max() <= 1e-11
    g.nb_free()


@pytest.mark.parametrize("N,eps,masses,n_sms", [(1200, 1e-4, "kroupa", 148), (300, 0.0, "equal", 5)])
def test_run_blocks_is_bitwise_the_separate_calls(SIM, N, eps, masses, n_sms):
    """nb_run_blocks (scheduler + plan on the device, predict-in-force, reduction + corrector in one kernel, the captured graph)
    against the same steps call by call: identical schedules, bit-identical states; step budget and t_end respected"""
    m, x, v = W.plummer(N, 77 + N, masses)
    g1, g2 = SIM(m, x, v, eps, n_sms=n_sms), SIM(m, x, v, eps, n_sms=n_sms)
    t_end = 2.0 ** -6
    steps, acts = 0, 0
    while True:
        t, n, act = g1.nb_next_block()
        if t > t_end: break
        g1.nb_predict(t); g1.nb_force(act, outputs=False); g1.nb_corrector(act, 0.0)
        steps += 1; acts += n
    assert steps >= 10
    s_a, t_a, n_a = g2.nb_run_blocks(t_end, max_steps=5)
    assert s_a == 5 and t_a > 0
    s_b, t_b, n_b = g2.nb_run_blocks(t_end / 2)
    assert t_b <= t_end / 2
    s_c, t_c, n_c = g2.nb_run_blocks(t_end)
    assert s_a + s_b + s_c == steps and n_a + n_b + n_c == acts and t_c == t_end
    assert g2.nb_run_blocks(t_end) == (0, -1.0, 0)
    for f in ("X", "V", "A", "J", "S", "C", "T", "DT"):
        assert np.array_equal(g1.nb_get_state(f), g2.nb_get_state(f)), f
    na, _ = g2.nb_step_log()
    assert na.size == steps and na.sum() == acts               # the device's own record of the steps
    t1, n1, a1 = g1.nb_next_block(); t2, n2, a2 = g2.nb_next_block()
    assert t1 == t2 and np.array_equal(a1, a2)
    assert g1.guards_intact() and g2.guards_intact()
    g1.nb_free(); g2.nb_free()


# ---------------------------------------------------------------------------------------------------------------
# config 5's plans on the host: N = 2^18 with a handful of active particles (one or two warp units x 1024-2048 slices; a whole
# reduction block per particle and the [component][row][slice] layout of the partial sums, which small N never reaches)
# ---------------------------------------------------------------------------------------------------------------
def reduce_threads(n_act, S):
    """nb_plan.h:nb_reduce_threads restated - ONLY to assert which reduction shape a case exercised"""
    T = 1
    while T < 256 and T * 4 <= S and n_act * T < (1 << 18): T *= 2
    return T


def test_large_n_small_active_sets(SIM, oracle):
    from paper_1411_5234_b200 import binding as B
    N, eps = 1 << 18, 1e-4
    m, x, v = W.plummer(N, W.BASE_SEED + 4, "equal")
    g = SIM(m, x, v, eps, skip_startup=True)                 # (the startup's 1.4e11 pairs are not for the host)
    rng = np.random.default_rng(5)
    a = rng.normal(size=(N, 3))
    g.nb_set_state("A", a)
    g.nb_predict(0.0)                                        # t_i = 0: the records are x, v and the a just set
    for n_act in (1, 3, 8, 24):
        idx = W.active_set(N, n_act, 50 + n_act)
        assert_force_parity(g.nb_force(idx), oracle.hermite6.force(m, x, v, a, eps, idx))
        p = B.nb_plan_force(N, n_act, 148)
        assert p.kernel == 1 and p.n_split >= 1024 and reduce_threads(n_act, p.n_split) == 256     # a reduction block per particle
    assert g.guards_intact()
    g.nb_free()


# ---------------------------------------------------------------------------------------------------------------
# the other orders (nb_config.order = 4 / 8, readings R21 / R22) through the host build: their startups (one pass; two passes
# with snap and crackle from the second), 80-B / 112-B records, 7 / 13 partial sums per particle in every kernel shape, the
# crackle output, shared steps, and block steps call by call against nb_run_blocks (bitwise)
# ---------------------------------------------------------------------------------------------------------------
def force_any_order(oracle, g, order, eps, idx):
    """the oracle's sums on the predicted records the kernels read: (a, jerk, snap, pot, crackle or None)"""
    m, rec = g.nb_get_state("M"), [g.nb_get_state(f) for f in ("XP", "VP", "AP")]
    if order == 8:
        a, j, s, c, p = oracle.hermite6.force8(m, *rec, g.nb_get_state("JP"), eps, idx)
        return a, j, s, p, c
    return oracle.hermite6.force(m, *rec, eps, idx) + (None,)


@pytest.mark.parametrize("order,n_sms", [(4, 148), (8, 148), (8, 3)])
def test_other_orders_startup_shapes_and_steps(SIM, oracle, order, n_sms):
    N, eps, dt = 700, 1e-3, 2.0 ** -9
    m, x, v = W.plummer(N, 4000 + order, "kroupa")
    g = SIM(m, x, v, eps, order=order, n_sms=n_sms)
    o = oracle.OracleSystem(m, x, v, eps, order=order)
    started = ("A", "J") if order == 4 else ("A", "J", "S", "C")
    for f in started:
        assert relvec(g.nb_get_state(f), getattr(o, f.lower())).max() <= TOL, f
    for f in {"S", "C", "A4", "A5"} - set(started) - ({"A4", "A5"} if order == 4 else set()):
        assert not g.nb_get_state(f).any(), f
    assert np.array_equal(g.nb_get_state("DT"), o.dt)
    rng = np.random.default_rng(order)
    for step in (1, 2, 3):
        g.nb_predict(step * dt); o.predict(step * dt)
        assert relvec(g.nb_get_state("XP"), o.xp).max() <= 1e-12 and relvec(g.nb_get_state("VP"), o.vp).max() <= 1e-11
        if step == 2:                                         # every kernel shape on identical records
            for n_act in (1, 3, 7, 16, 17, 33, 97, 300, 512, N):
                idx = None if n_act == N else rng.choice(N, n_act, replace=False).astype(np.int32)
                ga, gj, gs, gp = g.nb_force(idx)
                oa, oj, os_, op, oc = force_any_order(oracle, g, order, eps, idx)
                assert relvec(ga, oa).max() <= TOL and relvec(gj, oj).max() <= TOL and np.abs(gp / op - 1).max() <= TOL, n_act
                if order == 4:
                    assert not gs.any()                       # snap is not evaluated at this order
                else:
                    assert relvec(gs, os_).max() <= TOL and relvec(g.nb_force_crackle(n_act), oc).max() <= TOL, n_act
        g.nb_force(outputs=False); o.force()
        g.nb_corrector(None, dt); o.corrector(None, dt)
    for f, ref, tol in (("X", o.x, 1e-13), ("V", o.v, 1e-12), ("A", o.a, 1e-9), ("J", o.j, 1e-8)):
        assert relvec(g.nb_get_state(f), ref).max() <= tol, f
    Kg, Wg = g.nb_energy(); Ko, Wo = o.energy()
    assert abs((Kg + Wg) - (Ko + Wo)) / abs(Ko + Wo) <= 1e-10
    assert g.guards_intact()
    g.nb_free()


@pytest.mark.parametrize("order", [4, 8])
def test_other_orders_block_steps_and_run_blocks(SIM, oracle, order):
    N, eps, t_end = 300, 1e-3, 2.0 ** -6
    m, x, v = W.plummer(N, 4100 + order, "kroupa")
    g, g2 = SIM(m, x, v, eps, order=order), SIM(m, x, v, eps, order=order)
    o = oracle.OracleSystem(m, x, v, eps, order=order)
    steps = 0
    while True:
        tg, ng, actg = g.nb_next_block()
        to, acto = o.next_block()
        assert tg == to and np.array_equal(actg, acto)
        if to > t_end: break
        g.nb_predict(tg); g.nb_force(actg, outputs=False); g.nb_corrector(actg, 0.0)
        o.predict(to); o.force(acto); o.corrector(acto, 0.0)
        assert np.array_equal(g.nb_get_state("T"), o.t) and np.array_equal(g.nb_get_state("DT"), o.dt)
        steps += 1
    assert steps >= 8
    assert relvec(g.nb_get_state("X"), o.x).max() <= 1e-12 and relvec(g.nb_get_state("V"), o.v).max() <= 1e-11
    s2, t2, _ = g2.nb_run_blocks(t_end)
    assert s2 == steps and t2 == t_end
    for f in ("X", "V", "A", "J", "S", "C", "T", "DT") + (("A4", "A5") if order == 8 else ()):
        assert np.array_equal(g.nb_get_state(f), g2.nb_get_state(f)), f
    assert g.guards_intact() and g2.guards_intact()
    g.nb_free(); g2.nb_free()


# ---------------------------------------------------------------------------------------------------------------
# mixed precision (nb_config.precision = NB_PREC_MIXED) through the host build: the 64-B records the predictor
# writes beside the fp64 ones, li_mixed_body's fp32 sums flushed into fp64 per j-tile, the j-split and the reduction after it.
# CTA-tile evaluations carry the error of an fp32 pair; warp-unit evaluations of the same context stay fp64
# ---------------------------------------------------------------------------------------------------------------
def test_mixed_precision_on_the_host(SIM, oracle):
    from paper_1411_5234_b200 import binding as B
    N, eps = 640, 1e-3
    m, x, v = W.plummer(N, 4242)
    g = SIM(m, x, v, eps, precision=B.NB_PREC_MIXED)
    g.nb_predict(2.0 ** -8)
    assert B.nb_plan_force(N, N).kernel == 0 and B.nb_plan_force(N, 40).kernel == 1
    got, ref = g.nb_force(), oracle_on_records(oracle, g, eps, None)
    errs = [relvec(a, b) for a, b in zip(got[:3], ref[:3])] + [np.abs(got[3] / ref[3] - 1)]
    assert errs[0].max() > 1e-9                               # this really is the fp32 pair arithmetic
    for e, bound in zip(errs, (2e-5, 1e-4, 1e-3, 2e-6)):      # the bounds of the GPU test
        assert e.max() <= bound, (e.max(), bound)
    for arr in got[:3]:                                       # Newton's third law to fp32 round-off of the pair terms
        assert np.abs((m[:, None] * arr).sum(0)).max() <= 1e-5 * (m[:, None] * np.abs(arr)).sum()
    idx = W.active_set(N, 40, 3)
    assert_force_parity(g.nb_force(idx), oracle_on_records(oracle, g, eps, idx))
    steps, _, _ = g.nb_run_blocks(1e30, 3)
    assert steps == 3 and np.isfinite(g.nb_get_state("X")).all()
    assert g.guards_intact()
    g.nb_free()
    with pytest.raises(B.NBError):
        SIM(m, x, v, eps, precision=B.NB_PREC_MIXED, order=8)


# ---------------------------------------------------------------------------------------------------------------
# the boundary through the host build (host-pointer contexts): what include/nb.h promises about call order, argument and index
# errors, state access, the scheduler on crafted times, an eps whose square underflows, bitwise repeatability
# ---------------------------------------------------------------------------------------------------------------
def test_scheduler_on_crafted_times_and_state_io(SIM, oracle):
    N = 1500
    m, x, v = W.plummer(N, 9)
    g = SIM(m, x, v, 1e-3, skip_startup=True)
    assert np.array_equal(g.nb_get_state("M"), m) and np.array_equal(g.nb_get_state("X"), x) and np.array_equal(g.nb_get_state("V"), v)
    rng = np.random.default_rng(3)
    dt = 2.0 ** rng.integers(-12, -3, N)
    t = dt * rng.integers(0, 5, N)
    g.nb_set_state("T", t); g.nb_set_state("DT", dt)
    assert np.array_equal(g.nb_get_state("T"), t) and np.array_equal(g.nb_get_state("DT"), dt)
    tn, n, act = g.nb_next_block()
    act_o, tn_o = np.zeros(N, dtype=np.int32), C.c_double()
    n_o = oracle.lib("ld").oracle_next_block(N, oracle.hermite6._p(t), oracle.hermite6._p(dt), C.byref(tn_o), oracle.hermite6._pi(act_o))
    assert tn == tn_o.value and n == n_o and np.array_equal(act, act_o[:n_o])
    g.nb_set_state("T", np.zeros(N)); g.nb_set_state("DT", np.full(N, 0.125))            # everyone active
    tn, n, act = g.nb_next_block()
    assert tn == 0.125 and n == N and np.array_equal(act, np.arange(N, dtype=np.int32))
    idx = np.array([5, N - 1, 0, 17], dtype=np.int32)                                     # packed fields: neighbours untouched
    for f in ("X", "V", "A", "J", "S", "C"):
        val = rng.normal(size=(4, 3))
        g.nb_set_state(f, val, idx)
        assert np.array_equal(g.nb_get_state(f, idx), val) and np.array_equal(g.nb_get_state(f)[idx], val)
    assert np.array_equal(g.nb_get_state("M"), m) and np.array_equal(g.nb_get_state("T"), np.zeros(N))
    assert g.guards_intact()
    g.nb_free()


def test_call_order_argument_and_index_errors(SIM):
    from paper_1411_5234_b200 import binding as B
    N = 900
    m, x, v = W.plummer(N, 31)
    g = SIM(m, x, v, 1e-3)                                   # host pointers: index lists are verified by default
    with pytest.raises(B.NBError) as e:
        g.nb_force()
    assert e.value.status == B.NB_ESTATE                     # no nb_predict yet
    g.nb_predict(2.0 ** -10)
    with pytest.raises(B.NBError) as e:
        g.nb_corrector(None, 0.1)
    assert e.value.status == B.NB_ESTATE                     # no nb_force yet
    assert g.L.nb_force(g.ctx, None, N + 1, None, None, None, None) == B.NB_EINVAL
    assert g.L.nb_force(g.ctx, None, 5, None, None, None, None) == B.NB_EINVAL            # NULL list needs n_act == N
    assert g.L.nb_force(g.ctx, None, 0, None, None, None, None) == B.NB_OK                # empty active set: no-op
    good = W.active_set(N, 100, 1)
    for bad in (np.array([5, N, 7], dtype=np.int32), np.array([-1], dtype=np.int32), np.array([2 ** 31 - 1, 0], dtype=np.int32)):
        for call in (lambda: g.nb_force(bad), lambda: g.nb_get_state("X", bad), lambda: g.nb_set_state("X", np.zeros((bad.size, 3)), bad)):
            with pytest.raises(B.NBError) as e:
                call()
            assert e.value.status == B.NB_EINVAL
        assert g.nb_check_indices(bad) == B.NB_EINVAL
    dup = np.array([4, 9, 4], dtype=np.int32)
    with pytest.raises(B.NBError) as e:
        g.nb_force(dup)
    assert e.value.status == B.NB_EINVAL
    assert g.nb_check_indices(dup) == B.NB_EINVAL and g.nb_check_indices(dup, unique=False) == B.NB_OK
    assert np.array_equal(g.nb_get_state("X", dup), x[dup])                               # reading a particle twice is fine
    assert g.nb_check_indices(good) == B.NB_OK and g.nb_check_indices(np.arange(N, dtype=np.int32)) == B.NB_OK
    g.nb_force(good, outputs=False)                          # nothing was corrupted: the context still works
    with pytest.raises(B.NBError) as e:
        g.nb_corrector(np.concatenate([good[:-1], good[:1]]), 2.0 ** -10)
    assert e.value.status == B.NB_EINVAL
    g.nb_corrector(good, 2.0 ** -10)
    assert np.isfinite(g.nb_get_state("X")).all() and np.array_equal(g.nb_get_state("M"), m) and g.guards_intact()
    g.nb_free()
    gh = SIM(m, x, v, 1e-3, check_indices=-1, skip_startup=True)                          # checking switched off ...
    assert gh.nb_check_indices(dup) == B.NB_EINVAL                                        # ... the explicit call still checks
    gh.nb_free()
    for kw in (dict(order=5), dict(k_min=-3, k_max=-20), dict(eta=-1.0), dict(precision=7)):
        with pytest.raises(B.NBError) as e:
            SIM(m, x, v, 1e-3, **kw)
        assert e.value.status == B.NB_EINVAL


def test_tiny_softening_and_repeatability(SIM, oracle):
    """0 < eps < 1.5e-154: eps^2 underflows, the launch must take the index-masked (eps = 0) kernels and not produce NaN;
    and the same call twice gives the same bits (fixed-order reduction, work queue left at zero)."""
    N = 500
    m, x, v = W.plummer(N, 33)
    g0, g1 = SIM(m, x, v, 0.0), SIM(m, x, v, 1e-160)
    for f in ("A", "J", "S"):
        a0, a1 = g0.nb_get_state(f), g1.nb_get_state(f)
        assert np.isfinite(a1).all() and np.array_equal(a0, a1), f
    g1.nb_predict(2.0 ** -10)
    for n_act in (3, 50, 300, N):
        idx = None if n_act == N else W.active_set(N, n_act, 2)
        got = g1.nb_force(idx)
        assert_force_parity(got, oracle_on_records(oracle, g1, 0.0, idx))
        again = g1.nb_force(idx)
        assert all(np.array_equal(p, q) for p, q in zip(got, again)), n_act
    g0.nb_free(); g1.nb_free()


# ---------------------------------------------------------------------------------------------------------------
# the order of the CTAs and of the threads: a GPU starts and retires the CTAs of a grid in no defined order, and which thread
# of a CTA runs first between two synchronisation points is not defined either.  The host build runs both 0, 1, 2, ... by
# default; here the same calls run with every grid reversed / shuffled and with the threads of every CTA resumed in reverse /
# in a new random order every round (tests/host/simt/cuda_runtime.h: NB_SIMT_CTA_ORDER, NB_SIMT_THREAD_ORDER).  The work queue
# (first item = CTA number, then the counter), its self-resetting counters, the scheduler's last-block pass and the fixed-order
# reductions must give the same BITS whichever CTA comes first; and a shared-memory or global read that no barrier orders after
# its write would see the old value in one of the thread orders (a poor man's racecheck: compute-sanitizer is closed on the
# pool, profiles/r02_sanitizer.md).  The bulk copies of the j-tiles land "early" (at issue: shows a stage overwritten while it is
# still read) or "late" (NaN bytes at issue, data when the first thread waits on the mbarrier: shows a read that does not wait;
# NB_SIMT_BULK_COPY).  Not covered: memory-model subtleties of real concurrent execution
# ---------------------------------------------------------------------------------------------------------------
ORDERS = [("natural", "natural", "early"), ("reverse", "natural", "early"), ("shuffle", "natural", "early"), ("natural", "reverse", "early"),
          ("natural", "shuffle", "early"), ("shuffle", "shuffle", "early"), ("natural", "natural", "late"), ("shuffle", "shuffle", "late")]


@pytest.mark.parametrize("n_sms,order", [(148, 6), (3, 6), (5, 8), (148, 4)])
def test_results_do_not_depend_on_the_order_of_ctas_and_threads(SIM, n_sms, order):
    N, eps, t_end = 1100, 1e-4, 2.0 ** -7
    m, x, v = W.plummer(N, 606, "kroupa")
    rng = np.random.default_rng(6)
    lists = [None] + [rng.choice(N, n, replace=False).astype(np.int32) for n in (1, 7, 40, 97, 300, 640)]
    results, counters = [], []
    try:
        for cta_order, thread_order, bulk_copy in ORDERS:
            os.environ["NB_SIMT_CTA_ORDER"], os.environ["NB_SIMT_THREAD_ORDER"], os.environ["NB_SIMT_BULK_COPY"] = cta_order, thread_order, bulk_copy
            g = SIM(m, x, v, eps, n_sms=n_sms, order=order)
            out = [g.nb_get_state(f) for f in ("A", "J", "S", "DT")]                     # startup: all-active launches
            g.nb_predict(2.0 ** -10)
            for idx in lists:
                out += list(g.nb_force(idx))
                if order == 8: out.append(g.nb_force_crackle(N if idx is None else idx.size))
            steps, t_last, n_sum = g.nb_run_blocks(t_end)
            assert steps >= 3 and t_last == t_end
            out += [np.array([steps, n_sum])] + [g.nb_get_state(f) for f in ("X", "V", "A", "J", "S", "C", "T", "DT")]
            t, n, act = g.nb_next_block()
            out += [np.array([t, n]), act]
            assert g.guards_intact()
            g.L.nb_simt_permuted_launches.restype = g.L.nb_simt_reordered_ctas.restype = g.L.nb_simt_late_copies.restype = C.c_longlong
            counters.append((g.L.nb_simt_permuted_launches(), g.L.nb_simt_reordered_ctas(), g.L.nb_simt_late_copies()))
            g.nb_free()
            results.append(out)
    finally:
        for name in ("NB_SIMT_CTA_ORDER", "NB_SIMT_THREAD_ORDER", "NB_SIMT_BULK_COPY"): os.environ.pop(name, None)
    # the switches took effect (the counters are cumulative): multi-CTA launches ran permuted, CTAs ran their threads reordered,
    # tiles arrived late
    for k, (cta_order, thread_order, bulk_copy) in enumerate(ORDERS[1:], 1):
        assert (counters[k][0] - counters[k - 1][0] > 30) == (cta_order != "natural"), ORDERS[k]
        assert (counters[k][1] - counters[k - 1][1] > 100) == (thread_order != "natural"), ORDERS[k]
        assert (counters[k][2] - counters[k - 1][2] > 1000) == (bulk_copy == "late"), ORDERS[k]
    for k in range(1, len(ORDERS)):
        assert len(results[k]) == len(results[0])
        for i, (p, q) in enumerate(zip(results[0], results[k])):
            assert np.array_equal(p, q), (ORDERS[k], i)


# ---------------------------------------------------------------------------------------------------------------
# device-pointer contexts (nb_config.ptrs_on_device = 1) and the list nb_next_block leaves inside the context
# (NB_ACTIVE_INTERNAL): same kernels, same plan as a host-pointer context with an explicit list - the same bits
# ---------------------------------------------------------------------------------------------------------------
def test_device_pointer_context_and_internal_active_list(SIM):
    from paper_1411_5234_b200 import binding as B
    N, eps = 900, 1e-3
    m, x, v = W.plummer(N, 5, "kroupa")
    gh, gd = SIM(m, x, v, eps), SIM(m, x, v, eps, device_ptrs=True)
    for _ in range(6):
        th, nh, acth = gh.nb_next_block()
        td, nd, _ = gd.nb_next_block(want_list=False)
        assert th == td and nh == nd
        gh.nb_predict(th); gd.nb_predict(td)
        fh, fd = gh.nb_force(acth), gd.nb_force(B.ACTIVE_INTERNAL, n_act=nd)
        assert all(np.array_equal(a, b) for a, b in zip(fh, fd))
        with pytest.raises(B.NBError) as e:
            gd.nb_force(B.ACTIVE_INTERNAL, n_act=nd + 1)          # not the length of the internal list
        assert e.value.status == B.NB_ESTATE
        gh.nb_corrector(acth, 0.0); gd.nb_corrector(B.ACTIVE_INTERNAL, 0.0, n_act=nd)
    td, nd, actd = gd.nb_next_block()                             # the list written through a "device" pointer
    th, nh, acth = gh.nb_next_block()
    assert td == th and np.array_equal(actd, acth)
    for f in ("X", "V", "A", "J", "S", "C", "T", "DT"):
        assert np.array_equal(gh.nb_get_state(f), gd.nb_get_state(f)), f
    # index lists: the caller's contract by default in this mode, verified when asked for
    gc = SIM(m, x, v, eps, device_ptrs=True, check_indices=1, skip_startup=True)
    gc.nb_predict(0.0)
    with pytest.raises(B.NBError) as e:
        gc.nb_force(np.array([1, N + 5], dtype=np.int32))
    assert e.value.status == B.NB_EINVAL
    assert gc.nb_check_indices(acth) == B.NB_OK
    assert gh.guards_intact() and gd.guards_intact() and gc.guards_intact()
    gh.nb_free(); gd.nb_free(); gc.nb_free()
