"""The arithmetic of the CUDA sources against the oracle, WITHOUT a GPU: the device functions of the hot path are compiled for
the host (tests/host/kernel_source_host.cpp includes nb_predict.h as it is and the text of pair2 / pair2_o4 / pair_o8 /
pair_mixed / corrector_one cut out of the .cu files) and compared with oracle/ on seeded inputs.

What this pins down on a box with no GPU: every formula the kernels are compiled from - the pair evaluation at the three
orders (a, jerk, snap, crackle, pot; the self-pair mask; eps = 0), the predictor's Taylor chains, the Hermite correctors, the
interpolated higher derivatives and the power-of-two time-step criterion (bit-exact levels).  What it does not: the machine
code, the launch plans, the TMA staging, the j-split and its reduction - the `-m gpu` parity tests compare those through the
C ABI on the B200.  The product never runs this code (no CPU fallback: tests/test_abi_cpu.py).
"""
import ctypes as C
import os
import re
import subprocess

import numpy as np
import pytest

from paper_1411_5234_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
CSRC = os.path.join(ROOT, "paper_1411_5234_b200", "csrc")
TOL = 1e-11            # the GPU parity tolerance (north_star)

_d = C.POINTER(C.c_double)
_f = C.POINTER(C.c_float)
_i32 = C.POINTER(C.c_int32)


def _between(text, begin, end, include_end=False):
    assert text.count(begin) == 1, begin
    i = text.index(begin)
    j = text.index(end, i + len(begin))
    return text[i: j + (len(end) if include_end else 0)]


def extract(outdir):
    """cut the device functions out of the .cu files (markers are asserted: a renamed function fails here, loudly)"""
    force = open(os.path.join(CSRC, "nb_force.cu")).read()
    step = open(os.path.join(CSRC, "nb_step.cu")).read()
    parts = {}
    parts["extracted_force_structs.inc"] = "\n".join(
        _between(force, f"struct {name} {{", "};", include_end=True) for name in ("Sums", "IPart", "JRec")) + "\n"
    region = _between(force, "// NB_SCHED_BEGIN", "// NB_SCHED_END")
    assert all(f in region for f in ("void pair2(", "void pair2_o4(", "void pair_o8("))
    parts["extracted_pair_region.inc"] = region + "\n"
    mixed = _between(force, "struct IPartM {", "template <bool EPS0, bool MASK>\n__device__ __forceinline__ void pair_mixed(")
    mixed = "\n".join(l for l in mixed.split("\n") if l.startswith("struct "))          # the three structs; not the float4 loaders
    fn = _between(force, "template <bool EPS0, bool MASK>\n__device__ __forceinline__ void pair_mixed(", "\n}\n", include_end=True)
    parts["extracted_pair_mixed.inc"] = mixed + "\n" + fn
    helpers = _between(step, "__device__ __forceinline__ int clampi(", "// ------------------------------------------------------------------ a0: startup")
    corr = _between(step, "__device__ __forceinline__ void corrector_one(", "\n}\n", include_end=True)
    assert "norm3" in helpers and "ilog2_pos" in helpers and "s.order == 8" in corr and "s.order == 4" in corr
    parts["extracted_corrector.inc"] = helpers + "\n" + corr
    for name, text in parts.items():
        open(os.path.join(outdir, name), "w").write(text)


@pytest.fixture(scope="module")
def H(tmp_path_factory):
    out = str(tmp_path_factory.mktemp("kernel_source_host"))
    extract(out)
    so = os.path.join(out, "libkernel_source_host.so")
    cuda_inc = os.path.join(os.environ.get("CUDA_HOME", "/usr/local/cuda"), "include")
    if not os.path.exists(os.path.join(cuda_inc, "cuda_runtime.h")):
        pytest.skip("no CUDA headers")
    cmd = ["g++", "-O1", "-std=c++17", "-ffp-contract=off", "-w", "-shared", "-fPIC", "-I" + out, "-I" + CSRC,
           "-I" + os.path.join(ROOT, "include"), "-I" + cuda_inc, os.path.join(ROOT, "tests", "host", "kernel_source_host.cpp"), "-o", so]
    r = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    assert r.returncode == 0, r.stdout[-4000:]
    L = C.CDLL(so)
    L.host_force.argtypes = [C.c_int, C.c_int, _d, C.c_int, C.c_int, C.c_double, _i32, C.c_int, _d, _d, _d, _d, _d]
    L.host_force_mixed.argtypes = [C.c_int, C.c_int, _d, _f, _f, _f, C.c_int, C.c_float, _i32, C.c_int, _d, _d, _d, _d]
    L.host_predict.argtypes = [C.c_int, C.c_int] + [_d] * 7 + [C.c_double, C.c_int, _d]
    L.host_correct.argtypes = [C.c_int] + [_d] * 9 + [_i32, C.c_int, C.c_double, C.c_double, _d, _d, _d, _d, C.c_double, C.c_int, C.c_int]
    return L


def p(a): return a.ctypes.data_as(_d)
def pi32(a): return None if a is None else a.ctypes.data_as(_i32)


def relvec(g, o):
    return np.linalg.norm(g - o, axis=-1) / np.linalg.norm(o, axis=-1)


# ---------------------------------------------------------------------------------------------------------------
# marshalling only: the layouts of nb_internal.h (no arithmetic of the method)
# ---------------------------------------------------------------------------------------------------------------
def pack_records(m, xp, vp, ap, jp=None):
    """predicted records (xp, yp) (zp, m) (vxp, vyp) (vzp, axp) (ayp, azp) [(jxp, jyp) (jzp, -)], padded to an even count with
    a massless record far away (as the library pads its arrays)"""
    N = m.shape[0]
    q = 14 if jp is not None else 10
    n_even = N + (N & 1)
    rec = np.zeros((n_even, q))
    rec[:, 0:3] = 3e33
    rec[:N, 0:3], rec[:N, 3], rec[:N, 4:7], rec[:N, 7:10] = xp, m, vp, ap
    if jp is not None: rec[:N, 10:13] = jp
    return np.ascontiguousarray(rec), n_even


def pack_state(o):
    """OracleSystem -> st0 .. st6, dt, tn in the layout of nb_internal.h"""
    N = o.N
    st = [np.zeros((N, 4)) for _ in range(7)]
    st[0][:, :3], st[0][:, 3] = o.x, o.m
    st[1][:, :3], st[1][:, 3] = o.v, o.t
    st[2][:, :3], st[2][:, 3] = o.a, o.j[:, 0]
    st[3][:, 0:2], st[3][:, 2:4] = o.j[:, 1:3], o.s[:, 0:2]
    st[4][:, 0], st[4][:, 1:4] = o.s[:, 2], o.c
    st[5][:, :3], st[5][:, 3] = o.a4, o.a5[:, 0]
    st[6][:, 0:2] = o.a5[:, 1:3]
    return st, o.dt.copy(), (o.t + o.dt).copy()


def unpack_state(st):
    x, m, v, t = st[0][:, :3], st[0][:, 3], st[1][:, :3], st[1][:, 3]
    a = st[2][:, :3]
    j = np.column_stack([st[2][:, 3], st[3][:, 0], st[3][:, 1]])
    s = np.column_stack([st[3][:, 2], st[3][:, 3], st[4][:, 0]])
    c = st[4][:, 1:4]
    a4 = st[5][:, :3]
    a5 = np.column_stack([st[5][:, 3], st[6][:, 0], st[6][:, 1]])
    return dict(x=x, v=v, a=a, j=j, s=s, c=c, a4=a4, a5=a5, t=t, m=m)


def host_force(H, order, m, xp, vp, ap, jp, eps, idx, tile=16):
    rec, n_even = pack_records(m, xp, vp, ap, jp if order == 8 else None)
    n = m.shape[0] if idx is None else idx.shape[0]
    oa, oj, os_, oc, op = np.zeros((n, 3)), np.zeros((n, 3)), np.zeros((n, 3)), np.zeros((n, 3)), np.zeros(n)
    eps2 = eps * eps
    rc = H.host_force(order, int(not (eps2 >= np.finfo(np.float64).tiny)), p(rec), n_even, tile, eps2, pi32(idx), n,
                      p(oa), p(oj), p(os_), p(oc), p(op))
    assert rc == 0
    return oa, oj, os_, oc, op


def seeded_system(N, seed=7, masses="equal"):
    m, x, v = W.plummer(N, W.BASE_SEED + seed, masses)
    rng = np.random.default_rng(seed)
    a = rng.normal(size=(N, 3))          # any "predicted acceleration" and jerk: the evaluation is a pure function of the records
    j = rng.normal(size=(N, 3)) * 3.0
    return m, x, v, a, j


# ---------------------------------------------------------------------------------------------------------------
# a2: the pair evaluation
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("eps", [1e-4, 0.0])
@pytest.mark.parametrize("N,masses", [(150, "equal"), (97, "kroupa")])
def test_pair2_source_against_oracle(H, oracle, N, masses, eps):
    m, x, v, a, _ = seeded_system(N, masses=masses)
    idx = np.ascontiguousarray(W.active_set(N, 41, 3), dtype=np.int32)
    for sel in (None, idx):
        ga, gj, gs, _, gp = host_force(H, 6, m, x, v, a, None, eps, sel)
        oa, oj, os_, op = oracle.hermite6.force(m, x, v, a, eps, sel)
        assert relvec(ga, oa).max() <= TOL and relvec(gj, oj).max() <= TOL and relvec(gs, os_).max() <= TOL
        assert np.abs(gp / op - 1).max() <= TOL


@pytest.mark.parametrize("eps", [1e-4, 0.0])
def test_pair2_o4_source_against_oracle(H, oracle, eps):
    m, x, v, a, _ = seeded_system(131)
    ga, gj, gs, _, gp = host_force(H, 4, m, x, v, a, None, eps, None)
    oa, oj, _, op = oracle.hermite6.force(m, x, v, a, eps, None, want=("a", "j", "p"))
    assert relvec(ga, oa).max() <= TOL and relvec(gj, oj).max() <= TOL and np.abs(gp / op - 1).max() <= TOL
    assert not gs.any()                                    # the 4th-order variant leaves the snap sums at 0


@pytest.mark.parametrize("eps", [1e-4, 0.0])
def test_pair_o8_source_against_oracle(H, oracle, eps):
    m, x, v, a, j = seeded_system(120, masses="kroupa")
    idx = np.ascontiguousarray(W.active_set(120, 33, 5), dtype=np.int32)
    for sel in (None, idx):
        ga, gj, gs, gc, gp = host_force(H, 8, m, x, v, a, j, eps, sel)
        oa, oj, os_, oc, op = oracle.hermite6.force8(m, x, v, a, j, eps, sel)
        for g, o in ((ga, oa), (gj, oj), (gs, os_), (gc, oc)):
            assert relvec(g, o).max() <= TOL
        assert np.abs(gp / op - 1).max() <= TOL


def test_tile_size_and_self_mask_do_not_change_the_sums(H):
    """the masked copy of the loop is taken only in the tile that holds the particle: whatever the tile size, the sums of
    a, jerk, snap are bit-identical (the self pair adds exact zeros), pot too"""
    m, x, v, a, _ = seeded_system(64)
    r16 = host_force(H, 6, m, x, v, a, None, 1e-4, None, tile=16)
    r64 = host_force(H, 6, m, x, v, a, None, 1e-4, None, tile=64)
    r2 = host_force(H, 6, m, x, v, a, None, 1e-4, None, tile=2)
    for q16, q64, q2 in zip(r16, r64, r2):
        assert np.array_equal(q16, q64) and np.array_equal(q16, q2)


def test_pair_mixed_source_error_against_oracle(H, oracle):
    """nb_config.precision = NB_PREC_MIXED: fp64 differences + accumulation, fp32 pair arithmetic.  The bounds are
    those of the GPU test; here the MUFU.RSQ seed is the correctly rounded fp32 value"""
    N, eps = 2000, 1e-4
    m, x, v, a, _ = seeded_system(N)
    _, _, _, a0, _ = (None, None, None, *oracle.hermite6.force(m, x, v, np.zeros((N, 3)), eps, None)[:1], None)
    a = a0                                                  # a physical acceleration field (the startup's first pass)
    oa, oj, os_, op = oracle.hermite6.force(m, x, v, a, eps, None)
    ga, gj, gs, gp = np.zeros((N, 3)), np.zeros((N, 3)), np.zeros((N, 3)), np.zeros(N)
    mf, vf, af = m.astype(np.float32), np.ascontiguousarray(v, dtype=np.float32), np.ascontiguousarray(a, dtype=np.float32)
    fp = lambda q: q.ctypes.data_as(_f)
    assert H.host_force_mixed(0, N, p(np.ascontiguousarray(x)), fp(mf), fp(vf), fp(af), 128, np.float32(eps * eps), None, N,
                              p(ga), p(gj), p(gs), p(gp)) == 0
    ea, ej, es, ep = relvec(ga, oa), relvec(gj, oj), relvec(gs, os_), np.abs(gp / op - 1)
    assert ea.max() <= 2e-5 and ej.max() <= 1e-4 and es.max() <= 1e-3 and ep.max() <= 2e-6
    assert np.median(ea) <= 2e-6 and np.median(ej) <= 5e-6 and np.median(es) <= 2e-5


# ---------------------------------------------------------------------------------------------------------------
# a1: the predictor
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("order", [4, 6, 8])
def test_predictor_source_against_oracle(H, oracle, order):
    N = 200
    m, x, v = W.plummer(N, W.BASE_SEED + 9, "equal")
    o = oracle.OracleSystem(m, x, v, 1e-3, order=order)
    rng = np.random.default_rng(order)
    o.c[:] = rng.normal(size=(N, 3)) * 5.0                   # fill the higher derivatives the startup leaves at 0
    o.a4[:], o.a5[:] = rng.normal(size=(N, 3)) * 20.0, rng.normal(size=(N, 3)) * 100.0
    o.t[:] = rng.integers(0, 8, size=N) * 2.0 ** -7
    t = 2.0 ** -4 + 2.0 ** -9
    o.predict(t)
    st, _, _ = pack_state(o)
    q = 14 if order == 8 else 10
    rec = np.zeros((N, q))
    assert H.host_predict(order, N, *[p(s) for s in st], t, 0, p(rec)) == 0
    assert np.abs(rec[:, 0:3] / o.xp - 1).max() <= 1e-14 and np.abs(rec[:, 4:7] / o.vp - 1).max() <= 1e-13
    assert np.array_equal(rec[:, 3], m)
    if order != 4: assert np.abs(rec[:, 7:10] - o.ap).max() <= 1e-13 * np.abs(o.ap).max()
    if order == 8: assert np.abs(rec[:, 10:13] - o.jp).max() <= 1e-13 * np.abs(o.jp).max()
    # own_time: the record is the stored state (the startup evaluations use it)
    rec0 = np.zeros((N, q))
    assert H.host_predict(order, N, *[p(s) for s in st], t, 1, p(rec0)) == 0
    assert np.array_equal(rec0[:, 0:3], o.x) and np.array_equal(rec0[:, 4:7], o.v)


# ---------------------------------------------------------------------------------------------------------------
# a4 + a5: corrector, interpolated derivatives, time-step criterion and quantisation
# ---------------------------------------------------------------------------------------------------------------
def eta_p(o):
    return {4: o.eta, 6: o.eta ** 3, 8: o.eta ** 5}[o.order]


@pytest.mark.parametrize("order", [4, 6, 8])
def test_corrector_source_block_steps_against_oracle(H, oracle, order):
    """block steps: the oracle advances; before every corrector its state, forces and active list go through the host build
    of corrector_one and the results are compared: x, v and the derivatives to rounding, the new time-step LEVELS bit for bit"""
    N = 96
    m, x, v = W.plummer(N, W.BASE_SEED + 11, "kroupa")
    o = oracle.OracleSystem(m, x, v, 1e-2, order=order)
    seen = 0
    for step in range(40):
        tn, act = o.next_block()
        o.predict(tn)
        f = o.force(act)
        st, dt, tnext = pack_state(o)
        fa, fj, fs = (np.ascontiguousarray(q) for q in f[:3])
        fc = np.ascontiguousarray(f[4]) if order == 8 else np.zeros((act.shape[0], 3))
        assert H.host_correct(order, *[p(s) for s in st], p(dt), p(tnext), pi32(act), act.shape[0], 0.0, tn, p(fa), p(fj), p(fs), p(fc),
                              eta_p(o), o.k_min, o.k_max) == 0
        nrm = lambda q: np.linalg.norm(q, axis=-1)
        hh = 0.5 * (tn - o.t[act])
        scale = nrm(o.a[act]) + nrm(f[0]) + hh * (nrm(o.j[act]) + nrm(f[1]))
        if order != 4: scale = scale + hh ** 2 * (nrm(o.s[act]) + nrm(f[2]))
        if order == 8: scale = scale + hh ** 3 * (nrm(o.c[act]) + nrm(f[4]))
        o.corrector(act, 0.0)
        g = unpack_state(st)
        assert np.array_equal(dt, o.dt), (step, np.flatnonzero(dt != o.dt))                  # levels: bit-exact
        assert np.array_equal(g["t"], o.t) and np.array_equal(tnext, o.t + o.dt)
        assert np.abs(g["x"] - o.x).max() <= 1e-14 and np.abs(g["v"] - o.v).max() <= 1e-13
        for name in ("a", "j") + (("s",) if order != 4 else ()):
            assert np.array_equal(g[name][act], getattr(o, name)[act]), name              # copied from the evaluation
        # the interpolated higher derivatives are p-th differences of the end-point values divided by (h/2)^p: with identical
        # inputs on both sides the rounding of the combination (coefficients up to 1575) is what differs
        hi = {4: (("s", 2), ("c", 3)), 6: (("c", 3),), 8: (("a4", 4), ("a5", 5))}[order]
        for name, pw in hi:
            err = nrm(g[name][act] - getattr(o, name)[act])
            assert np.all(err <= 1e-12 * scale / hh ** pw), (name, (err * hh ** pw / scale).max())
        seen += act.shape[0]
    assert seen > 40


@pytest.mark.parametrize("order", [4, 6, 8])
def test_corrector_source_shared_step_against_oracle(H, oracle, order):
    N = 64
    m, x, v = W.plummer(N, W.BASE_SEED + 12, "equal")
    o = oracle.OracleSystem(m, x, v, 1e-2, order=order)
    h = 2.0 ** -8
    for step in range(3):
        t = o.t[0] + h
        o.predict(t)
        f = o.force(None)
        st, dt, tnext = pack_state(o)
        fa, fj, fs = (np.ascontiguousarray(q) for q in f[:3])
        fc = np.ascontiguousarray(f[4]) if order == 8 else np.zeros((N, 3))
        assert H.host_correct(order, *[p(s) for s in st], p(dt), p(tnext), None, N, h, t, p(fa), p(fj), p(fs), p(fc),
                              eta_p(o), o.k_min, o.k_max) == 0
        o.corrector(None, h)
        g = unpack_state(st)
        assert np.array_equal(dt, o.dt) and np.all(dt == h) and np.array_equal(g["t"], o.t)
        assert np.abs(g["x"] - o.x).max() <= 1e-14 and np.abs(g["v"] - o.v).max() <= 1e-13
