"""GPU parity tests: the CUDA path (through the C ABI, via the ctypes binding) against the CPU oracle,
element by element on the same seeded inputs.  Tolerances (BASELINE.json north_star):
  a, jerk, snap per particle: || gpu - oracle ||_2 / || oracle ||_2 <= 1e-11;  pot: relative 1e-11
  total energy after 8 steps: relative 1e-10
  indices, times, step levels: bit-exact.
"""
import ctypes as C

import numpy as np
import pytest

from paper_1411_5234_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL = 1e-11


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1411_5234_b200 import binding
    binding.lib()
    return binding


def relvec(g, o):
    return np.linalg.norm(g - o, axis=-1) / np.linalg.norm(o, axis=-1)


def assert_force_parity(g, o, tol=TOL):
    ga, gj, gs, gp = g
    oa, oj, os_, op = o
    assert relvec(ga, oa).max() <= tol, ("acc", relvec(ga, oa).max())
    assert relvec(gj, oj).max() <= tol, ("jerk", relvec(gj, oj).max())
    assert relvec(gs, os_).max() <= tol, ("snap", relvec(gs, os_).max())
    assert np.abs(gp / op - 1).max() <= tol, ("pot", np.abs(gp / op - 1).max())


def oracle_on_gpu_records(oracle, sysg, eps, idx):
    """O1 on the predicted records the GPU kernel read (nb_force is a pure function of them)."""
    m = sysg.nb_get_state("M")
    xp, vp, ap = sysg.nb_get_state("XP"), sysg.nb_get_state("VP"), sysg.nb_get_state("AP")
    return oracle.hermite6.force(m, xp, vp, ap, eps, idx)


# ------------------------------------------------------------------ config 1, end to end
def test_config1_force_and_8_steps(B, oracle):
    c, m, x, v = W.config_inputs(1)
    g = B.System(m, x, v, c.eps)
    o = oracle.OracleSystem(m, x, v, c.eps)
    # startup (two-pass) state
    for f, ref in (("A", o.a), ("J", o.j), ("S", o.s)):
        assert relvec(g.nb_get_state(f), ref).max() <= TOL
    assert np.array_equal(g.nb_get_state("DT"), o.dt)
    # one predict + force
    g.nb_predict(0.0); o.predict(0.0)
    assert_force_parity(g.nb_force(), o.force())
    Kg0, Wg0 = g.nb_energy()
    Ko0, Wo0 = o.energy()
    assert abs((Kg0 + Wg0) / (Ko0 + Wo0) - 1) <= 1e-12
    # 8 shared steps
    t = 0.0
    for _ in range(c.n_steps):
        t += c.dt
        g.nb_predict(t); g.nb_force(outputs=False); g.nb_corrector(None, c.dt)
        o.shared_step(c.dt)
    assert np.all(g.nb_get_state("T") == t)
    for f, ref, tol in (("X", o.x, 1e-13), ("V", o.v, 1e-12), ("A", o.a, TOL), ("J", o.j, TOL), ("S", o.s, TOL)):
        assert relvec(g.nb_get_state(f), ref).max() <= tol, f
    # crackle is a third difference of (a, h/2 jerk, (h/2)^2 snap) over the step, divided by (h/2)^3: a relative
    # difference d in the force results (allowed: 1e-11; typical: 1e-14) becomes d (|a| + hh |jerk| + hh^2 |snap|) / hh^3
    # in crackle, whatever the implementation.  Bound at a tenth of the force tolerance.
    hh = c.dt / 2
    nrm = lambda a: np.linalg.norm(a, axis=1)
    bound = 1e-12 * (nrm(o.a) + hh * nrm(o.j) + hh * hh * nrm(o.s)) / hh ** 3
    assert np.all(nrm(g.nb_get_state("C") - o.c) <= bound)
    Kg, Wg = g.nb_energy()
    Ko, Wo = o.energy()
    assert abs((Kg + Wg) - (Ko + Wo)) / abs(Ko + Wo) <= 1e-10
    g.nb_free()


# ------------------------------------------------------------------ force kernel shapes, ragged sizes, edge cases
@pytest.mark.parametrize("N,eps,masses", [(1000, 1e-3, "equal"), (4099, 1e-4, "kroupa"), (2, 0.0, "equal"), (257, 0.0, "kroupa"),
                                          (16500, 0.0, "kroupa")])
def test_force_parity_active_sets(B, oracle, N, eps, masses):
    m, x, v = W.plummer(N, 1000 + N, masses)
    g = B.System(m, x, v, eps)
    # advance once so that a, jerk, snap, crackle are all non-zero and D != 0 in the predictor
    g.nb_predict(2.0 ** -9); g.nb_force(outputs=False); g.nb_corrector(None, 2.0 ** -9)
    g.nb_predict(2.0 ** -9 + 2.0 ** -11)
    rng = np.random.default_rng(N)
    sizes = sorted({1, 2, 3, 5, 6, 7, 11, 13, 16, 17, 21, 24, 31, 33, 64, 96, 97, 129, 255, 256, 300, 1023, 1024, 1025, 2049, N} & set(range(1, N + 1)) | {N})
    if N > 10000:
        sizes = [1, 19, 5000, 16383, N]                  # warp units (5000: 39 full tiles + 8) and ragged CTA tiles (N = 128 * 128 + 116)
    for n_act in sizes:
        idx = None if n_act == N else rng.choice(N, n_act, replace=False).astype(np.int32)
        got = g.nb_force(idx)
        ref = oracle_on_gpu_records(oracle, g, eps, idx)
        assert_force_parity(got, ref)
        plan = B.nb_plan_force(N, n_act, 148)
        assert plan.kernel == (0 if n_act >= 256 and n_act * 100 >= 93 * 128 * ((n_act + 127) // 128) else 1)   # CTA tiles / warp units
    # permuted full list: row k <-> idx[k]
    perm = rng.permutation(N).astype(np.int32)
    got = g.nb_force(perm)
    ref = oracle_on_gpu_records(oracle, g, eps, perm)
    assert_force_parity(got, ref)
    g.nb_free()


def test_predictor_and_corrector_parity_block_steps(B, oracle):
    """Same block-step sequence on both sides, N = 384 Kroupa masses: scheduler output bit-exact,
    predictor/corrector/time-step levels compared after every block step."""
    N, eps = 384, 1e-3
    m, x, v = W.plummer(N, 77, "kroupa")
    g = B.System(m, x, v, eps)
    o = oracle.OracleSystem(m, x, v, eps)
    assert np.array_equal(g.nb_get_state("DT"), o.dt)
    n_steps = 0
    while True:
        tg, ng, actg = g.nb_next_block()
        to, acto = o.next_block()
        assert tg == to and ng == acto.size and np.array_equal(actg, acto)      # bit-exact
        if to > 2.0 ** -5:
            break
        g.nb_predict(tg); o.predict(to)
        for f, ref in (("XP", o.xp), ("VP", o.vp), ("AP", o.ap)):
            assert relvec(g.nb_get_state(f), ref).max() <= 1e-12, f
        assert_force_parity(g.nb_force(actg), o.force(acto), 1e-10)     # states differ at round-off by now
        g.nb_corrector(actg, 0.0); o.corrector(acto, 0.0)
        assert np.array_equal(g.nb_get_state("T"), o.t)
        assert np.array_equal(g.nb_get_state("DT"), o.dt)               # same level decisions
        n_steps += 1
    assert n_steps > 20
    for f, ref, tol in (("X", o.x, 1e-12), ("V", o.v, 1e-11)):
        assert relvec(g.nb_get_state(f), ref).max() <= tol
    g.nb_free()


def test_internal_active_list_and_device_pointers(B, oracle):
    import torch
    N, eps = 3000, 1e-3
    m, x, v = W.plummer(N, 5, "kroupa")
    gh = B.System(m, x, v, eps, host=True)
    dev = "cuda:0"
    gd = B.System(torch.tensor(m, device=dev), torch.tensor(x, device=dev), torch.tensor(v, device=dev), eps, host=False)
    for _ in range(5):
        th, nh, acth = gh.nb_next_block()
        td, nd, _ = gd.nb_next_block(want_list=False)
        assert th == td and nh == nd
        gh.nb_predict(th); gd.nb_predict(td)
        fh = gh.nb_force(acth)
        fd = gd.nb_force(B.ACTIVE_INTERNAL, n_act=nd)
        torch.cuda.synchronize()
        for a, b in zip(fh, fd):
            assert np.array_equal(a, b.cpu().numpy())                   # same kernels, same plan: bitwise equal
        gh.nb_corrector(acth, 0.0); gd.nb_corrector(B.ACTIVE_INTERNAL, 0.0, n_act=nd)
    torch.cuda.synchronize()
    assert np.array_equal(gh.nb_get_state("X"), gd.nb_get_state("X").cpu().numpy())
    gh.nb_free(); gd.nb_free()


def test_run_to_run_determinism(B):
    N = 20000
    m, x, v = W.plummer(N, 8)
    res = []
    for _ in range(2):
        g = B.System(m, x, v, 1e-4)
        g.nb_predict(2.0 ** -10)
        idx = W.active_set(N, 3000, 4)
        res.append((g.nb_force(idx), g.nb_force(None), g.nb_force(idx[:50].copy())))
        g.nb_free()
    for r0, r1 in zip(*res):
        for a, b in zip(r0, r1):
            assert np.array_equal(a, b)


def test_scheduler_bit_exact_on_crafted_times(B, oracle):
    N = 5000
    m, x, v = W.plummer(N, 9)
    g = B.System(m, x, v, 1e-3)
    rng = np.random.default_rng(3)
    lev = rng.integers(-12, -3, N)
    dt = 2.0 ** lev
    t = dt * rng.integers(0, 5, N)
    g.nb_set_state("T", t); g.nb_set_state("DT", dt)
    assert np.array_equal(g.nb_get_state("T"), t) and np.array_equal(g.nb_get_state("DT"), dt)
    tn, n, act = g.nb_next_block()
    act_o = np.zeros(N, dtype=np.int32)
    tn_o = C.c_double()
    n_o = oracle.lib("ld").oracle_next_block(N, oracle.hermite6._p(t), oracle.hermite6._p(dt), C.byref(tn_o),
                                             oracle.hermite6._pi(act_o))
    assert tn == tn_o.value and n == n_o and np.array_equal(act, act_o[:n_o])
    # everyone active
    g.nb_set_state("T", np.zeros(N)); g.nb_set_state("DT", np.full(N, 0.125))
    tn, n, act = g.nb_next_block()
    assert tn == 0.125 and n == N and np.array_equal(act, np.arange(N, dtype=np.int32))
    g.nb_free()


def test_state_io_and_errors(B):
    N = 700
    m, x, v = W.plummer(N, 10)
    g = B.System(m, x, v, 1e-3)
    assert np.array_equal(g.nb_get_state("M"), m) and np.array_equal(g.nb_get_state("X"), x)
    assert np.array_equal(g.nb_get_state("V"), v)
    idx = np.array([5, 699, 0, 17], dtype=np.int32)
    assert np.array_equal(g.nb_get_state("X", idx), x[idx])
    rng = np.random.default_rng(0)
    for f in ("X", "V", "A", "J", "S", "C"):
        val = rng.normal(size=(4, 3))
        g.nb_set_state(f, val, idx)
        assert np.array_equal(g.nb_get_state(f, idx), val)
        full = g.nb_get_state(f)
        assert np.array_equal(full[idx], val)
    # neighbours untouched by the packed-field writes
    assert np.array_equal(g.nb_get_state("M"), m)
    # call-order and argument errors
    with pytest.raises(B.NBError) as e:
        g.nb_force()
    assert e.value.status == B.NB_ESTATE
    g.nb_predict(0.0)
    with pytest.raises(B.NBError) as e:
        g.nb_corrector(None, 0.1)
    assert e.value.status == B.NB_ESTATE
    assert g.L.nb_force(g.ctx, None, N + 1, None, None, None, None) == B.NB_EINVAL
    assert g.L.nb_force(g.ctx, None, 5, None, None, None, None) == B.NB_EINVAL       # NULL list needs n_act == N
    assert g.L.nb_force(g.ctx, None, 0, None, None, None, None) == B.NB_OK           # empty active set: no-op
    g.nb_free()
    # workspace too small / bad arguments
    import torch
    ws = torch.empty(4096, dtype=torch.uint8, device="cuda:0")
    cfg = B.nb_config(0, None, C.c_void_p(ws.data_ptr()), 4096, 0, 0, 0, 0, 0, 0, 0, 0)
    ctx = C.c_void_p()
    mm = np.ascontiguousarray(m)
    args = (B._ptr(mm), B._ptr(np.ascontiguousarray(x)), B._ptr(np.ascontiguousarray(v)))
    assert B.lib().nb_init(C.byref(ctx), N, *args, 1e-3, C.byref(cfg)) == B.NB_ENOMEM
    assert B.lib().nb_init(C.byref(ctx), 0, *args, 1e-3, C.byref(cfg)) == B.NB_EINVAL
    assert B.lib().nb_init(C.byref(ctx), N, *args, -1.0, C.byref(cfg)) == B.NB_EINVAL


def test_newton_third_law_and_energy_on_gpu(B):
    """Properties that hold at any size: sum m a = sum m jerk = sum m snap = 0; 6th-order energy behaviour."""
    N = 30000
    m, x, v = W.plummer(N, 12, "kroupa")
    g = B.System(m, x, v, 1e-3)
    for f in ("A", "J", "S"):
        arr = g.nb_get_state(f)
        assert np.abs((m[:, None] * arr).sum(0)).max() <= 1e-13 * (m[:, None] * np.abs(arr)).sum()
    g.nb_free()


# ------------------------------------------------------------------ full sizes, sampled (configs 2, 4, 5)
@pytest.fixture(scope="module")
def big(B):
    c, m, x, v = W.config_inputs(4)
    g = B.System(m, x, v, c.eps)
    yield c, m, x, v, g
    g.nb_free()


def test_config4_full_size_sampled(big, B, oracle):
    c, m, x, v, g = big
    N = c.N
    g.nb_predict(0.0)
    ga, gj, gs, gp = g.nb_force()                    # the bench configuration: all N active
    ms = g.nb_last_force_ms()
    assert ms > 0
    # 4096 seeded particles plus the whole first and last i-tile of the launch (128 particles each)
    sample = np.unique(np.concatenate([W.active_set(N, 4096, 999), np.arange(128), np.arange(N - 128, N)])).astype(np.int32)
    a_state = g.nb_get_state("A")
    ref = oracle.hermite6.force(m, x, v, a_state, c.eps, sample)
    assert_force_parity((ga[sample], gj[sample], gs[sample], gp[sample]), ref)
    # properties over all N: Newton's third law, potential energy consistent with Henon units
    for arr in (ga, gj, gs):
        assert np.abs((m[:, None] * arr).sum(0)).max() <= 1e-12 * (m[:, None] * np.abs(arr)).sum()
    Wpot = 0.5 * (m * gp).sum()
    assert abs(Wpot + 0.5) < 0.01


@pytest.mark.parametrize("n_act", [1, 8, 64, 512, 4096, 32768])
def test_config5_small_active_sets_full_size(big, B, oracle, n_act):
    c, m, x, v, g = big
    idx = W.config5_active(n_act)
    g.nb_predict(0.0)
    got = g.nb_force(idx)
    # every row up to n_act = 4096; above, 4096 seeded rows plus the first and last 128 (first / last i-tile)
    rows = np.arange(n_act) if n_act <= 4096 else np.unique(np.concatenate(
        [np.random.default_rng(n_act).choice(n_act, 4096, replace=False), np.arange(128), np.arange(n_act - 128, n_act)]))
    a_state = g.nb_get_state("A")
    ref = oracle.hermite6.force(m, x, v, a_state, c.eps, idx[rows])
    assert_force_parity(tuple(a[rows] for a in got), ref)


@pytest.mark.slow
def test_config2_sampled_and_steps(B, oracle, capsys):
    """BASELINE.json configs[1]: N = 65536, full evaluation + 16 shared steps, "energy drift vs oracle".  The ORACLE runs the
    same 16 steps (startup + 16 evaluations + 2 for the energies, a few minutes of host time): final x, v, a, jerk, snap and
    the total energy are compared side by side, and both drifts are printed."""
    import time
    c, m, x, v = W.config_inputs(2)
    g = B.System(m, x, v, c.eps)
    K0, W0 = g.nb_energy()
    t = 0.0
    for _ in range(c.n_steps):
        t += c.dt
        g.nb_predict(t); g.nb_force(outputs=False); g.nb_corrector(None, c.dt)
    g.nb_predict(t)
    got = g.nb_force()
    sample = W.active_set(c.N, 128, 123)
    ref = oracle_on_gpu_records(oracle, g, c.eps, sample)
    assert_force_parity(tuple(a[sample] for a in got), ref)
    K1, W1 = g.nb_energy()
    drift_gpu = (K1 + W1) / (K0 + W0) - 1

    # the oracle through the same steps: x87 long double if the host finishes it in ~10 min, else its fp64 build
    probe = W.active_set(c.N, 256, 5)
    t0 = time.perf_counter()
    oracle.hermite6.force(m, x, v, np.zeros_like(x), c.eps, probe, kind="ld")
    rate = probe.size * (c.N - 1) / (time.perf_counter() - t0)
    kind = "ld" if (c.n_steps + 4) * c.N * (c.N - 1) / rate < 600 else "f64"
    t0 = time.perf_counter()
    o = oracle.OracleSystem(m, x, v, c.eps, kind=kind)
    Ko0, Wo0 = o.energy()
    for _ in range(c.n_steps):
        o.shared_step(c.dt)
    Ko1, Wo1 = o.energy()
    drift_or = (Ko1 + Wo1) / (Ko0 + Wo0) - 1
    with capsys.disabled():
        print(f"\n[config 2] 16 shared steps dt = 2^-12: dE/E GPU {drift_gpu:.6e}, oracle({kind}) {drift_or:.6e}; "
              f"|E_gpu - E_or|/|E_or| = {abs((K1 + W1) - (Ko1 + Wo1)) / abs(Ko1 + Wo1):.2e}; oracle took {time.perf_counter() - t0:.0f} s")
    assert abs((K0 + W0) - (Ko0 + Wo0)) / abs(Ko0 + Wo0) <= 1e-12
    assert abs((K1 + W1) - (Ko1 + Wo1)) / abs(Ko1 + Wo1) <= 1e-10                # north_star: energy vs oracle
    assert np.all(g.nb_get_state("T") == t) and np.all(o.t == t)
    for f, ref_, tol in (("X", o.x, 1e-12), ("V", o.v, 1e-11), ("A", o.a, TOL), ("J", o.j, TOL), ("S", o.s, TOL)):
        assert relvec(g.nb_get_state(f), ref_).max() <= tol, f
    # the drift itself is a property of the method at this shared step (reported above from both sides), bounded loosely
    assert abs(drift_gpu) < 1e-5 and abs(drift_or) < 1e-5 and abs(drift_gpu - drift_or) <= 1e-10
    g.nb_free()


def test_config3_full_size_sampled_block_steps(B, oracle):
    """Config 3 at its full size (N = 262144, Kroupa masses, block steps): advance on the GPU, then check sampled
    block steps piece by piece against the oracle started from the GPU's state - scheduler bit-exact, predictor on all
    N, the pairwise evaluation on up to 48 of the active particles (all N j-particles), corrector + time-step levels on
    all active particles from identical inputs."""
    import torch
    c, m, x, v = W.config_inputs(3)
    N = m.shape[0]
    dev = "cuda:0"
    g = B.System(torch.tensor(m, device=dev), torch.tensor(x, device=dev), torch.tensor(v, device=dev), c.eps, host=False)
    K0, W0 = g.nb_energy()
    steps, t_last, _ = g.nb_run_blocks(2.0 ** -8)
    assert steps > 50 and t_last == 2.0 ** -8
    get = lambda f: g.nb_get_state(f).cpu().numpy()
    o = oracle.OracleSystem.from_state(m, *(get(f) for f in ("X", "V", "A", "J", "S", "C", "T", "DT")), c.eps)
    rng = np.random.default_rng(3)
    kernels = set()
    for step in range(40):
        tg, ng, actg = g.nb_next_block()
        to, acto = o.next_block()
        actg = actg.cpu().numpy()
        assert tg == to and np.array_equal(actg, acto)                           # bit-exact schedule
        kernels.add(B.nb_plan_force(N, ng, 148).kernel)
        g.nb_predict(tg); o.predict(to)
        for f, ref in (("XP", o.xp), ("VP", o.vp), ("AP", o.ap)):
            assert relvec(get(f), ref).max() <= 1e-12, f
        got = tuple(q.cpu().numpy() for q in g.nb_force(torch.tensor(actg, device=dev)))
        rows = np.arange(ng) if ng <= 48 else np.sort(rng.choice(ng, 48, replace=False))
        ref = oracle.hermite6.force(m, o.xp, o.vp, o.ap, c.eps, acto[rows])
        assert_force_parity(tuple(q[rows] for q in got), ref)
        # corrector and time-step criterion on identical inputs: the oracle takes the GPU's a, jerk, snap
        o.f = got
        g.nb_corrector(torch.tensor(actg, device=dev), 0.0); o.corrector(acto, 0.0)
        for f, ref, tol in (("X", o.x, 1e-14), ("V", o.v, 1e-13), ("A", o.a, 0), ("J", o.j, 0), ("S", o.s, 0)):
            assert relvec(get(f)[acto], ref[acto]).max() <= tol, f
        assert np.array_equal(get("T"), o.t)
        assert np.array_equal(get("DT"), o.dt), "time-step levels"
        # resynchronise the oracle's x, v, crackle with the GPU's (round-off level) so that the next schedule stays comparable
        o.x[acto], o.v[acto], o.c[acto] = get("X")[acto], get("V")[acto], get("C")[acto]
    assert 1 in kernels                                                          # the warp-unit shape was exercised
    g.nb_free()


def test_run_blocks_is_bitwise_the_separate_calls(B):
    """nb_run_blocks (scheduler, plan and step on the device, CUDA graph) against the same steps driven call by call:
    identical schedules, bit-identical states; step budget and t_end respected; eps = 0 variant."""
    for N, eps, masses in ((3000, 1e-4, "kroupa"), (300, 0.0, "equal")):
        m, x, v = W.plummer(N, 77 + N, masses)
        g1 = B.System(m, x, v, eps)
        g2 = B.System(m, x, v, eps)
        t_end = 2.0 ** -5
        steps, acts = 0, 0
        while True:
            t, n, act = g1.nb_next_block()
            if t > t_end:
                break
            g1.nb_predict(t); g1.nb_force(act, outputs=False); g1.nb_corrector(act, 0.0)
            steps += 1; acts += n
        # in three instalments: a step budget, then a time limit, then the rest
        s_a, t_a, n_a = g2.nb_run_blocks(t_end, max_steps=5)
        assert s_a == 5 and t_a > 0
        s_b, t_b, n_b = g2.nb_run_blocks(t_end / 2)
        assert t_b <= t_end / 2
        s_c, t_c, n_c = g2.nb_run_blocks(t_end)
        assert s_a + s_b + s_c == steps and n_a + n_b + n_c == acts and t_c == t_end
        assert g2.nb_run_blocks(t_end) == (0, -1.0, 0)                    # nothing left below t_end
        for f in ("X", "V", "A", "J", "S", "C", "T", "DT"):
            assert np.array_equal(g1.nb_get_state(f), g2.nb_get_state(f)), f
        # the separate calls still work on a context that has run the graph
        t1, n1, a1 = g1.nb_next_block(); t2, n2, a2 = g2.nb_next_block()
        assert t1 == t2 and np.array_equal(a1, a2)
        g1.nb_free(); g2.nb_free()


def test_config3_reduced_twin_block_steps(B, oracle):
    """Config 3's recipe at N = 2048 run end to end to t = 1/8 on both sides."""
    _, m, x, v = W.config_inputs(3, N=2048)
    eps = W.CONFIGS[3].eps
    g = B.System(m, x, v, eps)
    o = oracle.OracleSystem(m, x, v, eps)
    Kg0, Wg0 = g.nb_energy()
    mism = 0
    n_blocks = 0
    while True:
        tg, ng, actg = g.nb_next_block()
        if tg > 0.125:
            break
        to, acto = o.next_block()
        if not (tg == to and np.array_equal(actg, acto)):
            mism += 1
            break
        g.nb_predict(tg); g.nb_force(actg, outputs=False); g.nb_corrector(actg, 0.0)
        o.predict(to); o.force(acto); o.corrector(acto, 0.0)
        n_blocks += 1
    assert mism == 0, f"schedules diverged after {n_blocks} block steps"
    assert np.all(g.nb_get_state("T") == 0.125)
    assert relvec(g.nb_get_state("X"), o.x).max() < 1e-9
    Kg, Wg = g.nb_energy()
    Ko, Wo = o.energy()
    assert abs((Kg + Wg) - (Ko + Wo)) / abs(Ko + Wo) < 1e-10
    assert abs((Kg + Wg) / (Kg0 + Wg0) - 1) < 1e-5
    g.nb_free()


# ------------------------------------------------------------------ 4th-order variant (nb_config.order = 4; R21)
def test_order4_force_steps_and_block_steps(B, oracle):
    N, eps = 1500, 1e-3
    m, x, v = W.plummer(N, 4004, "kroupa")
    g = B.System(m, x, v, eps, order=4)
    o = oracle.OracleSystem(m, x, v, eps, order=4)
    # startup: one evaluation gives a and jerk; snap = crackle = 0; same levels
    for f, ref in (("A", o.a), ("J", o.j)):
        assert relvec(g.nb_get_state(f), ref).max() <= TOL
    assert not g.nb_get_state("S").any() and not g.nb_get_state("C").any()
    assert np.array_equal(g.nb_get_state("DT"), o.dt)
    # shared steps: predictor, force (all three kernel shapes), corrector
    dt = 2.0 ** -9
    rng = np.random.default_rng(44)
    for step in range(1, 5):
        g.nb_predict(step * dt); o.predict(step * dt)
        for f, ref in (("XP", o.xp), ("VP", o.vp)):
            assert relvec(g.nb_get_state(f), ref).max() <= 1e-13, f
        if step == 2:
            for n_act in (1, 7, 16, 17, 64, 96, 97, 300):
                idx = rng.choice(N, n_act, replace=False).astype(np.int32)
                ga, gj, gs, gp = g.nb_force(idx)
                oa, oj, _, op = oracle_on_gpu_records(oracle, g, eps, idx)
                assert relvec(ga, oa).max() <= TOL and relvec(gj, oj).max() <= TOL and np.abs(gp / op - 1).max() <= TOL
                assert not gs.any()                                           # snap is not evaluated at this order
        ga, gj, gs, gp = g.nb_force()
        oa, oj, _, op = o.force()
        assert relvec(ga, oa).max() <= 1e-10 and relvec(gj, oj).max() <= 1e-10        # states differ at round-off after a step
        g.nb_corrector(None, dt); o.corrector(None, dt)
    for f, ref, tol in (("X", o.x, 1e-13), ("V", o.v, 1e-12), ("A", o.a, 1e-10), ("J", o.j, 1e-10)):
        assert relvec(g.nb_get_state(f), ref).max() <= tol, f
    # the interpolant's a'' and a''' amplify a force difference delta by 6/h^2 and 12/h^3 (see the crackle bound above)
    nrm = lambda q: np.linalg.norm(q, axis=-1)
    delta = 1e-11
    scale = nrm(o.a) + dt * nrm(o.j)
    assert np.all(nrm(g.nb_get_state("S") - o.s) <= delta * 12 * scale / dt ** 2)
    assert np.all(nrm(g.nb_get_state("C") - o.c) <= delta * 24 * scale / dt ** 3)
    Kg, Wg = g.nb_energy(); Ko, Wo = o.energy()
    assert abs((Kg + Wg) - (Ko + Wo)) / abs(Ko + Wo) < 1e-10
    g.nb_free()
    # block steps: same schedule on both sides, then nb_run_blocks bit-identical to the separate calls
    N = 384
    m, x, v = W.plummer(N, 4005, "kroupa")
    g, g2 = B.System(m, x, v, eps, order=4), B.System(m, x, v, eps, order=4)
    o = oracle.OracleSystem(m, x, v, eps, order=4)
    steps = 0
    while True:
        tg, ng, actg = g.nb_next_block()
        to, acto = o.next_block()
        assert tg == to and np.array_equal(actg, acto)
        if to > 2.0 ** -5:
            break
        g.nb_predict(tg); g.nb_force(actg, outputs=False); g.nb_corrector(actg, 0.0)
        o.predict(to); o.force(acto); o.corrector(acto, 0.0)
        assert np.array_equal(g.nb_get_state("DT"), o.dt)
        steps += 1
    assert steps > 20
    assert relvec(g.nb_get_state("X"), o.x).max() <= 1e-12
    s2, t2, _ = g2.nb_run_blocks(2.0 ** -5)
    assert s2 == steps and t2 == 2.0 ** -5
    for f in ("X", "V", "A", "J", "S", "C", "T", "DT"):
        assert np.array_equal(g.nb_get_state(f), g2.nb_get_state(f)), f
    g.nb_free(); g2.nb_free()


def test_order_is_validated(B):
    m, x, v = W.plummer(64, 1)
    for bad in (2, 5, 10):
        with pytest.raises(B.NBError):
            B.System(m, x, v, 1e-3, order=bad)


# ------------------------------------------------------------------ 8th-order variant (nb_config.order = 8; R22)
def test_order8_force_steps_and_block_steps(B, oracle):
    N, eps = 1500, 1e-3
    m, x, v = W.plummer(N, 8008, "kroupa")
    g = B.System(m, x, v, eps, order=8)
    o = oracle.OracleSystem(m, x, v, eps, order=8)
    # three-pass startup: a, jerk, snap, crackle; a4 = a5 = 0; same levels
    for f, ref in (("A", o.a), ("J", o.j), ("S", o.s), ("C", o.c)):
        assert relvec(g.nb_get_state(f), ref).max() <= TOL, f
    assert not g.nb_get_state("A4").any() and not g.nb_get_state("A5").any()
    assert np.array_equal(g.nb_get_state("DT"), o.dt)
    dt = 2.0 ** -8
    rng = np.random.default_rng(88)
    for step in range(1, 5):
        g.nb_predict(step * dt); o.predict(step * dt)
        # after the first step a4, a5 enter the predictor; they are 4th / 5th differences over the step, so a force
        # difference delta is amplified by ~105/hh^4, 315/hh^5 (hh = dt/2) whatever the implementation: with D = dt the
        # predicted jerk inherits ~200 delta |a| / hh, the predicted acceleration ~100 delta |a|
        tols = (1e-12, 1e-12, 1e-12, 1e-12) if step == 1 else (1e-12, 1e-11, 1e-9, None)
        for (f, ref), tol in zip((("XP", o.xp), ("VP", o.vp), ("AP", o.ap), ("JP", o.jp)), tols):
            if tol is not None:
                assert relvec(g.nb_get_state(f), ref).max() <= tol, (f, step)
            else:
                bound = 1e-11 * 200 * (np.linalg.norm(o.a, axis=-1) + dt * np.linalg.norm(o.j, axis=-1)) / (dt / 2)
                assert np.all(np.linalg.norm(g.nb_get_state(f) - ref, axis=-1) <= bound), (f, step)
        if step == 3:                                    # all three kernel shapes on identical records
            mm = g.nb_get_state("M")
            rec = [g.nb_get_state(f) for f in ("XP", "VP", "AP", "JP")]
            for n_act in (1, 7, 16, 17, 64, 96, 97, 300):
                idx = rng.choice(N, n_act, replace=False).astype(np.int32)
                ga, gj, gs, gp = g.nb_force(idx)
                gc = g.nb_force_crackle(n_act)
                oa, oj, os_, oc, op = oracle.hermite6.force8(mm, *rec, eps, idx)
                assert_force_parity((ga, gj, gs, gp), (oa, oj, os_, op))
                assert relvec(gc, oc).max() <= TOL, ("crackle", n_act, relvec(gc, oc).max())
        ga, gj, gs, gp = g.nb_force()
        gc = g.nb_force_crackle(N)
        oa, oj, os_, op, oc = o.force()
        assert_force_parity((ga, gj, gs, gp), (oa, oj, os_, op), 1e-9)     # states differ at round-off after a step
        assert relvec(gc, oc).max() <= 1e-8
        g.nb_corrector(None, dt); o.corrector(None, dt)
    for f, ref, tol in (("X", o.x, 1e-13), ("V", o.v, 1e-12), ("A", o.a, 1e-9), ("C", o.c, 1e-8)):
        assert relvec(g.nb_get_state(f), ref).max() <= tol, f
    # a4, a5 are fourth / fifth differences over the step: a relative force difference delta is amplified by ~105/hh^4, 315/hh^5
    nrm = lambda q: np.linalg.norm(q, axis=-1)
    hh, delta = dt / 2, 1e-9
    scale = nrm(o.a) + hh * nrm(o.j) + hh ** 2 * nrm(o.s) + hh ** 3 * nrm(o.c)
    assert np.all(nrm(g.nb_get_state("A4") - o.a4) <= delta * 400 * scale / hh ** 4)
    assert np.all(nrm(g.nb_get_state("A5") - o.a5) <= delta * 1200 * scale / hh ** 5)
    Kg, Wg = g.nb_energy(); Ko, Wo = o.energy()
    assert abs((Kg + Wg) - (Ko + Wo)) / abs(Ko + Wo) < 1e-10
    g.nb_free()
    # block steps: same schedule on both sides, then nb_run_blocks bit-identical to the separate calls
    N = 384
    m, x, v = W.plummer(N, 8009, "kroupa")
    g, g2 = B.System(m, x, v, eps, order=8), B.System(m, x, v, eps, order=8)
    o = oracle.OracleSystem(m, x, v, eps, order=8)
    steps = 0
    while True:
        tg, ng, actg = g.nb_next_block()
        to, acto = o.next_block()
        assert tg == to and np.array_equal(actg, acto)
        if to > 2.0 ** -5:
            break
        g.nb_predict(tg); g.nb_force(actg, outputs=False); g.nb_corrector(actg, 0.0)
        o.predict(to); o.force(acto); o.corrector(acto, 0.0)
        assert np.array_equal(g.nb_get_state("DT"), o.dt)
        steps += 1
    assert steps > 20
    assert relvec(g.nb_get_state("X"), o.x).max() <= 1e-12
    s2, t2, _ = g2.nb_run_blocks(2.0 ** -5)
    assert s2 == steps and t2 == 2.0 ** -5
    for f in ("X", "V", "A", "J", "S", "C", "A4", "A5", "T", "DT"):
        assert np.array_equal(g.nb_get_state(f), g2.nb_get_state(f)), f
    g.nb_free(); g2.nb_free()


@pytest.mark.parametrize("order", [4, 8])
@pytest.mark.parametrize("N,eps", [(2, 0.0), (257, 0.0), (1, 1e-3), (300, 1e-2)])
def test_other_orders_edge_sizes(B, oracle, order, N, eps):
    """Degenerate and ragged sizes at the 4th and 8th order: N = 1 (no pairs: all sums 0), N = 2 unsoftened, a ragged
    N with eps = 0 (index-masked self pair), a permuted full list, an empty active set."""
    m, x, v = W.plummer(max(N, 2), 900 + N + order, "kroupa")
    m, x, v = m[:N].copy(), x[:N].copy(), v[:N].copy()
    g = B.System(m, x, v, eps, order=order)
    g.nb_predict(2.0 ** -10)
    assert g.nb_force(np.zeros(0, dtype=np.int32))[0].shape == (0, 3)        # n_act = 0 is a no-op
    rng = np.random.default_rng(N)
    perm = rng.permutation(N).astype(np.int32)
    ga, gj, gs, gp = g.nb_force(perm)
    mm = g.nb_get_state("M")
    rec = [g.nb_get_state(f) for f in ("XP", "VP", "AP")]
    if N == 1:
        assert not ga.any() and not gj.any() and not gs.any() and not gp.any()
        g.nb_free()
        return
    if order == 8:
        gc = g.nb_force_crackle(N)
        oa, oj, os_, oc, op = oracle.hermite6.force8(mm, *rec, g.nb_get_state("JP"), eps, perm)
        assert_force_parity((ga, gj, gs, gp), (oa, oj, os_, op))
        assert relvec(gc, oc).max() <= TOL
    else:
        oa, oj, _, op = oracle.hermite6.force(mm, *rec, eps, perm)
        assert relvec(ga, oa).max() <= TOL and relvec(gj, oj).max() <= TOL and np.abs(gp / op - 1).max() <= TOL
        assert not gs.any()
    g.nb_corrector(perm, 2.0 ** -10)
    assert np.all(g.nb_get_state("T") == 2.0 ** -10) and np.isfinite(g.nb_get_state("X")).all()
    g.nb_free()


def test_max_split_and_probes(B, oracle):
    """nb_set_max_split(1) (the "Bfactor off" arm of the Fig. 1 sweep) changes the launch, not the result beyond the
    summation order; the operand-source probes return the pipe model's 2 / 3 / 2-3 cycles."""
    N, eps = 5000, 1e-3
    m, x, v = W.plummer(N, 606)
    g = B.System(m, x, v, eps)
    g.nb_predict(2.0 ** -9)
    for n_act in (3, 40, 700, N):
        idx = None if n_act == N else np.random.default_rng(n_act).choice(N, n_act, replace=False).astype(np.int32)
        g.nb_set_max_split(0); split = g.nb_force(idx)
        g.nb_set_max_split(1); nosplit = g.nb_force(idx)
        ref = oracle_on_gpu_records(oracle, g, eps, idx)
        assert_force_parity(split, ref); assert_force_parity(nosplit, ref)
    g.nb_set_max_split(0)
    with pytest.raises(B.NBError):
        g.nb_set_max_split(-1)
    g.nb_free()
    from paper_1411_5234_b200 import probes
    cyc = probes.dfma_sources(1965.0)
    assert 1.9 < cyc["two_sources"] < 2.4 and 2.8 < cyc["three_sources"] < 3.5
    assert cyc["two_sources"] <= cyc["three_sources_one_reused"] <= cyc["three_sources"]
    # a context keeps working after a probe ran on the device in between (every entry point sets its own device)
    g = B.System(m, x, v, eps)
    probes.fp64_peak(0.05)
    g.nb_predict(2.0 ** -9)
    assert np.isfinite(g.nb_force(None)[0]).all()
    g.nb_free()


# ------------------------------------------------------------------ boundary: index verification, devices, tiny eps
def test_bad_index_lists_are_rejected(B):
    """nb_config.check_indices (default: on for host-pointer contexts): an out-of-range or duplicate index returns
    NB_EINVAL before anything reads through the list; the context stays usable."""
    import torch
    N = 3000
    m, x, v = W.plummer(N, 31)
    g = B.System(m, x, v, 1e-3)
    g.nb_predict(2.0 ** -10)
    good = W.active_set(N, 200, 1)
    for bad in (np.array([5, N, 7], dtype=np.int32), np.array([-1], dtype=np.int32), np.array([2 ** 31 - 1, 0], dtype=np.int32)):
        with pytest.raises(B.NBError) as e:
            g.nb_force(bad)
        assert e.value.status == B.NB_EINVAL
        with pytest.raises(B.NBError) as e:
            g.nb_get_state("X", bad)
        assert e.value.status == B.NB_EINVAL
        with pytest.raises(B.NBError) as e:
            g.nb_set_state("X", np.zeros((bad.size, 3)), bad)
        assert e.value.status == B.NB_EINVAL
        assert g.nb_check_indices(bad) == B.NB_EINVAL
    dup = np.array([4, 9, 4], dtype=np.int32)
    with pytest.raises(B.NBError) as e:
        g.nb_force(dup)
    assert e.value.status == B.NB_EINVAL
    assert g.nb_check_indices(dup) == B.NB_EINVAL and g.nb_check_indices(dup, unique=False) == B.NB_OK
    assert np.array_equal(g.nb_get_state("X", dup), x[dup])                     # reading the same particle twice is fine
    assert g.nb_check_indices(good) == B.NB_OK and g.nb_check_indices(np.arange(N, dtype=np.int32)) == B.NB_OK
    # nothing was corrupted, the context still works, and the corrector refuses a bad list too
    fa = g.nb_force(good)
    with pytest.raises(B.NBError) as e:
        g.nb_corrector(np.concatenate([good[:-1], good[:1]]), 2.0 ** -10)
    assert e.value.status == B.NB_EINVAL
    g.nb_corrector(good, 2.0 ** -10)
    assert np.isfinite(g.nb_get_state("X")).all() and np.array_equal(g.nb_get_state("M"), m)
    g.nb_free()
    # device-pointer context: off by default (asynchronous calls), on when asked for
    dev = "cuda:0"
    args = (torch.tensor(m, device=dev), torch.tensor(x, device=dev), torch.tensor(v, device=dev))
    gd = B.System(*args, 1e-3, host=False, check_indices=1)
    gd.nb_predict(2.0 ** -10)
    with pytest.raises(B.NBError) as e:
        gd.nb_force(torch.tensor([1, N + 5], dtype=torch.int32, device=dev))
    assert e.value.status == B.NB_EINVAL
    assert gd.nb_check_indices(torch.tensor(good, device=dev)) == B.NB_OK
    gd.nb_free()
    gh = B.System(m, x, v, 1e-3, check_indices=-1)                               # host pointers, checking switched off
    assert gh.nb_check_indices(dup) == B.NB_EINVAL                               # the explicit call still checks
    gh.nb_free()


def test_contexts_survive_a_device_switch(B):
    """Every entry point runs on its context's device whatever the caller's current device is (two GPUs needed for the
    cross-device part; on one GPU the call sequence still runs with the guard in place)."""
    import torch
    N = 2000
    m, x, v = W.plummer(N, 32)
    g = B.System(m, x, v, 1e-3)
    ref = B.System(m, x, v, 1e-3)
    other = 1 if torch.cuda.device_count() > 1 else 0
    torch.cuda.set_device(other)
    try:
        for s_ in (g, ref):
            if s_ is ref:
                torch.cuda.set_device(0)
            t, n, act = s_.nb_next_block()
            s_.nb_predict(t); s_.nb_force(act, outputs=False); s_.nb_corrector(act, 0.0)
            s_.nb_run_blocks(2.0 ** -6, max_steps=5)
            E = s_.nb_energy()
        assert torch.cuda.current_device() == 0
        torch.cuda.set_device(other)
        xg = g.nb_get_state("X")
        assert torch.cuda.current_device() == other                              # the caller's device is restored
    finally:
        torch.cuda.set_device(0)
    assert np.array_equal(xg, ref.nb_get_state("X"))
    g.nb_free(); ref.nb_free()


def test_tiny_softening_is_treated_as_zero(B, oracle):
    """0 < eps < 1.5e-154: eps^2 underflows; the launch must take the index-masked (eps = 0) kernels, not produce NaN."""
    N = 600
    m, x, v = W.plummer(N, 33)
    g0, g1 = B.System(m, x, v, 0.0), B.System(m, x, v, 1e-160)
    for f in ("A", "J", "S"):
        a0, a1 = g0.nb_get_state(f), g1.nb_get_state(f)
        assert np.isfinite(a1).all() and np.array_equal(a0, a1), f
    g1.nb_predict(2.0 ** -10)
    for n_act in (3, 50, N):
        idx = None if n_act == N else W.active_set(N, n_act, 2)
        got = g1.nb_force(idx)
        assert_force_parity(got, oracle_on_gpu_records(oracle, g1, 0.0, idx))
    g0.nb_free(); g1.nb_free()


# ------------------------------------------------------------------ f4: mixed precision, f1: the step log
def test_mixed_precision_accuracy_against_oracle(B, oracle, capsys):
    """nb_config.precision = NB_PREC_MIXED: fp64 position differences and accumulation, fp32 elsewhere (the precision scheme of
    the paper's template), for evaluations that run as CTA tiles.  Its per-particle error against the long-double
    oracle is MEASURED here and bounded; smaller active sets must still be fp64-exact."""
    N, eps = 20000, 1e-4
    m, x, v = W.plummer(N, 4242)
    g = B.System(m, x, v, eps, precision=B.NB_PREC_MIXED)
    g64 = B.System(m, x, v, eps)
    t = 2.0 ** -8
    for s_ in (g, g64):
        s_.nb_predict(t)
    assert B.nb_plan_force(N, N).kernel == 0
    got = g.nb_force()
    ref = oracle_on_gpu_records(oracle, g64, eps, None)
    errs = [relvec(a, b) for a, b in zip(got[:3], ref[:3])] + [np.abs(got[3] / ref[3] - 1)]
    with capsys.disabled():
        print("\n[mixed precision] N = %d all active, error vs oracle: " % N +
              ", ".join(f"{n} max {e.max():.2e} median {np.median(e):.2e}" for n, e in zip(("acc", "jerk", "snap", "pot"), errs)))
    assert errs[0].max() > 1e-9                                                  # this really is the fp32 pair arithmetic
    for e, bound in zip(errs, (2e-5, 1e-4, 1e-3, 2e-6)):
        assert e.max() <= bound, (e.max(), bound)
    assert np.median(errs[0]) <= 2e-6 and np.median(errs[1]) <= 5e-6 and np.median(errs[2]) <= 2e-5
    # Newton's third law holds to fp32 round-off of the pair terms
    for arr in got[:3]:
        assert np.abs((m[:, None] * arr).sum(0)).max() <= 1e-5 * (m[:, None] * np.abs(arr)).sum()
    # a small active set runs as warp units: fp64 as ever
    idx = W.active_set(N, 100, 3)
    assert_force_parity(g.nb_force(idx), oracle_on_gpu_records(oracle, g, eps, idx))
    # a few shared steps: energy conserved to single-precision-force level, run_blocks works in this mode too
    K0, W0 = g.nb_energy()
    for k in range(1, 5):
        g.nb_predict(k * 2.0 ** -10); g.nb_force(outputs=False); g.nb_corrector(None, 2.0 ** -10)
    K1, W1 = g.nb_energy()
    E0_64 = sum(g64.nb_energy())
    for k in range(1, 5):
        g64.nb_predict(k * 2.0 ** -10); g64.nb_force(outputs=False); g64.nb_corrector(None, 2.0 ** -10)
    d_mixed, d_64 = (K1 + W1) / (K0 + W0) - 1, sum(g64.nb_energy()) / E0_64 - 1
    with capsys.disabled():
        print(f"[mixed precision] dE/E over 4 shared steps: mixed {d_mixed:.3e}, fp64 {d_64:.3e}")
    assert abs(d_mixed) < 1e-4 and abs(d_mixed - d_64) < 2e-5
    steps, _, _ = g.nb_run_blocks(1e30, 5)
    assert steps == 5 and np.isfinite(g.nb_get_state("X")).all()
    g.nb_free(); g64.nb_free()
    with pytest.raises(B.NBError):
        B.System(m, x, v, eps, precision=B.NB_PREC_MIXED, order=4)
    with pytest.raises(B.NBError):
        B.System(m, x, v, eps, precision=7)


def test_step_log_records_every_block_step(B):
    N = 3000
    m, x, v = W.plummer(N, 515, "kroupa")
    g = B.System(m, x, v, 1e-4)
    s1, _, a1 = g.nb_run_blocks(1e30, 40)
    na, tu = g.nb_step_log()
    assert s1 == 40 and na.size == 40 and na.sum() == a1 and tu[0] == 0.0 and np.all(np.diff(tu) > 0)
    s2, _, a2 = g.nb_run_blocks(1e30, 25)
    na2, tu2 = g.nb_step_log(30)
    assert na2.size == 30 and na2[5:].sum() == a2 and np.array_equal(na2[:5], na[-5:])   # the last 30 of 65, oldest first
    assert np.all((na2 >= 1) & (na2 <= N))
    g.nb_free()


def test_workspace_guard_bands_stay_untouched(B):
    """Memory safety without compute-sanitizer (closed on this pool, profiles/r02_sanitizer.md): 1 MiB bands of 0xA5 on both
    sides of the workspace must survive every kernel of the library - all force shapes at ragged sizes, block steps through
    the graph and by separate calls, the index check, state I/O, the other orders and the mixed-precision records."""
    N = 4099                                                 # ragged: pads to 4352
    m, x, v = W.plummer(N, 616, "kroupa")
    for kw in (dict(), dict(order=4), dict(order=8), dict(precision=B.NB_PREC_MIXED)):
        g = B.System(m, x, v, 1e-4, guard_bytes=1 << 20, **kw)
        assert g.guards_intact()
        g.nb_run_blocks(1e30, 20)
        for _ in range(4):
            tn, n, act = g.nb_next_block()
            g.nb_predict(tn); g.nb_force(act, outputs=False); g.nb_corrector(act, 0.0)
        g.nb_predict(tn)
        for n_act in (1, 5, 17, 31, 100, 300, 1024, 4000, N):
            g.nb_force(None if n_act == N else W.active_set(N, n_act, n_act))
        assert g.nb_check_indices(np.array([N - 1, 0, N - 1], dtype=np.int32)) == B.NB_EINVAL
        g.nb_set_state("X", x[-3:], np.array([N - 1, N - 2, N - 3], dtype=np.int32))
        g.nb_get_state("S"); g.nb_energy(); g.nb_step_log()
        assert g.guards_intact(), kw
        g.nb_free()


# ------------------------------------------------------------------ the rescheduled machine code against ptxas's own
def test_sass_sched_build_is_bitwise_the_ptxas_build(B, tmp_path):
    """sass_sched.py permutes and re-registers the instructions of the FP64 pair loops; the arithmetic is untouched, so every
    result has to be bit-identical to the library built from the cubin as ptxas emitted it (libnb_ptxas.so, build.py)."""
    import os, subprocess, sys
    from paper_1411_5234_b200 import build
    if not build.sass_sched_enabled() or not os.path.exists(build.PTXAS_LIB):
        pytest.skip("built without sass_sched (NB_SASS_SCHED=0)")
    log = os.path.join(build.HERE, "build", "keep_nb_force", "sass_sched.log")
    if os.path.exists(log):
        assert "sass_sched: 0 blocks rescheduled" not in open(log).read(), "the scheduler changed nothing: nothing to compare"
    files = {}
    for name, libpath in (("sched", build.LIB), ("ptxas", build.PTXAS_LIB)):
        files[name] = str(tmp_path / f"{name}.npz")
        env = dict(os.environ, NB_LIB=libpath)
        subprocess.run([sys.executable, "-m", "paper_1411_5234_b200.dump_case", files[name]], check=True, env=env,
                       cwd=os.path.dirname(build.HERE))
    a, b = np.load(files["sched"]), np.load(files["ptxas"])
    assert sorted(a.files) == sorted(b.files) and len(a.files) > 90
    for k in a.files:
        x, y = a[k], b[k]
        assert x.dtype == y.dtype and x.shape == y.shape
        assert not np.isnan(x).any(), k
        assert np.array_equal(x.view(np.uint64), y.view(np.uint64)), (k, int((x != y).sum()))
