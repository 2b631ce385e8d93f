"""Pins of the CPU oracle against things other than itself (prompt section 3).

Each test names the part of oracle/nb_oracle.c it pins and what it is pinned to.  None of them
touches the CUDA path.
"""
import os

import mpmath as mp
import numpy as np
import pytest

from paper_1411_5234_b200 import workloads as W

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def circular_binary(eps):
    s = 1.0 + eps * eps
    omega = np.sqrt(1.0 / s ** 1.5)
    m = np.array([0.5, 0.5])
    x = np.array([[0.5, 0, 0], [-0.5, 0, 0]], dtype=np.float64)
    v = np.array([[0, 0.5 * omega, 0], [0, -0.5 * omega, 0]], dtype=np.float64)
    return m, x, v, omega, s


# ---------------------------------------------------------------- P1: closed form, golden values
def test_p1_circular_binary_closed_form_and_startup(oracle):
    rows = [l.split() for l in open(os.path.join(GOLDEN, "circular_binary.txt")) if l.strip() and l[0] != "#"]
    assert len(rows) == 2
    for row in rows:
        eps, g_omega, g_ax, g_jy, g_sx, g_pot = map(float, row)
        m, x, v, omega, s = circular_binary(eps)
        sysm = oracle.OracleSystem(m, x, v, eps)           # two-pass startup (O5) -> a, jerk, snap
        a, j, sn = sysm.a[0], sysm.j[0], sysm.s[0]
        # against the printed values (12 digits)
        assert abs(omega - g_omega) < 2e-12
        assert abs(a[0] - g_ax) < 2e-11 and abs(j[1] - g_jy) < 2e-11 and abs(sn[0] - g_sx) < 2e-11
        assert abs(sysm.pot0[0] - g_pot) < 2e-11
        # against the closed form, to rounding: a1 = (-1/2 s^-3/2,0,0), jerk = omega x a, snap = -omega^2 a
        ax = -0.5 * s ** -1.5
        np.testing.assert_allclose(a, [ax, 0, 0], rtol=0, atol=4e-16)
        np.testing.assert_allclose(j, [0, omega * ax, 0], rtol=0, atol=4e-16)
        np.testing.assert_allclose(sn, [-omega ** 2 * ax, 0, 0], rtol=0, atol=4e-16)
        np.testing.assert_allclose(sysm.pot0, [-0.5 * s ** -0.5] * 2, rtol=0, atol=4e-16)
        # particle 2 is the mirror image
        np.testing.assert_allclose(sysm.a[1], -a, atol=1e-16)
        np.testing.assert_allclose(sysm.j[1], -j, atol=1e-16)
        np.testing.assert_allclose(sysm.s[1], -sn, atol=1e-16)


def test_startup_levels_closed_form_on_circular_binary(oracle):
    """O5 (oracle_startup_levels, reading R8/R11): on the circular binary |jerk| = omega |a| exactly, so the startup step is
    dt0 = 2^floor(log2(eta_s / omega)) clamped to [2^k_min, 2^k_max].  eta_s values chosen so that eta_s/omega and
    eta_s*omega (|a| and |jerk| swapped) fall on different sides of a power of two, plus both clamps."""
    for eps, d in ((0.0, 1.0), (0.1, 1.0), (0.0, 0.25), (0.1, 0.5)):
        s = d * d + eps * eps
        omega = np.sqrt(1.0 / s ** 1.5)                     # M = 1: omega^2 = M / (d^2 + eps^2)^(3/2)
        m = np.array([0.5, 0.5])
        x = np.array([[0.5 * d, 0, 0], [-0.5 * d, 0, 0]])
        v = np.array([[0, 0.5 * d * omega, 0], [0, -0.5 * d * omega, 0]])
        for eta_s in (0.01, 2.0 ** -6 * 0.999 * omega, 2.0 ** -6 * 1.001 * omega, 2.0 ** -9 * 1.3, 0.3):
            o = oracle.OracleSystem(m, x, v, eps, eta_s=eta_s)
            k = int(np.floor(np.log2(eta_s / omega)))
            assert np.all(o.dt == 2.0 ** min(max(k, -20), -3)), (eps, d, eta_s, o.dt, k)
        # the two values around 2^-6 really straddle the power of two
        assert np.floor(np.log2(2.0 ** -6 * 0.999)) == -7 and np.floor(np.log2(2.0 ** -6 * 1.001)) == -6
        # clamps
        assert np.all(oracle.OracleSystem(m, x, v, eps, eta_s=1e-9).dt == 2.0 ** -20)
        assert np.all(oracle.OracleSystem(m, x, v, eps, eta_s=50.0).dt == 2.0 ** -3)
        assert np.all(oracle.OracleSystem(m, x, v, eps, eta_s=0.01, k_min=-5, k_max=-4).dt == 2.0 ** -5)


# ---------------------------------------------------------------- P9: 50-digit brute force + differentiation
@pytest.mark.parametrize("N,eps,seed", [(2, 0.0, 1), (3, 0.05, 2), (3, 0.0, 3), (4, 0.3, 4)])
def test_p9_tiny_systems_against_mpmath(oracle, N, eps, seed):
    """a, pot by the definition (eq. 1-2) and jerk, snap by differentiating a(tau) along
    x(tau) = x + v tau + a_p tau^2/2, all in 50-digit arithmetic.  Pins every coefficient of O1."""
    mp.mp.dps = 50
    rng = np.random.default_rng(seed)
    m = rng.uniform(0.2, 1.0, N)
    x, v, ap = rng.normal(size=(N, 3)), rng.normal(size=(N, 3)), rng.normal(size=(N, 3))
    idx = np.arange(N, dtype=np.int32)[::-1].copy()           # also pins the row k <-> idx[k] mapping
    acc, jerk, snap, pot = oracle.hermite6.force(m, x, v, ap, eps, idx)

    def a_of_tau(i, c, tau):
        tot = mp.mpf(0)
        for jj in range(N):
            if jj == i:
                continue
            d = [(mp.mpf(x[jj, k]) + mp.mpf(v[jj, k]) * tau + mp.mpf(ap[jj, k]) * tau ** 2 / 2)
                 - (mp.mpf(x[i, k]) + mp.mpf(v[i, k]) * tau + mp.mpf(ap[i, k]) * tau ** 2 / 2) for k in range(3)]
            s = d[0] ** 2 + d[1] ** 2 + d[2] ** 2 + mp.mpf(eps) ** 2
            tot += mp.mpf(m[jj]) * d[c] / s ** mp.mpf(1.5)
        return tot

    for k, i in enumerate(idx):
        for c in range(3):
            a_ref = a_of_tau(i, c, mp.mpf(0))
            j_ref = mp.diff(lambda t: a_of_tau(i, c, t), 0, 1)
            s_ref = mp.diff(lambda t: a_of_tau(i, c, t), 0, 2)
            scale_a = max(abs(float(a_ref)), 1e-3)
            assert abs(acc[k, c] - float(a_ref)) <= 4e-16 * max(scale_a, np.abs(acc[k]).max())
            assert abs(jerk[k, c] - float(j_ref)) <= 4e-16 * max(abs(float(j_ref)), np.abs(jerk[k]).max())
            assert abs(snap[k, c] - float(s_ref)) <= 4e-16 * max(abs(float(s_ref)), np.abs(snap[k]).max())
        p_ref = -sum(mp.mpf(m[jj]) / mp.sqrt(sum((mp.mpf(x[jj, q]) - mp.mpf(x[i, q])) ** 2 for q in range(3))
                                              + mp.mpf(eps) ** 2) for jj in range(N) if jj != i)
        assert abs(pot[k] - float(p_ref)) <= 4e-16 * abs(float(p_ref))


# ---------------------------------------------------------------- P2: Newton's third law
def test_p2_newtons_third_law(oracle):
    m, x, v = W.plummer(64, 7, "kroupa")
    sysm = oracle.OracleSystem(m, x, v, 1e-2)
    for arr in (sysm.a, sysm.j, sysm.s):
        total = (m[:, None] * arr).sum(0)
        scale = (m[:, None] * np.abs(arr)).sum()
        assert np.abs(total).max() <= 1e-15 * scale


# ---------------------------------------------------------------- P3: finite differences of a
def test_p3_finite_differences_reproduce_jerk_and_snap(oracle):
    N, eps, h = 64, 1e-2, 1e-3
    m, x, v = W.plummer(N, 11)
    sysm = oracle.OracleSystem(m, x, v, eps)
    a0 = sysm.a.copy()

    def acc_at(tau):
        xt = x + v * tau + a0 * tau ** 2 / 2 + sysm.j * tau ** 3 / 6 + sysm.s * tau ** 4 / 24
        return oracle.hermite6.force(m, xt, np.zeros_like(x), np.zeros_like(x), eps, want=("a",))[0]

    am2, am1, a00, ap1, ap2 = acc_at(-2 * h), acc_at(-h), acc_at(0.0), acc_at(h), acc_at(2 * h)
    jerk_fd = (am2 - 8 * am1 + 8 * ap1 - ap2) / (12 * h)
    snap_fd = (-am2 + 16 * am1 - 30 * a00 + 16 * ap1 - ap2) / (12 * h * h)
    rel_j = np.linalg.norm(jerk_fd - sysm.j, axis=1) / np.linalg.norm(sysm.j, axis=1)
    rel_s = np.linalg.norm(snap_fd - sysm.s, axis=1) / np.linalg.norm(sysm.s, axis=1)
    assert rel_j.max() < 2e-5 and rel_s.max() < 2e-5


# ---------------------------------------------------------------- P4: polynomial exactness
def test_p4_predictor_exact_for_quintic(oracle):
    rng = np.random.default_rng(5)
    N = 7
    # x(t) = sum_k c_k (t - t_i)^k / k!, k = 0..5  ->  x, v, a, j, s, c are the c_k
    coef = rng.normal(size=(6, N, 3))
    ti = rng.choice([0.0, 0.25, 0.5, 0.625], N)
    t = 0.75
    xp, vp, ap = np.zeros((N, 3)), np.zeros((N, 3)), np.zeros((N, 3))
    L = oracle.lib("ld")
    P = oracle.hermite6._p
    L.oracle_predict(N, t, P(ti), *[P(np.ascontiguousarray(c)) for c in coef], P(xp), P(vp), P(ap))
    D = (t - ti)[:, None]
    fact = [1, 1, 2, 6, 24, 120]
    x_ref = sum(coef[k] * D ** k / fact[k] for k in range(6))
    v_ref = sum(coef[k] * D ** (k - 1) / fact[k - 1] for k in range(1, 6))
    a_ref = sum(coef[k] * D ** (k - 2) / fact[k - 2] for k in range(2, 6))
    np.testing.assert_allclose(xp, x_ref, rtol=0, atol=2e-15)
    np.testing.assert_allclose(vp, v_ref, rtol=0, atol=2e-15)
    np.testing.assert_allclose(ap, a_ref, rtol=0, atol=2e-15)


def test_p4_corrector_exact_for_polynomial_acceleration(oracle):
    """If a(t) is a polynomial of degree <= 5 the velocity corrector and the recovered a''', a'''',
    a''''' are exact; for degree <= 4 the position corrector is exact too (Hermite quadrature)."""
    rng = np.random.default_rng(6)
    L = oracle.lib("ld")
    P = oracle.hermite6._p
    for deg in (4, 5):
        h, t0 = 0.25, 0.5
        pa = [np.polynomial.Polynomial(rng.normal(size=deg + 1)) for _ in range(3)]     # a_c(t)
        pv = [p.integ() + rng.normal() for p in pa]
        px = [p.integ() + rng.normal() for p in pv]
        ev = lambda polys, k, t: np.array([[p.deriv(k)(t) if k else p(t) for p in polys]])
        x, v = ev(px, 0, t0), ev(pv, 0, t0)
        a, j, s = ev(pa, 0, t0), ev(pa, 1, t0), ev(pa, 2, t0)
        c = np.zeros((1, 3))
        t1 = t0 + h
        a1, j1, s1 = ev(pa, 0, t1), ev(pa, 1, t1), ev(pa, 2, t1)
        ti, dt = np.array([t0]), np.array([h])
        L.oracle_correct(1, None, 1, h, t1, P(a1), P(j1), P(s1), P(x), P(v), P(a), P(j), P(s), P(c),
                         P(ti), P(dt), 0.45, -20, -3)
        np.testing.assert_allclose(v, ev(pv, 0, t1), rtol=0, atol=1e-14)
        if deg == 4:
            np.testing.assert_allclose(x, ev(px, 0, t1), rtol=0, atol=1e-14)
        np.testing.assert_allclose(c, ev(pa, 3, t1), rtol=0, atol=2e-11)
        np.testing.assert_allclose(a, a1)
        assert ti[0] == t1 and dt[0] == h
        d345 = np.zeros(9)
        L.oracle_hermite_derivs(h, P(ev(pa, 0, t0)), P(ev(pa, 1, t0)), P(ev(pa, 2, t0)), P(a1), P(j1), P(s1), P(d345))
        np.testing.assert_allclose(d345[:3], ev(pa, 3, t1)[0], atol=2e-11)
        np.testing.assert_allclose(d345[3:6], ev(pa, 4, t1)[0], atol=2e-10)
        np.testing.assert_allclose(d345[6:], ev(pa, 5, t1)[0], atol=2e-8)


# ---------------------------------------------------------------- P5: Kepler closed form, 6th order
def kepler_run(oracle, n):
    e = 0.5
    m = np.array([0.5, 0.5])
    x = np.array([[0.75, 0, 0], [-0.75, 0, 0]])
    vy = 0.5 * np.sqrt((1 - e) / (1 + e))
    v = np.array([[0, vy, 0], [0, -vy, 0]])
    sysm = oracle.OracleSystem(m, x, v, 0.0)
    K0, W0 = sysm.energy()
    for _ in range(n):
        sysm.shared_step(2 * np.pi / n)
    K1, W1 = sysm.energy()
    return sysm, np.abs(sysm.x - x).max(), abs((K1 + W1) - (K0 + W0)) / abs(K0 + W0)


def test_p5_kepler_orbit_returns_with_sixth_order_convergence(oracle):
    res = {n: kepler_run(oracle, n) for n in (256, 512, 1024)}
    dx = [res[n][1] for n in (256, 512, 1024)]
    dE = [res[n][2] for n in (256, 512, 1024)]
    # one period brings the orbit back (closed form: period 2 pi for a = 1, M = 1)
    assert dx[0] < 1e-7 and dx[1] < 2e-9 and dx[2] < 4e-11
    assert dE[0] < 2e-8 and dE[2] < 2e-12
    # halving dt divides the error by ~2^6 (allow 40x): the scheme is 6th order
    assert dx[0] / dx[1] > 40 and dx[1] / dx[2] > 40
    assert dE[0] / dE[1] > 40 and dE[1] / dE[2] > 40
    # orbital elements from the final state: a = -M/(2 E_rel), e from the Laplace-Runge-Lenz vector
    s = res[1024][0]
    r, w = s.x[0] - s.x[1], s.v[0] - s.v[1]
    E_rel = 0.5 * w @ w - 1.0 / np.linalg.norm(r)
    ecc = np.cross(w, np.cross(r, w)) - r / np.linalg.norm(r)
    assert abs(-1.0 / (2 * E_rel) - 1.0) < 1e-11 and abs(np.linalg.norm(ecc) - 0.5) < 1e-11
    # 4th-order schemes would fail this; so would a wrong corrector coefficient (1/10, 1/120)


# ---------------------------------------------------------------- P6: time-step criterion
def test_p6_criterion_closed_form_and_levels(oracle):
    L = oracle.lib("ld")
    P = oracle.hermite6._p
    # |a^(k)| = w^k |a|  =>  A1 = sqrt2 w |a|, A4 = sqrt2 w^4 |a|  =>  dt_crit = eta / w exactly
    for w_ in (0.7, 3.0, 41.0):
        d = np.zeros((6, 3))
        for k in range(6):
            d[k, k % 3] = 2.5 * w_ ** k
        dtc = L.oracle_aarseth6_dt(P(d), 0.45)
        assert abs(dtc * w_ / 0.45 - 1) < 1e-15
        assert L.oracle_aarseth6_level(P(d), 0.45, -40, 10) == int(np.floor(np.log2(0.45 / w_)))
    # clamping and degenerate inputs
    d = np.zeros((6, 3)); d[0, 0] = d[1, 0] = d[2, 0] = 1.0           # A4 = 0 -> largest step
    assert L.oracle_aarseth6_level(P(d), 0.45, -20, -3) == -3
    d[3:, 0] = 1e30                                                  # tiny dt_crit -> k_min
    assert L.oracle_aarseth6_level(P(d), 0.45, -20, -3) == -20


def test_p6_criterion_on_integrated_circular_binary(oracle):
    eps = 0.0
    m, x, v, omega, _ = circular_binary(eps)
    sysm = oracle.OracleSystem(m, x, v, eps)
    n = 512
    h = 2 * np.pi / omega / n
    L = oracle.lib("ld")
    P = oracle.hermite6._p
    for _ in range(8):
        a0, j0, s0 = sysm.a.copy(), sysm.j.copy(), sysm.s.copy()
        sysm.shared_step(h)
    d345 = np.zeros(9)
    L.oracle_hermite_derivs(h, P(a0[0].copy()), P(j0[0].copy()), P(s0[0].copy()),
                            P(sysm.a[0].copy()), P(sysm.j[0].copy()), P(sysm.s[0].copy()), P(d345))
    d = np.concatenate([sysm.a[0], sysm.j[0], sysm.s[0], d345])
    assert abs(L.oracle_aarseth6_dt(P(d), 0.45) * omega / 0.45 - 1.0) < 0.01
    # the stored a''' is the interpolant's: |a'''| = omega^3 |a| on the circular orbit
    assert abs(np.linalg.norm(sysm.c[0]) / (omega ** 3 * np.linalg.norm(sysm.a[0])) - 1) < 1e-3


# ---------------------------------------------------------------- P7: energy conservation (config 1)
def test_p7_energy_conservation_config1(oracle):
    c, m, x, v = W.config_inputs(1)

    def drift(dt, n):
        s = oracle.OracleSystem(m, x, v, c.eps)
        K0, W0 = s.energy()
        for _ in range(n):
            s.shared_step(dt)
        K1, W1 = s.energy()
        return abs(K1 + W1 - K0 - W0) / abs(K0 + W0), K0 + W0, K0 / abs(W0)

    d1, E0, Q0 = drift(1.0 / 1024, 8)
    d2, _, _ = drift(1.0 / 512, 4)
    d0, _, _ = drift(1.0 / 2048, 16)
    assert abs(E0 + 0.25) < 0.03 and abs(Q0 - 0.5) < 0.05         # Henon units, virial equilibrium
    # this seed holds a close pair (max |a| = 24, startup level 2^-16), so dt = 1/1024 leaves a
    # truncation error of 2.4e-10; what the method fixes is its ORDER: error / ~2^6 per halving of dt
    assert d1 < 1e-9 and d0 < 1e-11
    assert d2 / d1 > 24 and d1 / d0 > 40


# ---------------------------------------------------------------- P8: Plummer mean field
def test_p8_plummer_mean_field(oracle):
    N = 16384
    m, x, v = W.plummer(N, 99)
    acc = oracle.hermite6.force(m, x, v, np.zeros_like(x), 1e-3, kind="f64", want=("a",))[0]
    r = np.linalg.norm(x, axis=1)
    a_r = (acc * x).sum(1) / r
    aP = 3 * np.pi / 16
    ana = -r / (r * r + aP * aP) ** 1.5
    for lo, hi in [(0.3, 0.6), (0.6, 1.0), (1.0, 2.0), (2.0, 5.0)]:
        sel = (r >= lo) & (r < hi)
        assert sel.sum() > 500
        assert abs(a_r[sel].mean() / ana[sel].mean() - 1) < 0.03


# ---------------------------------------------------------------- scheduler and block steps
def test_scheduler_min_and_active_list(oracle):
    ti = np.array([0.0, 0.25, 0.25, 0.0, 0.375])
    dt = np.array([0.5, 0.125, 0.25, 0.375, 0.125])
    act = np.zeros(5, dtype=np.int32)
    import ctypes as C
    tn = C.c_double()
    n = oracle.lib("ld").oracle_next_block(5, oracle.hermite6._p(ti), oracle.hermite6._p(dt), C.byref(tn),
                                           oracle.hermite6._pi(act))
    assert tn.value == 0.375 and n == 2 and list(act[:2]) == [1, 3]


def test_block_time_steps_stay_on_dyadic_grid_and_conserve_energy(oracle):
    N = 192
    m, x, v = W.plummer(N, 21, "kroupa")
    s = oracle.OracleSystem(m, x, v, 1e-3)
    K0, W0 = s.energy()
    lv = np.log2(s.dt)
    assert np.all(lv == np.round(lv)) and lv.min() >= -20 and lv.max() <= -3
    steps, n_corr = 0, 0
    while True:
        tn, act = s.next_block()
        if tn > 0.125:
            break
        s.block_step()
        steps += 1
        n_corr += act.size
        # every particle's time is a multiple of its step (block synchronisation)
        assert np.all(np.mod(s.t, s.dt) == 0.0)
        lv = np.log2(s.dt)
        assert np.all(lv == np.round(lv)) and lv.min() >= -20 and lv.max() <= -3
    assert np.all(s.t == 0.125) and steps > 8 and n_corr > N
    K1, W1 = s.energy()
    assert abs(K1 + W1 - K0 - W0) / abs(K0 + W0) < 1e-6


def test_f64_variant_agrees_with_long_double(oracle):
    m, x, v = W.plummer(512, 3)
    ap = np.random.default_rng(0).normal(size=x.shape)
    ref = oracle.hermite6.force(m, x, v, ap, 1e-3, kind="ld")
    f64 = oracle.hermite6.force(m, x, v, ap, 1e-3, kind="f64")
    for r, f in zip(ref[:3], f64[:3]):
        assert (np.linalg.norm(r - f, axis=1) / np.linalg.norm(r, axis=1)).max() < 1e-12
    assert np.abs(ref[3] / f64[3] - 1).max() < 1e-13


# ---------------------------------------------------------------- 4th-order variant (R21)
def test_o4_predictor_and_corrector_polynomial_exactness(oracle):
    """Predictor exact for cubic x(t); corrector exact in v and in the recovered a'', a''' for cubic a(t), exact in x for
    quadratic a(t) (two-point cubic Hermite quadrature)."""
    rng = np.random.default_rng(14)
    L = oracle.lib("ld")
    P = oracle.hermite6._p
    N = 5
    coef = rng.normal(size=(4, N, 3))                       # x, v, a, j at t_i
    ti = rng.choice([0.0, 0.25, 0.5], N)
    t = 0.75
    xp, vp = np.zeros((N, 3)), np.zeros((N, 3))
    L.oracle_predict4(N, t, P(ti), *[P(np.ascontiguousarray(c)) for c in coef], P(xp), P(vp))
    D = (t - ti)[:, None]
    np.testing.assert_allclose(xp, coef[0] + D * coef[1] + D ** 2 / 2 * coef[2] + D ** 3 / 6 * coef[3], rtol=0, atol=2e-15)
    np.testing.assert_allclose(vp, coef[1] + D * coef[2] + D ** 2 / 2 * coef[3], rtol=0, atol=2e-15)
    for deg in (2, 3):
        h, t0 = 0.25, 0.5
        pa = [np.polynomial.Polynomial(rng.normal(size=deg + 1)) for _ in range(3)]
        pv = [p.integ() + rng.normal() for p in pa]
        px = [p.integ() + rng.normal() for p in pv]
        ev = lambda polys, k, tt: np.array([[p.deriv(k)(tt) if k else p(tt) for p in polys]])
        x, v, a, j = ev(px, 0, t0), ev(pv, 0, t0), ev(pa, 0, t0), ev(pa, 1, t0)
        s, c = np.zeros((1, 3)), np.zeros((1, 3))
        t1 = t0 + h
        a1, j1 = ev(pa, 0, t1), ev(pa, 1, t1)
        tt, dt = np.array([t0]), np.array([h])
        L.oracle_correct4(1, None, 1, h, t1, P(a1), P(j1), P(x), P(v), P(a), P(j), P(s), P(c), P(tt), P(dt), 0.14, -20, -3)
        np.testing.assert_allclose(v, ev(pv, 0, t1), rtol=0, atol=1e-14)
        if deg == 2:
            np.testing.assert_allclose(x, ev(px, 0, t1), rtol=0, atol=1e-14)
        np.testing.assert_allclose(s, ev(pa, 2, t1), rtol=0, atol=1e-12)
        np.testing.assert_allclose(c, ev(pa, 3, t1), rtol=0, atol=1e-11)
        assert tt[0] == t1 and dt[0] == h and np.array_equal(a, a1) and np.array_equal(j, j1)


def test_o4_kepler_orbit_fourth_order_convergence(oracle):
    """The e = 0.5 orbit of P5 with the 4th-order scheme: halving dt divides the error by ~2^4, not 2^6."""
    e = 0.5
    m = np.array([0.5, 0.5])
    x = np.array([[0.75, 0, 0], [-0.75, 0, 0]])
    vy = 0.5 * np.sqrt((1 - e) / (1 + e))
    v = np.array([[0, vy, 0], [0, -vy, 0]])
    dx, dE = [], []
    for n in (512, 1024, 2048):
        o = oracle.OracleSystem(m, x, v, 0.0, order=4)
        E0 = sum(o.energy())
        for _ in range(n):
            o.shared_step(2 * np.pi / n)
        dx.append(np.abs(o.x - x).max()); dE.append(abs(sum(o.energy()) / E0 - 1))
    assert dx[0] < 1e-4 and dx[2] < 1e-6
    assert 12 < dx[0] / dx[1] < 20 and 12 < dx[1] / dx[2] < 20
    assert 12 < dE[0] / dE[1] < 40 and 12 < dE[1] / dE[2] < 40


def test_o4_criterion_closed_form_and_block_steps(oracle):
    L = oracle.lib("ld")
    P = oracle.hermite6._p
    # |a^(k)| = w^k |a|  =>  A1 = sqrt2 w |a|, A2 = sqrt2 w^2 |a|  =>  dt_crit = eta / w
    for w_ in (0.7, 3.0, 41.0):
        d = np.zeros((4, 3))
        for k in range(4):
            d[k, k % 3] = 2.5 * w_ ** k
        assert abs(L.oracle_aarseth4_dt(P(d), 0.14) * w_ / 0.14 - 1) < 1e-15
    # block steps on a small Plummer sphere stay on the dyadic grid and conserve energy
    m, x, v = W.plummer(96, 11)
    o = oracle.OracleSystem(m, x, v, 1e-2, order=4)
    E0 = sum(o.energy())
    n = 0
    while True:
        tn, act = o.next_block()
        if tn > 0.125:
            break
        o.predict(tn); o.force(act); o.corrector(act, 0.0)
        n += 1
        # block rule (R12): every particle's time is a multiple of its power-of-two step, levels stay in range
        assert np.all(np.mod(o.t, o.dt) == 0.0)
        lv = np.log2(o.dt)
        assert np.all(lv == np.round(lv)) and lv.min() >= -20 and lv.max() <= -3
    assert np.all(o.t == 0.125) and n > 10
    assert abs(sum(o.energy()) / E0 - 1) < 1e-5


# ---------------------------------------------------------------- 8th-order variant (R22)
@pytest.mark.parametrize("N,eps,seed", [(2, 0.0, 21), (3, 0.05, 22), (4, 0.3, 23)])
def test_o8_crackle_against_mpmath_differentiation(oracle, N, eps, seed):
    """a, jerk, snap, crackle of O1/8 = a(tau) and its first three derivatives along
    x(tau) = x + v tau + a_p tau^2/2 + j_p tau^3/6, in 50-digit arithmetic: pins alpha, beta, gamma and every coefficient."""
    mp.mp.dps = 50
    rng = np.random.default_rng(seed)
    m = rng.uniform(0.2, 1.0, N)
    x, v, ap, jp = (rng.normal(size=(N, 3)) for _ in range(4))
    idx = np.arange(N, dtype=np.int32)[::-1].copy()
    acc, jerk, snap, crk, pot = oracle.hermite6.force8(m, x, v, ap, jp, eps, idx)
    a6, j6, s6, p6 = oracle.hermite6.force(m, x, v, ap, eps, idx)
    assert np.array_equal(acc, a6) and np.array_equal(jerk, j6) and np.array_equal(pot, p6)
    np.testing.assert_allclose(snap, s6, rtol=1e-14)

    def pos(i, k, tau):
        return mp.mpf(x[i, k]) + mp.mpf(v[i, k]) * tau + mp.mpf(ap[i, k]) * tau ** 2 / 2 + mp.mpf(jp[i, k]) * tau ** 3 / 6

    def a_of_tau(i, c, tau):
        tot = mp.mpf(0)
        for jj in range(N):
            if jj == i:
                continue
            d = [pos(jj, k, tau) - pos(i, k, tau) for k in range(3)]
            s = d[0] ** 2 + d[1] ** 2 + d[2] ** 2 + mp.mpf(eps) ** 2
            tot += mp.mpf(m[jj]) * d[c] / s ** mp.mpf(1.5)
        return tot

    for k, i in enumerate(idx):
        for c in range(3):
            c_ref = mp.diff(lambda t: a_of_tau(i, c, t), 0, 3)
            s_ref = mp.diff(lambda t: a_of_tau(i, c, t), 0, 2)
            assert abs(crk[k, c] - float(c_ref)) <= 1e-15 * max(abs(float(c_ref)), np.abs(crk[k]).max())
            assert abs(snap[k, c] - float(s_ref)) <= 4e-16 * max(abs(float(s_ref)), np.abs(snap[k]).max())


def test_o8_newtons_third_law_and_startup(oracle):
    m, x, v = W.plummer(48, 8, "kroupa")
    o = oracle.OracleSystem(m, x, v, 1e-2, order=8)
    for arr in (o.a, o.j, o.s, o.c):                         # crackle obeys it only if dj uses the same jerk array for i and j
        total = (m[:, None] * arr).sum(0)
        assert np.abs(total).max() <= 1e-15 * (m[:, None] * np.abs(arr)).sum()
    o6 = oracle.OracleSystem(m, x, v, 1e-2, order=6)
    assert np.array_equal(o.a, o6.a) and np.array_equal(o.j, o6.j)
    np.testing.assert_allclose(o.s, o6.s, rtol=1e-14)          # same sum, another order of the operations


def test_o8_predictor_and_corrector_polynomial_exactness(oracle):
    rng = np.random.default_rng(18)
    L = oracle.lib("ld")
    P = oracle.hermite6._p
    N = 5
    coef = rng.normal(size=(8, N, 3))                       # x, v, a, j, s, c, a4, a5 at t_i
    ti = rng.choice([0.0, 0.25, 0.5], N)
    t = 0.75
    out = [np.zeros((N, 3)) for _ in range(4)]
    L.oracle_predict8(N, t, P(ti), *[P(np.ascontiguousarray(c)) for c in coef], *[P(o) for o in out])
    D = (t - ti)[:, None]
    fact = [1, 1, 2, 6, 24, 120, 720, 5040]
    for lo, got in enumerate(out):                           # x_p, v_p, a_p, j_p
        ref = sum(coef[k] * D ** (k - lo) / fact[k - lo] for k in range(lo, 8))
        np.testing.assert_allclose(got, ref, rtol=0, atol=4e-15)
    for deg in (6, 7):
        h, t0 = 0.25, 0.5
        pa = [np.polynomial.Polynomial(rng.normal(size=deg + 1)) for _ in range(3)]
        pv = [p.integ() + rng.normal() for p in pa]
        px = [p.integ() + rng.normal() for p in pv]
        ev = lambda polys, k, tt: np.array([[p.deriv(k)(tt) if k else p(tt) for p in polys]])
        x, v = ev(px, 0, t0), ev(pv, 0, t0)
        a, j, s, c = (ev(pa, k, t0) for k in range(4))
        a4, a5 = np.zeros((1, 3)), np.zeros((1, 3))
        t1 = t0 + h
        a1, j1, s1, c1 = (ev(pa, k, t1) for k in range(4))
        d = np.zeros(12)
        L.oracle_hermite8_derivs(h, P(a), P(j), P(s), P(c), P(a1), P(j1), P(s1), P(c1), P(d))
        for r, tol in zip(range(4), (1e-9, 1e-8, 1e-6, 1e-5)):
            np.testing.assert_allclose(d[3 * r:3 * r + 3], ev(pa, 4 + r, t1)[0], rtol=0, atol=tol)
        tt, dt = np.array([t0]), np.array([h])
        L.oracle_correct8(1, None, 1, h, t1, P(a1), P(j1), P(s1), P(c1), P(x), P(v), P(a), P(j), P(s), P(c), P(a4), P(a5),
                          P(tt), P(dt), 0.75, -20, -3)
        np.testing.assert_allclose(v, ev(pv, 0, t1), rtol=0, atol=1e-14)
        if deg == 6:
            np.testing.assert_allclose(x, ev(px, 0, t1), rtol=0, atol=1e-14)
        np.testing.assert_allclose(a4, ev(pa, 4, t1), rtol=0, atol=1e-9)
        np.testing.assert_allclose(a5, ev(pa, 5, t1), rtol=0, atol=1e-8)
        assert tt[0] == t1 and np.array_equal(c, c1)


def test_o8_kepler_orbit_eighth_order_convergence(oracle):
    e = 0.5
    m = np.array([0.5, 0.5])
    x = np.array([[0.75, 0, 0], [-0.75, 0, 0]])
    vy = 0.5 * np.sqrt((1 - e) / (1 + e))
    v = np.array([[0, vy, 0], [0, -vy, 0]])
    dx = []
    for n in (64, 128, 256):
        o = oracle.OracleSystem(m, x, v, 0.0, order=8)
        for _ in range(n):
            o.shared_step(2 * np.pi / n)
        dx.append(np.abs(o.x - x).max())
    assert dx[0] < 1e-4 and dx[2] < 1e-9
    assert dx[0] / dx[1] > 150 and dx[1] / dx[2] > 150           # ~2^8 per halving: 8th order (6th gives ~64)


def test_o8_criterion_closed_form_and_block_steps(oracle):
    L = oracle.lib("ld")
    P = oracle.hermite6._p
    for w_ in (0.7, 3.0, 41.0):                                   # |a^(k)| = w^k |a|  =>  (A1/A6)^(1/5) = 1/w
        d = np.zeros((8, 3))
        for k in range(8):
            d[k, k % 3] = 2.5 * w_ ** k
        assert abs(L.oracle_aarseth8_dt(P(d), 0.75) * w_ / 0.75 - 1) < 1e-15
    m, x, v = W.plummer(96, 11)
    o = oracle.OracleSystem(m, x, v, 1e-2, order=8)
    E0 = sum(o.energy())
    n = 0
    while True:
        tn, act = o.next_block()
        if tn > 0.125:
            break
        o.predict(tn); o.force(act); o.corrector(act, 0.0)
        n += 1
        # block rule (R12): every particle's time is a multiple of its power-of-two step, levels stay in range
        assert np.all(np.mod(o.t, o.dt) == 0.0)
        lv = np.log2(o.dt)
        assert np.all(lv == np.round(lv)) and lv.min() >= -20 and lv.max() <= -3
    assert np.all(o.t == 0.125) and n > 10
    assert abs(sum(o.energy()) / E0 - 1) < 1e-6
