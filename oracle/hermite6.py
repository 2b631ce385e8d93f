"""ctypes front end of oracle/nb_oracle.c and the Hermite-6 step sequencing around it.

TEST INFRASTRUCTURE (see nb_oracle.c's header).  `OracleSystem` strings the C functions O1..O7
together in the order of one block step (predict all, evaluate the active
particles once, correct them) and performs the two-pass startup (reading R8).  It holds
no arithmetic of its own beyond choosing which C function to call on which arrays.

Two builds of the same source: `liboracle_ld.so` (REAL = long double, the parity reference) and
`liboracle_f64.so` (REAL = double, the CPU baseline that bench.py times).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "nb_oracle.c")
_LIBS = {"ld": os.path.join(_HERE, "liboracle_ld.so"), "f64": os.path.join(_HERE, "liboracle_f64.so")}
_loaded: dict = {}

_d = C.POINTER(C.c_double)
_i32 = C.POINTER(C.c_int32)


def build(force: bool = False) -> None:
    """Compile both variants with gcc (-O2, OpenMP over i, no fast-math, no FMA contraction)."""
    for kind, path in _LIBS.items():
        if not force and os.path.exists(path) and os.path.getmtime(path) >= os.path.getmtime(_SRC):
            continue
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-ffp-contract=off", "-shared", "-fPIC", _SRC, "-o", path, "-lm"]
        if kind == "f64":
            cmd.insert(1, "-DREAL=double")
        subprocess.run(cmd, check=True)


def lib(kind: str = "ld") -> C.CDLL:
    if kind in _loaded:
        return _loaded[kind]
    build()
    L = C.CDLL(_LIBS[kind])
    L.oracle_real_bytes.restype = C.c_int
    L.oracle_force.argtypes = [C.c_int64, _d, _d, _d, _d, C.c_double, _i32, C.c_int64, _d, _d, _d, _d]
    L.oracle_force.restype = None
    L.oracle_predict.argtypes = [C.c_int64, C.c_double, _d] + [_d] * 6 + [_d] * 3
    L.oracle_predict.restype = None
    L.oracle_startup_levels.argtypes = [C.c_int64, _d, _d, C.c_double, C.c_int, C.c_int, _d]
    L.oracle_startup_levels.restype = None
    L.oracle_correct.argtypes = [C.c_int64, _i32, C.c_int64, C.c_double, C.c_double, _d, _d, _d,
                                 _d, _d, _d, _d, _d, _d, _d, _d, C.c_double, C.c_int, C.c_int]
    L.oracle_correct.restype = None
    L.oracle_aarseth6_level.argtypes = [_d, C.c_double, C.c_int, C.c_int]
    L.oracle_aarseth6_level.restype = C.c_int
    L.oracle_aarseth6_dt.argtypes = [_d, C.c_double]
    L.oracle_aarseth6_dt.restype = C.c_double
    L.oracle_hermite_derivs.argtypes = [C.c_double] + [_d] * 7
    L.oracle_hermite_derivs.restype = None
    L.oracle_predict4.argtypes = [C.c_int64, C.c_double, _d] + [_d] * 4 + [_d] * 2
    L.oracle_predict4.restype = None
    L.oracle_correct4.argtypes = [C.c_int64, _i32, C.c_int64, C.c_double, C.c_double, _d, _d,
                                  _d, _d, _d, _d, _d, _d, _d, _d, C.c_double, C.c_int, C.c_int]
    L.oracle_correct4.restype = None
    L.oracle_aarseth4_dt.argtypes = [_d, C.c_double]
    L.oracle_aarseth4_dt.restype = C.c_double
    L.oracle_force8.argtypes = [C.c_int64, _d, _d, _d, _d, _d, C.c_double, _i32, C.c_int64, _d, _d, _d, _d, _d]
    L.oracle_force8.restype = None
    L.oracle_predict8.argtypes = [C.c_int64, C.c_double, _d] + [_d] * 8 + [_d] * 4
    L.oracle_predict8.restype = None
    L.oracle_correct8.argtypes = [C.c_int64, _i32, C.c_int64, C.c_double, C.c_double, _d, _d, _d, _d,
                                  _d, _d, _d, _d, _d, _d, _d, _d, _d, _d, C.c_double, C.c_int, C.c_int]
    L.oracle_correct8.restype = None
    L.oracle_hermite8_derivs.argtypes = [C.c_double] + [_d] * 9
    L.oracle_hermite8_derivs.restype = None
    L.oracle_aarseth8_dt.argtypes = [_d, C.c_double]
    L.oracle_aarseth8_dt.restype = C.c_double
    L.oracle_next_block.argtypes = [C.c_int64, _d, _d, _d, _i32]
    L.oracle_next_block.restype = C.c_int64
    L.oracle_energy.argtypes = [C.c_int64, _d, _d, _d, _d, _d]
    L.oracle_energy.restype = None
    _loaded[kind] = L
    return L


def _p(a):
    return None if a is None else a.ctypes.data_as(_d)


def _pi(a):
    return None if a is None else a.ctypes.data_as(_i32)


def _f64(a, shape=None):
    a = np.ascontiguousarray(a, dtype=np.float64)
    if shape is not None:
        assert a.shape == shape, (a.shape, shape)
    return a


def force(m, xp, vp, ap, eps, idx=None, kind="ld", want=("a", "j", "s", "p")):
    """O1 on explicit arrays: returns (acc[n,3], jerk[n,3], snap[n,3], pot[n]) for the active rows."""
    N = m.shape[0]
    m, xp, vp, ap = _f64(m, (N,)), _f64(xp, (N, 3)), _f64(vp, (N, 3)), _f64(ap, (N, 3))
    if idx is not None:
        idx = np.ascontiguousarray(idx, dtype=np.int32)
    n = N if idx is None else idx.shape[0]
    acc, jerk, snap, pot = np.zeros((n, 3)), np.zeros((n, 3)), np.zeros((n, 3)), np.zeros(n)
    lib(kind).oracle_force(N, _p(m), _p(xp), _p(vp), _p(ap), float(eps), _pi(idx), n,
                           _p(acc) if "a" in want else None, _p(jerk) if "j" in want else None,
                           _p(snap) if "s" in want else None, _p(pot) if "p" in want else None)
    return acc, jerk, snap, pot


def force8(m, xp, vp, ap, jp, eps, idx=None, kind="ld"):
    """O1/8 on explicit arrays: (acc, jerk, snap, crackle [n,3], pot[n]) for the active rows."""
    N = m.shape[0]
    m, xp, vp, ap, jp = _f64(m, (N,)), _f64(xp, (N, 3)), _f64(vp, (N, 3)), _f64(ap, (N, 3)), _f64(jp, (N, 3))
    if idx is not None:
        idx = np.ascontiguousarray(idx, dtype=np.int32)
    n = N if idx is None else idx.shape[0]
    out = [np.zeros((n, 3)) for _ in range(4)] + [np.zeros(n)]
    lib(kind).oracle_force8(N, _p(m), _p(xp), _p(vp), _p(ap), _p(jp), float(eps), _pi(idx), n, *[_p(o) for o in out])
    return tuple(out)


class OracleSystem:
    """Mirror of the C ABI (include/nb.h) on the CPU: init / predict / force / corrector / next_block."""

    def __init__(self, m, x, v, eps, eta=None, eta_s=0.01, k_min=-20, k_max=-3, kind="ld", order=6):
        assert order in (4, 6, 8)
        eta = {4: 0.14, 6: 0.45, 8: 0.75}[order] if eta is None else eta
        self.L = lib(kind)
        self.kind = kind
        self.order = order
        self.N = N = int(m.shape[0])
        self.eps, self.eta, self.eta_s, self.k_min, self.k_max = float(eps), eta, eta_s, k_min, k_max
        self.m = _f64(m, (N,)).copy()
        self.x, self.v = _f64(x, (N, 3)).copy(), _f64(v, (N, 3)).copy()
        self.a, self.j, self.s, self.c = (np.zeros((N, 3)) for _ in range(4))
        self.t = np.zeros(N)
        self.dt = np.zeros(N)
        self.xp, self.vp, self.ap = np.zeros((N, 3)), np.zeros((N, 3)), np.zeros((N, 3))
        self.a4, self.a5, self.jp = np.zeros((N, 3)), np.zeros((N, 3)), np.zeros((N, 3))      # 8th order only
        self.t_pred = 0.0
        self.f = None
        # Startup (R8): pass 1 with a := 0 gives a, jerk; pass 2 with that a gives snap; a''' := 0.
        zero = np.zeros((N, 3))
        a1, j1, _, p1 = force(self.m, self.x, self.v, zero, self.eps, kind=kind)
        if order == 4:                                      # a and jerk need no second pass; snap, crackle := 0
            self.a[:], self.j[:] = a1, j1
            self.pot0 = p1
        elif order == 8:                                    # R22: a third pass with a and jerk gives crackle; a4 = a5 := 0
            a2, j2, _, _, _ = force8(self.m, self.x, self.v, a1, zero, self.eps, kind=kind)
            a3, j3, s3, c3, p3 = force8(self.m, self.x, self.v, a2, j2, self.eps, kind=kind)
            self.a[:], self.j[:], self.s[:], self.c[:] = a3, j3, s3, c3
            self.pot0 = p3
        else:
            a2, j2, s2, p2 = force(self.m, self.x, self.v, a1, self.eps, kind=kind)
            self.a[:], self.j[:], self.s[:] = a2, j2, s2
            self.pot0 = p2
        self.L.oracle_startup_levels(N, _p(self.a), _p(self.j), eta_s, k_min, k_max, _p(self.dt))

    @classmethod
    def from_state(cls, m, x, v, a, j, s, c, t, dt, eps, eta=0.45, eta_s=0.01, k_min=-20, k_max=-3, kind="ld", order=6):
        """A system that continues from a given state (no startup evaluation): for checks at sizes where the two
        O(N^2) startup passes are out of reach."""
        o = cls.__new__(cls)
        o.L, o.kind, o.order = lib(kind), kind, order
        o.N = N = int(m.shape[0])
        o.eps, o.eta, o.eta_s, o.k_min, o.k_max = float(eps), eta, eta_s, k_min, k_max
        o.m = _f64(m, (N,)).copy()
        o.x, o.v, o.a, o.j, o.s, o.c = (_f64(q, (N, 3)).copy() for q in (x, v, a, j, s, c))
        o.t, o.dt = _f64(t, (N,)).copy(), _f64(dt, (N,)).copy()
        o.xp, o.vp, o.ap = np.zeros((N, 3)), np.zeros((N, 3)), np.zeros((N, 3))
        o.a4, o.a5, o.jp = np.zeros((N, 3)), np.zeros((N, 3)), np.zeros((N, 3))
        o.t_pred, o.f = 0.0, None
        return o

    def predict(self, t):
        if self.order == 8:
            self.L.oracle_predict8(self.N, float(t), _p(self.t), _p(self.x), _p(self.v), _p(self.a), _p(self.j), _p(self.s),
                                   _p(self.c), _p(self.a4), _p(self.a5), _p(self.xp), _p(self.vp), _p(self.ap), _p(self.jp))
            self.t_pred = float(t)
            return
        if self.order == 4:
            self.L.oracle_predict4(self.N, float(t), _p(self.t), _p(self.x), _p(self.v), _p(self.a), _p(self.j),
                                   _p(self.xp), _p(self.vp))
            self.ap[:] = 0.0                                # not used by a and jerk
            self.t_pred = float(t)
            return
        self.L.oracle_predict(self.N, float(t), _p(self.t), _p(self.x), _p(self.v), _p(self.a),
                              _p(self.j), _p(self.s), _p(self.c), _p(self.xp), _p(self.vp), _p(self.ap))
        self.t_pred = float(t)

    def force(self, idx=None):
        if self.order == 8:                                 # (a, jerk, snap, pot, crackle): crackle last, so f[:4] reads as at order 6
            a, j, s, c, p = force8(self.m, self.xp, self.vp, self.ap, self.jp, self.eps, idx, kind=self.kind)
            self.f = (a, j, s, p, c)
            return self.f
        want = ("a", "j", "p") if self.order == 4 else ("a", "j", "s", "p")
        self.f = force(self.m, self.xp, self.vp, self.ap, self.eps, idx, kind=self.kind, want=want)
        return self.f

    def corrector(self, idx=None, dt=0.0):
        if idx is not None:
            idx = np.ascontiguousarray(idx, dtype=np.int32)
        n = self.N if idx is None else idx.shape[0]
        a1, j1, s1 = self.f[:3]
        assert a1.shape[0] == n
        if self.order == 8:
            self.L.oracle_correct8(self.N, _pi(idx), n, float(dt), self.t_pred, _p(a1), _p(j1), _p(s1), _p(self.f[4]),
                                   _p(self.x), _p(self.v), _p(self.a), _p(self.j), _p(self.s), _p(self.c), _p(self.a4), _p(self.a5),
                                   _p(self.t), _p(self.dt), self.eta, self.k_min, self.k_max)
            return
        if self.order == 4:
            self.L.oracle_correct4(self.N, _pi(idx), n, float(dt), self.t_pred, _p(a1), _p(j1),
                                   _p(self.x), _p(self.v), _p(self.a), _p(self.j), _p(self.s), _p(self.c),
                                   _p(self.t), _p(self.dt), self.eta, self.k_min, self.k_max)
            return
        self.L.oracle_correct(self.N, _pi(idx), n, float(dt), self.t_pred, _p(a1), _p(j1), _p(s1),
                              _p(self.x), _p(self.v), _p(self.a), _p(self.j), _p(self.s), _p(self.c),
                              _p(self.t), _p(self.dt), self.eta, self.k_min, self.k_max)

    def next_block(self):
        act = np.zeros(self.N, dtype=np.int32)
        tn = C.c_double(0.0)
        n = self.L.oracle_next_block(self.N, _p(self.t), _p(self.dt), C.byref(tn), _pi(act))
        return tn.value, act[:n].copy()

    def energy(self):
        """Energy of the stored state (all particles must be synchronised at one time)."""
        assert np.all(self.t == self.t[0])
        _, _, _, pot = force(self.m, self.x, self.v, self.a, self.eps, kind=self.kind, want=("p",))
        K, W = C.c_double(0.0), C.c_double(0.0)
        self.L.oracle_energy(self.N, _p(self.m), _p(self.v), _p(pot), C.byref(K), C.byref(W))
        return K.value, W.value

    def shared_step(self, dt):
        """One Hermite-6 step with a shared time step: predict(t+dt) -> force(all) -> corrector(all, dt)."""
        t = self.t[0] + dt
        self.predict(t)
        self.force(None)
        self.corrector(None, dt)

    def block_step(self):
        tn, act = self.next_block()
        self.predict(tn)
        self.force(act)
        self.corrector(act, 0.0)
        return tn, act
