"""Thin ctypes binding of include/nb.h — same names, argument marshalling only.

Every step of the path runs in the CUDA kernels of libnb.so.  PyTorch is used for what the
task statement allows: device memory (the workspace and device-side buffers), streams and,
in bench.py, torch.distributed.  There is NO CPU fallback: if libnb.so is missing or cannot be
loaded, importing `lib()` raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("NB_LIB") or os.path.join(_HERE, "libnb.so")   # NB_LIB: another build of the same library (build comparisons)

NB_OK, NB_EINVAL, NB_ENOMEM, NB_ESTATE, NB_ECUDA = 0, -1, -2, -3, -4
NB_PREC_FP64, NB_PREC_MIXED = 0, 1
FIELDS = dict(M=0, X=1, V=2, A=3, J=4, S=5, C=6, T=7, DT=8, XP=9, VP=10, AP=11, A4=12, A5=13, JP=14)
_WIDTH = {0: 1, 7: 1, 8: 1}
ACTIVE_INTERNAL = C.c_void_p(1)

EXPORTS = ["nb_workspace_bytes", "nb_plan_force", "nb_set_max_split", "nb_init", "nb_predict", "nb_force", "nb_force_crackle", "nb_corrector",
           "nb_next_block", "nb_run_blocks", "nb_get_state", "nb_set_state", "nb_energy", "nb_check_indices", "nb_resident_ctas", "nb_step_log",
           "nb_launch_count", "nb_last_force_ms", "nb_strerror", "nb_last_error", "nb_free"]


class nb_config(C.Structure):
    _fields_ = [("device", C.c_int), ("stream", C.c_void_p), ("workspace", C.c_void_p),
                ("workspace_bytes", C.c_size_t), ("ptrs_on_device", C.c_int),
                ("eta", C.c_double), ("eta_s", C.c_double), ("k_min", C.c_int), ("k_max", C.c_int), ("order", C.c_int),
                ("check_indices", C.c_int), ("precision", C.c_int)]


class nb_plan(C.Structure):
    _fields_ = [("kernel", C.c_int), ("n_units", C.c_int), ("n_split", C.c_int), ("slice_tiles", C.c_int),
                ("grid", C.c_int), ("unit", C.c_int), ("tile", C.c_int), ("ctas_per_sm", C.c_int), ("predict_in_force", C.c_int),
                ("waves", C.c_double)]


class NBError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"nb status {status}: {msg}")
        self.status = status


_lib = None


def lib() -> C.CDLL:
    """Load libnb.so (build it with `python -m paper_1411_5234_b200.build`).  Fails loudly if absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_1411_5234_b200.build` "
                          "(there is no CPU fallback for the CUDA path)")
    L = C.CDLL(LIB_PATH)
    vp, i64, dbl = C.c_void_p, C.c_int64, C.c_double
    L.nb_workspace_bytes.argtypes = [i64]; L.nb_workspace_bytes.restype = C.c_size_t
    L.nb_plan_force.argtypes = [i64, i64, C.c_int, C.POINTER(nb_plan)]; L.nb_plan_force.restype = C.c_int
    L.nb_set_max_split.argtypes = [vp, i64]; L.nb_set_max_split.restype = C.c_int
    L.nb_init.argtypes = [C.POINTER(vp), i64, vp, vp, vp, dbl, C.POINTER(nb_config)]; L.nb_init.restype = C.c_int
    L.nb_predict.argtypes = [vp, dbl]; L.nb_predict.restype = C.c_int
    L.nb_force.argtypes = [vp, vp, i64, vp, vp, vp, vp]; L.nb_force.restype = C.c_int
    L.nb_force_crackle.argtypes = [vp, vp]; L.nb_force_crackle.restype = C.c_int
    L.nb_corrector.argtypes = [vp, vp, i64, dbl]; L.nb_corrector.restype = C.c_int
    L.nb_next_block.argtypes = [vp, C.POINTER(dbl), vp, C.POINTER(i64)]; L.nb_next_block.restype = C.c_int
    L.nb_run_blocks.argtypes = [vp, dbl, i64, C.POINTER(i64), C.POINTER(dbl), C.POINTER(i64)]; L.nb_run_blocks.restype = C.c_int
    L.nb_get_state.argtypes = [vp, C.c_int, vp, i64, vp]; L.nb_get_state.restype = C.c_int
    L.nb_set_state.argtypes = [vp, C.c_int, vp, i64, vp]; L.nb_set_state.restype = C.c_int
    L.nb_energy.argtypes = [vp, C.POINTER(dbl), C.POINTER(dbl)]; L.nb_energy.restype = C.c_int
    L.nb_check_indices.argtypes = [vp, vp, i64, C.c_int]; L.nb_check_indices.restype = C.c_int
    L.nb_resident_ctas.argtypes = [vp, C.c_int]; L.nb_resident_ctas.restype = C.c_int
    L.nb_step_log.argtypes = [vp, i64, vp, vp]; L.nb_step_log.restype = i64
    L.nb_launch_count.argtypes = [vp]; L.nb_launch_count.restype = i64
    L.nb_last_force_ms.argtypes = [vp]; L.nb_last_force_ms.restype = dbl
    L.nb_strerror.argtypes = [C.c_int]; L.nb_strerror.restype = C.c_char_p
    L.nb_last_error.argtypes = [vp]; L.nb_last_error.restype = C.c_char_p
    L.nb_free.argtypes = [vp]; L.nb_free.restype = None
    _lib = L
    return L


def nb_workspace_bytes(N: int) -> int:
    return lib().nb_workspace_bytes(N)


def nb_plan_force(N: int, n_act: int, n_sm: int = 148) -> nb_plan:
    p = nb_plan()
    rc = lib().nb_plan_force(N, n_act, n_sm, C.byref(p))
    if rc != NB_OK:
        raise NBError(rc, lib().nb_strerror(rc).decode())
    return p


def _ptr(a):
    """Raw address of a numpy array (host) or a torch tensor (device or pinned host); None -> NULL."""
    if a is None:
        return None
    if isinstance(a, C.c_void_p):
        return a
    if isinstance(a, np.ndarray):
        assert a.flags["C_CONTIGUOUS"]
        return C.c_void_p(a.ctypes.data)
    assert a.is_contiguous()
    return C.c_void_p(a.data_ptr())


class System:
    """One particle system on one GPU: owns the torch workspace and the nb_ctx.  Methods are the ABI calls.

    host=True : array arguments are numpy arrays (HOST pointers; the library copies and synchronises).
    host=False: array arguments are torch CUDA tensors (DEVICE pointers; calls are asynchronous).
    """

    def __init__(self, m, x, v, eps, host=True, device=0, eta=0.0, eta_s=0.0, k_min=0, k_max=0, stream=None, order=0,
                 check_indices=0, precision=0, guard_bytes=0):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1411_5234_b200 needs a CUDA device; there is no CPU fallback")
        self._torch = torch
        self.L = lib()
        self.host = host
        self.device = device
        self.N = int(m.shape[0])
        self.ctx = C.c_void_p()
        torch.cuda.set_device(device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(device)
        nbytes = self.L.nb_workspace_bytes(self.N)
        # guard_bytes > 0: bands of 0xA5 before and after the workspace that nothing may touch (guards_intact(); compute-sanitizer
        # is not available on every pool, this is the memory-safety check that always is)
        self._guard = (int(guard_bytes) + 255) // 256 * 256
        self.workspace = torch.empty(nbytes + 256 + 2 * self._guard, dtype=torch.uint8, device=f"cuda:{device}")
        if self._guard:
            self.workspace.fill_(0xA5)
        base = (self.workspace.data_ptr() + self._guard + 255) // 256 * 256
        self._ws_off, self._ws_bytes = base - self.workspace.data_ptr(), nbytes
        self.cfg = nb_config(device, C.c_void_p(self.stream.cuda_stream), C.c_void_p(base), nbytes,
                             0 if host else 1, eta, eta_s, k_min, k_max, order, check_indices, precision)
        m, x, v = self._in(m, (self.N,)), self._in(x, (self.N, 3)), self._in(v, (self.N, 3))
        self._check(self.L.nb_init(C.byref(self.ctx), self.N, _ptr(m), _ptr(x), _ptr(v), float(eps), C.byref(self.cfg)))

    # -- marshalling helpers
    def _in(self, a, shape=None, dtype=np.float64):
        if self.host:
            a = np.ascontiguousarray(a, dtype=dtype)
        else:
            tdt = self._torch.float64 if dtype == np.float64 else self._torch.int32
            assert a.is_cuda and a.dtype == tdt
            a = a.contiguous()
        if shape is not None:
            assert tuple(a.shape) == tuple(shape), (tuple(a.shape), shape)
        return a

    def _out(self, *shape):
        if self.host:
            return np.empty(shape, dtype=np.float64)
        return self._torch.empty(shape, dtype=self._torch.float64, device=f"cuda:{self.device}")

    def _check(self, rc):
        if rc != NB_OK:
            detail = self.L.nb_last_error(self.ctx).decode() if self.ctx else ""
            raise NBError(rc, self.L.nb_strerror(rc).decode() + (f" [{detail}]" if detail else ""))

    # -- the ABI
    def nb_predict(self, t):
        self._check(self.L.nb_predict(self.ctx, float(t)))

    def nb_force(self, active_idx=None, n_act=None, outputs=True):
        """Returns (a, jerk, snap, pot) for the active rows; outputs=False keeps the results inside the context."""
        if active_idx is None:
            n = self.N if n_act is None else n_act
            ip = None
        elif isinstance(active_idx, C.c_void_p):
            n, ip = n_act, active_idx
        else:
            active_idx = self._in(active_idx, dtype=np.int32)
            n = int(active_idx.shape[0])
            ip = _ptr(active_idx)
        if outputs:
            a, j, s, p = self._out(n, 3), self._out(n, 3), self._out(n, 3), self._out(n)
        else:
            a = j = s = p = None
        self._check(self.L.nb_force(self.ctx, ip, n, _ptr(a), _ptr(j), _ptr(s), _ptr(p)))
        return a, j, s, p

    def nb_force_crackle(self, n):
        """Crackle [n, 3] of the last nb_force over n active particles (8th order)."""
        out = self._out(n, 3)
        self._check(self.L.nb_force_crackle(self.ctx, _ptr(out)))
        return out

    def nb_corrector(self, active_idx=None, dt=0.0, n_act=None):
        if active_idx is None:
            n, ip = (self.N if n_act is None else n_act), None
        elif isinstance(active_idx, C.c_void_p):
            n, ip = n_act, active_idx
        else:
            active_idx = self._in(active_idx, dtype=np.int32)
            n, ip = int(active_idx.shape[0]), _ptr(active_idx)
        self._check(self.L.nb_corrector(self.ctx, ip, n, float(dt)))

    def nb_set_max_split(self, max_split):
        self._check(self.L.nb_set_max_split(self.ctx, int(max_split)))

    def nb_next_block(self, want_list=True):
        t, n = C.c_double(), C.c_int64()
        if not want_list:
            self._check(self.L.nb_next_block(self.ctx, C.byref(t), None, C.byref(n)))
            return t.value, n.value, None
        if self.host:
            buf = np.empty(self.N, dtype=np.int32)
        else:
            buf = self._torch.empty(self.N, dtype=self._torch.int32, device=f"cuda:{self.device}")
        self._check(self.L.nb_next_block(self.ctx, C.byref(t), _ptr(buf), C.byref(n)))
        return t.value, n.value, buf[:n.value]

    def nb_run_blocks(self, t_end, max_steps=1 << 62):
        """Returns (steps_done, t_last, sum_n_act)."""
        steps, t_last, sum_act = C.c_int64(), C.c_double(), C.c_int64()
        self._check(self.L.nb_run_blocks(self.ctx, float(t_end), int(max_steps), C.byref(steps), C.byref(t_last), C.byref(sum_act)))
        return steps.value, t_last.value, sum_act.value

    def nb_get_state(self, field, idx=None, n=None):
        f = FIELDS[field] if isinstance(field, str) else field
        if idx is not None:
            idx = self._in(idx, dtype=np.int32)
            n = int(idx.shape[0])
        n = self.N if n is None else n
        out = self._out(n) if _WIDTH.get(f, 3) == 1 else self._out(n, 3)
        self._check(self.L.nb_get_state(self.ctx, f, _ptr(idx), n, _ptr(out)))
        return out

    def nb_set_state(self, field, values, idx=None):
        f = FIELDS[field] if isinstance(field, str) else field
        values = self._in(values)
        if idx is not None:
            idx = self._in(idx, dtype=np.int32)
        n = int(values.shape[0])
        self._check(self.L.nb_set_state(self.ctx, f, _ptr(idx), n, _ptr(values)))

    def nb_energy(self):
        k, w = C.c_double(), C.c_double()
        self._check(self.L.nb_energy(self.ctx, C.byref(k), C.byref(w)))
        return k.value, w.value

    def nb_check_indices(self, idx, unique=True):
        """NB_OK (0) or NB_EINVAL (-1): the status itself, not an exception."""
        idx = self._in(idx, dtype=np.int32)
        return self.L.nb_check_indices(self.ctx, _ptr(idx), int(idx.shape[0]), 1 if unique else 0)

    def nb_step_log(self, capacity=8192):
        """(n_act[int64], t_us[float64]) of the most recent block steps of nb_run_blocks, oldest first."""
        na, tu = np.empty(capacity, dtype=np.int64), np.empty(capacity, dtype=np.float64)
        n = self.L.nb_step_log(self.ctx, capacity, C.c_void_p(na.ctypes.data), C.c_void_p(tu.ctypes.data))
        if n < 0:
            self._check(int(n))
        return na[:n], tu[:n]

    def nb_resident_ctas(self, kernel):
        return self.L.nb_resident_ctas(self.ctx, int(kernel))

    def guards_intact(self):
        """True if no byte outside [workspace, workspace + nb_workspace_bytes) of the allocation was written."""
        self._torch.cuda.synchronize()
        lo, hi = self.workspace[:self._ws_off], self.workspace[self._ws_off + self._ws_bytes:]
        return bool((lo == 0xA5).all().item()) and bool((hi == 0xA5).all().item())

    def nb_launch_count(self):
        return self.L.nb_launch_count(self.ctx)

    def nb_last_force_ms(self):
        return self.L.nb_last_force_ms(self.ctx)

    def nb_free(self):
        if self.ctx:
            self.L.nb_free(self.ctx)
            self.ctx = C.c_void_p()

    def __del__(self):
        try:
            self.nb_free()
        except Exception:
            pass
