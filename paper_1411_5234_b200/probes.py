"""ctypes loader of libnbprobe.so (csrc/nb_probe.h): measurement aids for bench.py and the profiling scripts.

Not part of the method and not part of libnb.so: register-resident instruction streams that measure the FP64 FMA peak,
the cycles a DFMA holds the pipe by operand source, and the rates behind the mixed-precision decision.
"""
from __future__ import annotations

import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libnbprobe.so")
EXPORTS = ["nbp_fp64_peak", "nbp_dfma_sources", "nbp_mixed_rates"]
MIXED_KINDS = ("ffma_three_sources", "f2f_round_trip_d2f_f2d", "f2f_round_trip_plus_dadd", "f2d_dadd_fadd",
               "float_float_accumulate", "dfma_plus_ffma_pair", "ffma_one_source_reused", "ffma_immediates",
               "ffma2_three_sources", "ffma2_one_source_reused")
_lib = None


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_1411_5234_b200.build`")
        L = C.CDLL(LIB_PATH)
        vp, dbl = C.c_void_p, C.c_double
        L.nbp_fp64_peak.argtypes = [C.c_int, vp, vp, C.c_size_t, dbl, C.POINTER(dbl), C.POINTER(C.c_int)]
        L.nbp_dfma_sources.argtypes = [C.c_int, vp, vp, C.c_size_t, C.c_int, dbl, C.POINTER(dbl)]
        L.nbp_mixed_rates.argtypes = [C.c_int, vp, vp, C.c_size_t, C.c_int, dbl, C.POINTER(dbl)]
        for f in EXPORTS:
            getattr(L, f).restype = C.c_int
        _lib = L
    return _lib


def _ws(device):
    import torch
    ws = torch.empty(65536 + 256, dtype=torch.uint8, device=f"cuda:{device}")
    return ws, C.c_void_p((ws.data_ptr() + 255) // 256 * 256), C.c_void_p(torch.cuda.current_stream(device).cuda_stream)


def fp64_peak(seconds=1.0, device=0):
    """Sustained FP64 FMA rate of the device in TFLOP/s (FMA = 2 flop) and its SM count."""
    ws, base, st = _ws(device)
    tf, nsm = C.c_double(), C.c_int()
    rc = lib().nbp_fp64_peak(device, st, base, 65536, float(seconds), C.byref(tf), C.byref(nsm))
    if rc != 0:
        raise RuntimeError(f"nbp_fp64_peak: {rc}")
    return tf.value, nsm.value


def dfma_sources(sm_mhz, device=0):
    """Cycles per warp-wide DFMA and SM sub-partition for 2-source, 3-source and 3-source-with-reuse streams."""
    ws, base, st = _ws(device)
    out = {}
    for kind, name in enumerate(("two_sources", "three_sources", "three_sources_one_reused")):
        cyc = C.c_double()
        rc = lib().nbp_dfma_sources(device, st, base, 65536, kind, float(sm_mhz), C.byref(cyc))
        if rc != 0:
            raise RuntimeError(f"nbp_dfma_sources: {rc}")
        out[name] = cyc.value
    return out


def mixed_rates(sm_mhz, device=0):
    """Cycles per warp instruction (or per accumulated element) of the streams a mixed-precision pair would use."""
    ws, base, st = _ws(device)
    out = {}
    for kind, name in enumerate(MIXED_KINDS):
        cyc = C.c_double()
        rc = lib().nbp_mixed_rates(device, st, base, 65536, kind, float(sm_mhz), C.byref(cyc))
        if rc != 0:
            raise RuntimeError(f"nbp_mixed_rates: {rc}")
        out[name] = cyc.value
    return out


if __name__ == "__main__":
    import json
    import sys
    mhz = float(sys.argv[1]) if len(sys.argv) > 1 else 1965.0
    print(json.dumps({"sm_mhz": mhz, "fp64_peak_tflops": fp64_peak(1.0)[0], "dfma_sources": dfma_sources(mhz),
                      "mixed_rates": mixed_rates(mhz)}, indent=1))
