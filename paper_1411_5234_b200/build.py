"""Build libnb.so (the product) and libnbprobe.so (measurement aids) in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_1411_5234_b200.build [--force]
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libnb.so")
PROBE_LIB = os.path.join(HERE, "libnbprobe.so")          # measurement aids (csrc/nb_probe.h), loaded by bench.py only
SOURCES = ["nb_api.cu", "nb_force.cu", "nb_step.cu"]
PROBE_SOURCES = ["nb_probe.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-I" + os.path.join(ROOT, "include")]


def _nvcc() -> str:
    for p in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if p and (os.path.isabs(p) and os.path.exists(p) or not os.path.isabs(p)):
            return p
    return "nvcc"


def _headers():
    return glob.glob(os.path.join(CSRC, "*.h")) + glob.glob(os.path.join(ROOT, "include", "*.h"))


def stale() -> bool:
    """True if a library is missing or older than any source or header (every csrc/*.h and include/*.h counts)."""
    for lib, sources in ((LIB, SOURCES), (PROBE_LIB, PROBE_SOURCES)):
        if not os.path.exists(lib):
            return True
        t = os.path.getmtime(lib)
        if any(os.path.getmtime(d) > t for d in [os.path.join(CSRC, s) for s in sources] + _headers()):
            return True
    return False


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not stale():
        return LIB
    objdir = os.path.join(HERE, "build")
    os.makedirs(objdir, exist_ok=True)
    procs, objs = [], {}
    for s in SOURCES + PROBE_SOURCES:
        o = os.path.join(objdir, s.replace(".cu", ".o"))
        cmd = [_nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", os.path.join(CSRC, s), "-o", o]
        procs.append((cmd, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
        objs[s] = o
    for cmd, p in procs:
        out, _ = p.communicate()
        if verbose or p.returncode != 0:
            sys.stderr.write(out)
        if p.returncode != 0:
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
    arch = ["-gencode", "arch=compute_100a,code=sm_100a"]
    subprocess.run([_nvcc(), "-shared", "-o", LIB] + [objs[s] for s in SOURCES] + arch, check=True)
    subprocess.run([_nvcc(), "-shared", "-o", PROBE_LIB] + [objs[s] for s in PROBE_SOURCES] + arch, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
