"""Build libnb.so (the product) and libnbprobe.so (measurement aids) in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_1411_5234_b200.build [--force] [-v]

nb_force.cu takes one more step: between ptxas and the host compile its cubin goes through sass_sched.py, which puts the FP64
pair loops into the order they are written in (see that file).  NB_SASS_SCHED=0 in the environment builds without that step
(the GPU tests compare the two builds bit for bit).
"""
from __future__ import annotations

import glob
import os
import shlex
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libnb.so")
PROBE_LIB = os.path.join(HERE, "libnbprobe.so")          # measurement aids (csrc/nb_probe.h), loaded by bench.py only
PTXAS_LIB = os.path.join(HERE, "libnb_ptxas.so")         # the same library with nb_force.cu as ptxas scheduled it: only the test
                                                         # that compares the two builds bit for bit loads it (NB_LIB=...)
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


SCHEDULED = ["nb_force.cu"]          # sources whose cubin goes through sass_sched.py


def sass_sched_enabled() -> bool:
    return os.environ.get("NB_SASS_SCHED", "1") != "0"


def _flags():
    # NB_SASS_SCHED=all (not run on a GPU yet, see sass_sched.EXPERIMENTAL): every pair loop is rescheduled, none keeps the branches
    return NVCC_FLAGS + (["-DNB_PIN_UNSCHEDULED=false"] if os.environ.get("NB_SASS_SCHED") == "all" else [])


def _compile_scheduled(src: str, obj: str, objdir: str, verbose: bool) -> None:
    """nvcc -c with the intermediate files kept; then the cubin is rescheduled and the last two steps of nvcc's own recipe
    (fatbinary, host compile of the .cudafe1.cpp that embeds the fat binary) are run again on it."""
    from . import sass_sched
    keep = os.path.join(objdir, "keep_" + os.path.basename(src).replace(".cu", ""))
    shutil.rmtree(keep, ignore_errors=True)
    os.makedirs(keep)
    base = [_nvcc()] + _flags() + ["--keep", "--keep-dir", keep, "-c", src, "-o", obj]
    out = subprocess.run(base + (["-Xptxas", "-v"] if verbose else []), stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    if verbose or out.returncode != 0:
        sys.stderr.write(out.stdout)
    if out.returncode != 0:
        raise RuntimeError("nvcc failed: " + " ".join(base))
    shutil.copy(obj, obj.replace(".o", ".ptxas.o"))                    # the object as nvcc made it (for libnb_ptxas.so)
    stem = os.path.basename(src).replace(".cu", "")
    cubin = os.path.join(keep, stem + ".cubin")
    shutil.copy(cubin, cubin + ".ptxas")                               # what ptxas emitted, for comparison
    log = open(os.path.join(keep, "sass_sched.log"), "w")
    try:
        sass_sched.run(cubin + ".ptxas", cubin, src, report=True, log=log)
    except Exception as e:                          # the tool is an optimisation: without it the library is ptxas's code
        log.write(f"sass_sched: FAILED ({type(e).__name__}: {e}); 0 blocks rescheduled, the cubin is left as ptxas emitted it\n")
        sys.stderr.write(f"WARNING: sass_sched failed ({type(e).__name__}: {e}); {os.path.basename(src)} keeps ptxas's schedule\n")
        shutil.copy(cubin + ".ptxas", cubin)
    log.close()
    if verbose:
        sys.stderr.write(open(log.name).read())
    dry = subprocess.run(base + ["--dryrun"], stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True, check=True).stdout
    steps = [l[3:] for l in dry.split("\n") if l.startswith("#$ ")]
    redo = [l for l in steps if l.startswith("fatbinary ")] + [l for l in steps if l.startswith("gcc ") and " -c " in l and ".cudafe1.cpp" in l]
    if len(redo) != 2:
        raise RuntimeError("unexpected nvcc recipe: " + dry)
    env = dict(os.environ, PATH=os.path.dirname(_nvcc()) + os.pathsep + os.environ.get("PATH", ""))
    for l in redo:
        subprocess.run(shlex.split(l), check=True, env=env)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not stale():
        return LIB
    objdir = os.path.join(HERE, "build")
    os.makedirs(objdir, exist_ok=True)
    procs, objs = [], {}
    for s in SOURCES + PROBE_SOURCES:
        o = os.path.join(objdir, s.replace(".cu", ".o"))
        objs[s] = o
        if s in SCHEDULED and sass_sched_enabled():
            continue
        cmd = [_nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", os.path.join(CSRC, s), "-o", o]
        procs.append((cmd, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    for s in SCHEDULED:
        if sass_sched_enabled():
            _compile_scheduled(os.path.join(CSRC, s), objs[s], objdir, verbose)
    for cmd, p in procs:
        out, _ = p.communicate()
        if verbose or p.returncode != 0:
            sys.stderr.write(out)
        if p.returncode != 0:
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
    arch = ["-gencode", "arch=compute_100a,code=sm_100a"]
    subprocess.run([_nvcc(), "-shared", "-o", LIB] + [objs[s] for s in SOURCES] + arch, check=True)
    if sass_sched_enabled():
        subprocess.run([_nvcc(), "-shared", "-o", PTXAS_LIB] + [objs[s].replace(".o", ".ptxas.o") if s in SCHEDULED else objs[s]
                                                                for s in SOURCES] + arch, check=True)
    elif os.path.exists(PTXAS_LIB):
        os.remove(PTXAS_LIB)
    subprocess.run([_nvcc(), "-shared", "-o", PROBE_LIB] + [objs[s] for s in PROBE_SOURCES] + arch, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
