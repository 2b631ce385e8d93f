"""CPU-only checks of the boundary: libnb.so builds for sm_100a, loads, exports every symbol that
include/nb.h declares, and its pure host logic (workspace sizing, launch planning, argument
validation) behaves.  No kernel is launched here."""
import ctypes as C
import os
import re
import subprocess

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def B():
    from paper_1411_5234_b200 import build, binding
    build.build()
    binding.lib()
    return binding


def test_library_exports_every_declared_symbol(B):
    hdr = open(os.path.join(ROOT, "include", "nb.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = sorted(set(re.findall(r"\b(nb_[a-z0-9_]+)\s*\(", hdr)))
    assert declared == sorted(B.EXPORTS)
    L = B.lib()
    for name in declared:
        assert hasattr(L, name), name
    # the product library holds the method's calls and their helpers only: measurement aids live in libnbprobe.so
    assert not [n for n in declared if "probe" in n]


def test_probe_library_is_separate_and_exports_its_header(B):
    from paper_1411_5234_b200 import probes
    hdr = open(os.path.join(ROOT, "paper_1411_5234_b200", "csrc", "nb_probe.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = sorted(set(re.findall(r"\b(nbp_[a-z0-9_]+)\s*\(", hdr)))
    assert declared == sorted(probes.EXPORTS)
    L = probes.lib()
    for name in declared:
        assert hasattr(L, name), name
    assert L.nbp_fp64_peak(0, None, None, 0, 1.0, None, None) == -1            # argument validation needs no GPU
    for name in declared:
        assert not hasattr(B.lib(), name), name                                 # ... and none of it is in libnb.so


def test_build_staleness_tracks_every_header(B):
    from paper_1411_5234_b200 import build
    hs = {os.path.basename(h) for h in build._headers()}
    assert {"nb.h", "nb_internal.h", "nb_plan.h", "nb_probe.h"} <= hs
    assert not build.stale()


def test_struct_layouts_match_header(B):
    # nb_config: int, void*, void*, size_t, int, double, double, int, int, int, int  (natural alignment)
    assert C.sizeof(B.nb_config) == 80 and B.nb_config.order.offset == 64 and B.nb_config.check_indices.offset == 68 and B.nb_config.precision.offset == 72
    assert B.nb_config.workspace.offset == 16 and B.nb_config.eta.offset == 40 and B.nb_config.k_max.offset == 60
    assert C.sizeof(B.nb_plan) == 48 and B.nb_plan.waves.offset == 40 and B.nb_plan.predict_in_force.offset == 32


def test_workspace_bytes(B):
    assert B.nb_workspace_bytes(0) == 0 and B.nb_workspace_bytes(-5) == 0
    b1, b2 = B.nb_workspace_bytes(1), B.nb_workspace_bytes(256)
    assert b1 == b2 and b1 % 256 == 0                        # padded to 256 particles
    assert B.nb_workspace_bytes(257) > b2
    big = B.nb_workspace_bytes(1 << 20)
    assert 600e6 < big < 1.6e9                               # ~1.3 GB for 2^20 particles: fits 180 GB many times over


def wu_units(n_act):
    """The unit table of the warp-unit shape, restated from include/nb.h and csrc/nb_plan.h: n_act = 32 a + r -> a units of
    32, then r from its highest bit down, except that a rest missing at most an eighth (or one particle) of the next power of
    two is padded."""
    units, k = [(32 * u, 32, 32) for u in range(n_act // 32)], 32 * (n_act // 32)
    rem = n_act % 32
    while rem:
        pc = 1 << (rem - 1).bit_length()
        p, valid = (pc, rem) if pc - rem <= (pc // 8 if pc >= 16 else 1) else (1 << (rem.bit_length() - 1),) * 2
        units.append((k, p, valid))
        k += valid; rem -= valid
    return units


def test_warp_unit_decomposition():
    for n in range(1, 300):
        u = wu_units(n)
        assert sum(v for _, _, v in u) == n and u[0][0] == 0
        assert all(k0 == sum(v for _, _, v in u[:i]) for i, (k0, _, _) in enumerate(u))      # rows are contiguous
        assert all(p in (1, 2, 4, 8, 16, 32) and p - max(1, p // 8) <= v <= p for _, p, v in u)   # at most an eighth (or one) padded
        assert sum(p for _, p, _ in u) <= n * 8 / 7 + 1                                         # lanes spent vs particles
    assert [p for _, p, _ in wu_units(97)] == [32, 32, 32, 1]
    assert wu_units(31) == [(0, 32, 31)] and wu_units(21) == [(0, 16, 16), (16, 4, 4), (20, 1, 1)]
    assert wu_units(24) == [(0, 16, 16), (16, 8, 8)] and wu_units(3) == [(0, 4, 3)] and wu_units(28) == [(0, 32, 28)]


@pytest.mark.parametrize("N", [1, 2, 255, 1024, 5000, 65536, 262144, 1 << 20])
def test_plan_invariants(B, N):
    for n_act in sorted({1, 2, 7, 16, 17, 64, 96, 97, 255, 256, 300, 512, 1024, 1025, 1100, 4096, 16383, 16384, 32768, N // 3 + 1, N} & set(range(1, N + 1)) | {N}):
        for n_sm in (148, 132, 8):
            p = B.nb_plan_force(N, n_act, n_sm)
            Npad = (N + 255) // 256 * 256
            assert p.kernel == (0 if n_act >= 256 and n_act * 100 >= 93 * 128 * ((n_act + 127) // 128) else 1)
            assert p.unit == (128 if p.kernel == 0 else 32) and p.tile == (128 if p.kernel == 0 else 64)
            n_tiles = Npad // p.tile
            assert Npad % p.tile == 0
            assert p.n_units == ((n_act + 127) // 128 if p.kernel == 0 else len(wu_units(n_act)))
            assert p.predict_in_force == (1 if p.kernel == 1 and p.n_units <= 2 else 0)
            assert 1 <= p.ctas_per_sm <= 32 and 1 <= p.grid <= n_sm * p.ctas_per_sm
            S, st = p.n_split, p.slice_tiles
            assert S >= 1 and st >= 1
            assert S * st >= n_tiles and (S - 1) * st < n_tiles            # slices cover all j-tiles, none empty
            rows = p.n_units * 128 if p.kernel == 0 else n_act
            assert S * rows <= 8 * Npad + (1 << 19)                        # partial-sum buffer capacity
            # small active sets are split so that the device is filled
            resident = n_sm * p.ctas_per_sm * (4 if p.kernel == 1 else 1)       # warp units: 4 warps per CTA
            if p.n_units < resident and n_tiles >= 16 * resident:
                assert p.n_units * S >= 0.4 * resident


def test_plan_rejects_bad_sizes(B):
    p = B.nb_plan()
    L = B.lib()
    assert L.nb_plan_force(0, 1, 148, C.byref(p)) == B.NB_EINVAL
    assert L.nb_plan_force(10, 11, 148, C.byref(p)) == B.NB_EINVAL
    assert L.nb_plan_force(10, 0, 148, C.byref(p)) == B.NB_EINVAL
    assert L.nb_plan_force(10, 5, 0, C.byref(p)) == B.NB_EINVAL
    assert L.nb_plan_force(10, 5, 148, None) == B.NB_EINVAL


def test_argument_validation_without_gpu(B):
    L = B.lib()
    ctx = C.c_void_p()
    m = np.ones(4); x = np.zeros((4, 3)); v = np.zeros((4, 3))
    cfg = B.nb_config(0, None, None, 0, 0, 0, 0, 0, 0, 0, 0, 0)
    pm, px, pv = B._ptr(m), B._ptr(x), B._ptr(v)
    assert L.nb_init(C.byref(ctx), 4, pm, px, pv, 1e-3, C.byref(cfg)) == B.NB_ENOMEM       # no workspace
    assert L.nb_init(C.byref(ctx), 0, pm, px, pv, 1e-3, C.byref(cfg)) == B.NB_EINVAL
    assert L.nb_init(C.byref(ctx), 4, None, px, pv, 1e-3, C.byref(cfg)) == B.NB_EINVAL
    assert L.nb_init(C.byref(ctx), 4, pm, px, pv, float("nan"), C.byref(cfg)) == B.NB_EINVAL
    bad = B.nb_config(0, None, None, 0, 0, 0, 0, -3, -20, 0, 0, 0)                                   # k_min > k_max
    assert L.nb_init(C.byref(ctx), 4, pm, px, pv, 1e-3, C.byref(bad)) == B.NB_EINVAL
    assert L.nb_predict(None, 0.0) == B.NB_EINVAL
    assert L.nb_force(None, None, 0, None, None, None, None) == B.NB_EINVAL
    assert L.nb_check_indices(None, None, 0, 1) == B.NB_EINVAL
    assert L.nb_launch_count(None) == 0
    assert L.nb_strerror(B.NB_ESTATE).decode().startswith("call order")
    assert L.nb_strerror(12345).decode() == "unknown status"
    L.nb_free(None)


def test_product_path_has_no_oracle_or_cpu_fallback():
    """The package never imports oracle/, and System refuses to run without CUDA."""
    pkg = os.path.join(ROOT, "paper_1411_5234_b200")
    for fn in os.listdir(pkg):
        if fn.endswith(".py"):
            src = open(os.path.join(pkg, fn)).read()
            assert not re.search(r"^\s*(from|import)\s+oracle\b", src, flags=re.M), fn
    import torch
    if not torch.cuda.is_available():
        from paper_1411_5234_b200 import binding
        with pytest.raises(RuntimeError):
            binding.System(np.ones(2), np.zeros((2, 3)), np.zeros((2, 3)), 1e-3)


def test_plan_invariants_random_sizes(B):
    """The same invariants on 3000 seeded random (N, n_act, n_sm), log-uniform up to the N <= 2^30 the library accepts: slices
    cover the j-tiles with none empty, the launch fits the device, the partial sums fit the workspace, nothing that the kernels
    index with int overflows (such plans must be refused with NB_EINVAL, and only far beyond the paper's sizes)."""
    rng = np.random.default_rng(20260101)
    p, L = B.nb_plan(), B.lib()
    refused = 0
    for _ in range(3000):
        N = int(2 ** rng.uniform(0, 30))
        n_act = max(1, min(N, int(2 ** rng.uniform(0, np.log2(N) + 0.01)))) if rng.random() < 0.8 else N
        n_sm = int(rng.choice([1, 3, 8, 108, 132, 148, 160]))
        rc = L.nb_plan_force(N, n_act, n_sm, C.byref(p))
        if rc != B.NB_OK:
            assert rc == B.NB_EINVAL and N > 1 << 24, (N, n_act, n_sm, rc)
            refused += 1
            continue
        Npad = (N + 255) // 256 * 256
        n_tiles = Npad // p.tile
        S, st = p.n_split, p.slice_tiles
        assert p.kernel in (0, 1) and p.n_units >= 1 and S >= 1 and st >= 1, (N, n_act, n_sm)
        assert S * st >= n_tiles and (S - 1) * st < n_tiles, (N, n_act, n_sm)
        assert 1 <= p.grid <= n_sm * p.ctas_per_sm, (N, n_act, n_sm)
        rows = p.n_units * 128 if p.kernel == 0 else n_act
        assert S * rows <= 8 * Npad + (1 << 19), (N, n_act, n_sm)
        assert p.n_units * S < 2 ** 31 and rows < 2 ** 31, (N, n_act, n_sm)
        assert n_act > 4096 or p.n_units == ((n_act + 127) // 128 if p.kernel == 0 else len(wu_units(n_act))), (N, n_act, n_sm)
    assert refused < 300, refused


def test_shipped_kernels_fit_the_occupancy_the_plan_assumes(B):
    """The launch plan counts LI_CTAS_PER_SM = WU_CTAS_PER_SM = 4 resident CTAs of 128 threads per multiprocessor
    (csrc/nb_internal.h); with 65536 registers that is at most 128 registers per thread.  Read from the machine code of the
    shipped libnb.so (cuobjdump, no GPU): every force kernel fits, none has a local-memory frame beyond a few spill slots, and
    the static shared memory of every kernel stays under the 48 KiB that needs no opt-in."""
    import shutil
    if shutil.which("cuobjdump") is None:
        pytest.skip("cuobjdump (CUDA toolkit) is not on PATH")
    B.lib()
    out = subprocess.run(["cuobjdump", "--dump-resource-usage", B.LIB_PATH], stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    assert out.returncode == 0, out.stdout[-2000:]
    lines = out.stdout.split("\n")
    usage = {}
    for k, l in enumerate(lines):
        m_ = re.match(r"\s*Function (\S+):", l)
        if m_ and k + 1 < len(lines):
            r = dict(kv.split(":") for kv in re.findall(r"\b(?:REG|STACK|SHARED|LOCAL):\d+", lines[k + 1]))
            usage[m_.group(1)] = {key: int(val) for key, val in r.items()}
    force = {n: u for n, u in usage.items() if re.search(r"force_(li|lim|wu|step)_kernel", n)}
    assert len(force) >= 20, sorted(usage)                       # li / wu / step x eps x orders 4, 6, 8 + the mixed kernel x eps
    for n, u in force.items():
        assert u["REG"] <= 128, (n, u)                           # 4 CTAs x 128 threads x 128 registers = the register file
        assert u["LOCAL"] == 0 and u["STACK"] <= 96, (n, u)
    for n, u in usage.items():
        assert u["SHARED"] <= 48 * 1024 and u["REG"] <= 255, (n, u)
    assert any("reduce_correct_kernel" in n for n in usage) and any("sched_kernel" in n for n in usage) and any("predict_kernel" in n for n in usage)
