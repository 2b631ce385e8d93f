#!/usr/bin/env python
"""bench.py — headline benchmark of the Hermite-6 pairwise evaluation on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--N particles]

One STEP = one pass of the whole hot path over the workload: nb_predict(t + dt) for all N, nb_force for
all N active (the lanes-over-i kernel + the j-split partial-sum reduction), nb_corrector for all N.
Workload at N = 1 GPU: BASELINE.json configs[3] — N = 2^20 equal-mass Plummer sphere, eps = 1e-4, all
active.  Multi-GPU (--gpus N under torchrun): replicas only: every rank steps its
own system of the same size (seed + rank); no data-path collective; scaling = weak.

Prints ONE JSON line (rank 0).  `--impl reference` times the CPU oracle (oracle/, fp64 build) on the host
cores on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_1411_5234_b200 import workloads as W  # noqa: E402

METRIC = "fp64 pairwise interactions/s (acc+jerk+snap) at N=2^20"
UNIT = "interactions/s"
FLOP_EXEC = 86   # ALGORITHMIC flop per interaction: 2*32 FMA + 11 MUL + 11 ADD; this is what roofline.achieved counts
FLOP_PIPE = 85   # of which the shipped SASS executes 85 on the FP64 pipe (32 DFMA + 11 DMUL + 10 DADD, profiles/r02_sass_tables.md);
                 # the 86th (2 c1) is an exponent increment on the integer pipe.  roofline.frac_pipe_executed uses this count
FLOP_CONV = 97   # customary acc+jerk+snap operation count of the Hermite-6 literature (a labelled convention)
FP64_LANES_PER_SM = 64
DT_BENCH = 2.0 ** -14
# dram__bytes_read.sum + dram__bytes_write.sum per force launch, by N, from the committed ncu --set full captures (profiles/)
TRAFFIC = {1048576: 656.7e6 + 647.6e6, 262144: 41.2e6 + 160.5e6}


def n_cores() -> int:
    return len(os.sched_getaffinity(0))


# ------------------------------------------------------------------------------------------ multi-rank plumbing
def replica_seed(base_seed: int, rank: int, world: int) -> int:
    """Replicas only: rank r of an N > 1 run steps its own realisation of the workload."""
    return base_seed if world == 1 else base_seed + 1000 * rank


def max_over_ranks(x: float, world: int, device="cpu") -> float:
    """The job's time is the slowest rank's (all-reduce MAX; works on nccl with a cuda device and on gloo with cpu)."""
    if world == 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(world: int, steps: int, units_per_step_per_rank: float, ms: float) -> float:
    """Units all ranks processed / the max-over-ranks time (weak scaling: per-rank work is fixed)."""
    return world * steps * units_per_step_per_rank / (ms * 1e-3)


# ------------------------------------------------------------------------------------------ clocks
class ClockSampler:
    """nvidia-smi clocks/throttle reasons sampled DURING the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.rows, self.proc, self.gpu = [], None, gpu_index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "200", "-i", str(self.gpu)], stdout=subprocess.PIPE, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([s.strip() for s in line.split(",")])

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        time.sleep(0.05)
        sm, smax, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); smax.append(float(r[1])); pw.append(float(r[2]))
            except (ValueError, IndexError):
                continue
            for n, val in zip(names, r[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------ CPU oracle legs
def time_oracle_sample(m, x, v, a, eps, seconds: float, seed: int):
    """The oracle as it stands (fp64 build, OpenMP over i) on a bounded sample: K_i sampled i-particles
    against all N j-particles.  Returns (interactions/s, sample description)."""
    import oracle
    N = m.shape[0]
    probe = W.active_set(N, min(N, 64), seed)
    t0 = time.perf_counter()
    oracle.hermite6.force(m, x, v, a, eps, probe, kind="f64")
    rate = probe.size * (N - 1) / (time.perf_counter() - t0)
    k = int(min(N, max(64, rate * seconds / (N - 1))))
    idx = W.active_set(N, k, seed + 1)
    t0 = time.perf_counter()
    oracle.hermite6.force(m, x, v, a, eps, idx, kind="f64")
    el = time.perf_counter() - t0
    return k * (N - 1) / el, f"{k} seeded i-particles x all {N} j-particles ({k * (N - 1):.3g} interactions, {el:.1f} s)"


def run_reference(args, cfg_dict):
    """--impl reference: the CPU oracle, rank 0 only."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    c, m, x, v = W.config_inputs(4, N=args.N)
    a = np.zeros_like(x)
    N = m.shape[0]
    import oracle
    oracle.build()
    # size one step at ~4 s of CPU work
    probe = W.active_set(N, min(N, 64), 7)
    t0 = time.perf_counter()
    oracle.hermite6.force(m, x, v, a, c.eps, probe, kind="f64")
    rate = probe.size * (N - 1) / (time.perf_counter() - t0)
    k = int(min(N, max(64, rate * 4.0 / (N - 1))))
    for w in range(args.warmup):
        oracle.hermite6.force(m, x, v, a, c.eps, W.active_set(N, k, 100 + w), kind="f64")
    t0 = time.perf_counter()
    for s in range(args.steps):
        oracle.hermite6.force(m, x, v, a, c.eps, W.active_set(N, k, 200 + s), kind="f64")
    el = time.perf_counter() - t0
    value = args.steps * k * (N - 1) / el
    sample = f"each step = {k} seeded i-particles x all {N} j-particles of the same workload"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": el / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": cfg_dict,
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": n_cores(), "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------ the CUDA arm
def run_ours(args, cfg_dict):
    import torch
    import torch.distributed as dist
    from paper_1411_5234_b200 import binding as B

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device — the CUDA path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    c, m, x, v = W.config_inputs(4, N=args.N)
    if world > 1:                                       # replicas: every rank its own realisation
        m, x, v = W.plummer(m.shape[0], replica_seed(c.seed, rank, world), c.masses)
    N = m.shape[0]
    inter_per_step = N * (N - 1)

    dev = f"cuda:{local}"
    g = B.System(torch.tensor(m, device=dev), torch.tensor(x, device=dev), torch.tensor(v, device=dev), c.eps,
                 host=False, device=local)
    torch.cuda.synchronize()

    t_sim = [0.0]

    def step():
        t_sim[0] += DT_BENCH
        g.nb_predict(t_sim[0])
        g.nb_force(None, outputs=False)
        g.nb_corrector(None, DT_BENCH)

    for _ in range(args.warmup):
        step()
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    launches0 = g.nb_launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    force_ms = []
    ev0.record()
    for _ in range(args.steps):
        step()
        force_ms.append(g.nb_last_force_ms())           # CUDA events on the launch stream, recorded by nb_force
    ev1.record()
    barrier()
    ms = ev0.elapsed_time(ev1)
    launches = g.nb_launch_count() - launches0
    clocks = sampler.stop() if rank == 0 else None
    ms = max_over_ranks(ms, world, dev)
    value = whole_job_value(world, args.steps, inter_per_step, ms)

    # ---- end to end through the C ABI with HOST buffers (pinned): H2D of x, v and D2H of a, jerk, snap, pot every step
    gh = B.System(m, x, v, c.eps, host=True, device=local)
    pin = lambda arr: torch.from_numpy(arr.copy()).pin_memory().numpy()
    xh, vh = pin(x), pin(v)
    h2d = xh.nbytes + vh.nbytes
    d2h = N * 10 * 8
    t_h = [0.0]

    def step_host():
        t_h[0] += DT_BENCH
        gh.nb_set_state("X", xh); gh.nb_set_state("V", vh)
        gh.nb_predict(t_h[0])
        out = gh.nb_force(None)
        gh.nb_corrector(None, DT_BENCH)
        return out

    e2e_steps = max(1, min(args.steps, 2))
    step_host()
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        res = step_host()
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    e2e_s = max_over_ranks(e2e_s, world, dev)
    e2e_value = whole_job_value(world, e2e_steps, inter_per_step, e2e_s * 1e3)
    assert np.isfinite(res[0]).all()

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (nb_force: FP64 ALU pipe)
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except OSError:
        pass
    n_sm = torch.cuda.get_device_properties(local).multi_processor_count
    sm_max_mhz = float(peaks.get("sm_max_mhz") or (clocks or {}).get("sm_max_mhz") or 1965.0)
    peak_nominal = n_sm * FP64_LANES_PER_SM * 2 * sm_max_mhz * 1e6 / 1e12       # TFLOP/s, all-FMA
    from paper_1411_5234_b200 import probes as P          # libnbprobe.so: measurement aids, not part of libnb.so
    peak_measured, _ = P.fp64_peak(1.0, local)
    pipe_probe = P.dfma_sources(sm_max_mhz, local)            # cycles per DFMA: 2 / 3 / 3-with-reuse register sources
    f_ms = float(np.mean(force_ms))
    achieved = FLOP_EXEC * inter_per_step / (f_ms * 1e-3) / 1e12
    roofline = {"bound": "alu", "kernel": "force_li_kernel<false, 6> (+ reduce_partials_kernel<10>)", "achieved": achieved,
                "peak": peak_nominal, "unit": "TFLOP/s", "frac": achieved / peak_nominal,
                "frac_pipe_executed": FLOP_PIPE * inter_per_step / (f_ms * 1e-3) / 1e12 / peak_nominal,
                "peak_source": f"derived: {n_sm} SMs x {FP64_LANES_PER_SM} FP64 FMA lanes x 2 x {sm_max_mhz:.0f} MHz (DESIGN.md)",
                "peak_measured_dfma": peak_measured, "frac_of_measured_dfma": achieved / peak_measured,
                "flop_per_interaction": FLOP_EXEC, "pipe_probe": pipe_probe, "tflops_conv97": FLOP_CONV * inter_per_step / (f_ms * 1e-3) / 1e12,
                "kernel_ms": f_ms, "kernel_share_of_step": f_ms * args.steps / ms,
                "interactions_per_s_kernel": inter_per_step / (f_ms * 1e-3),
                "traffic": TRAFFIC.get(N),
                "traffic_source": "profiles/r02_force_li_full.md (dram__bytes_read.sum + dram__bytes_write.sum of one ncu --set full capture "
                                  "of this kernel at this N; null at sizes that were not captured)"}

    # ---- the paper's own precision scheme, measured beside the fp64 path on the same workload: one evaluation
    gm = B.System(torch.tensor(m, device=dev), torch.tensor(x, device=dev), torch.tensor(v, device=dev), c.eps, host=False, device=local,
                  precision=B.NB_PREC_MIXED)
    gm.nb_predict(DT_BENCH)
    mixed_ms = []
    for _ in range(2):
        gm.nb_force(None, outputs=False)
        mixed_ms.append(gm.nb_last_force_ms())
    gm.nb_free()
    mixed = {"what": "nb_config.precision = NB_PREC_MIXED (fp64 position differences and accumulation, fp32 pair arithmetic); NOT the headline: "
                     "about 1e-6 per particle against the oracle (tests/test_gpu_parity.py::test_mixed_precision_accuracy_against_oracle)",
             "interactions_per_s_kernel": inter_per_step / (min(mixed_ms) * 1e-3), "kernel_ms": min(mixed_ms), "speedup_over_fp64": f_ms / min(mixed_ms)}

    # ---- the oracle timed beside it (rank 0, bounded sample)
    cpu_val, sample = time_oracle_sample(m, x, v, np.zeros_like(x), c.eps, args.cpu_seconds, 31)
    cpu = {"value": cpu_val, "unit": UNIT, "cores": n_cores(), "kind": "oracle", "sample": sample}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": cfg_dict, "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "steps": e2e_steps},
            "gpu_launches": int(launches), "roofline": roofline, "cpu_baseline": cpu, "mixed_precision": mixed}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--N", type=int, default=None, help="override the particle count (development; default 2^20)")
    ap.add_argument("--cpu-seconds", type=float, default=12.0, help="CPU work budget of the cpu_baseline sample")
    args = ap.parse_args()
    N = args.N or W.CONFIGS[4].N
    cfg_dict = {"workload": f"BASELINE.json configs[3]: N={N} equal-mass Plummer sphere (seeded, Henon units), eps=1e-4, fp64, "
                            "all N active; step = nb_predict + nb_force(all) + nb_corrector(all)",
                "N": N, "n_act": N, "eps": 1e-4, "dt": DT_BENCH,
                "parallelism": "single GPU" if args.gpus == 1 else f"{args.gpus} independent replicas, one system per GPU, no collective "
                                                                    "(the path is not sharded in this build: DESIGN.md 9)",
                "l2": "per-step working set (state 176 MB + j-records 84 MB + partial sums 671 MB + results 84 MB) exceeds the 126 MB L2"}
    if args.impl == "reference":
        run_reference(args, cfg_dict)
    else:
        run_ours(args, cfg_dict)


if __name__ == "__main__":
    main()
