"""Performance of nb_force against the number of active particles, with the j-split on and off.

    python -m paper_1411_5234_b200.sweep_nact [--N 262144] [--reps 5] [--eps 1e-4]

This is the B200 analogue of the paper's Fig. 1 (HiGPUs on a GTX TITAN Black, "a typical N-body
simulation with N ~ 260,000", performance as a function of the m active particles with the `Bfactor` variable on and
off).  The figure's data are not in the paper's text, so only the shape can be compared: without the split the rate
collapses once m falls below the number of lanes the GPU keeps busy, with it the rate stays within a small factor of
the all-active one.  Prints a markdown table: device time of the force launch (+ partial-sum reduction), pairwise
interactions/s and TFLOP/s at 86 flop per interaction, for the split chosen by the cost model and for S = 1.
Seeded Plummer sphere of BASELINE.json configs[2]'s size (equal masses, the rate does not depend on them).
"""
from __future__ import annotations

import argparse

import numpy as np

from . import binding as B
from . import workloads as W

FLOP = 86


def sweep(N: int, reps: int, eps: float, device: int = 0):
    import torch
    m, x, v = W.plummer(N, W.BASE_SEED + 2, "equal")
    dev = f"cuda:{device}"
    g = B.System(torch.tensor(m, device=dev), torch.tensor(x, device=dev), torch.tensor(v, device=dev), eps, host=False, device=device)
    g.nb_predict(2.0 ** -10)
    sizes = sorted({1 << k for k in range(0, N.bit_length())} | {3, 24, 96, 97, 1536, 30720, 98304, N} & set(range(1, N + 1)))
    rows = []
    for n_act in sizes:
        idx = None if n_act == N else torch.tensor(W.active_set(N, n_act, 5), device=dev)
        rec = {"n_act": n_act}
        for arm, cap in (("split", 0), ("nosplit", 1)):
            g.nb_set_max_split(cap)
            ts = []
            for _ in range(reps + 1):
                g.nb_force(idx, outputs=False)
                ts.append(g.nb_last_force_ms())
            rec[arm] = min(ts[1:]) * 1e-3                      # the first call warms up
        p = B.nb_plan_force(N, n_act, torch.cuda.get_device_properties(device).multi_processor_count)
        rec["S"], rec["kernel"], rec["sub"] = p.n_split, p.kernel, p.sub
        rows.append(rec)
    g.nb_set_max_split(0)
    g.nb_free()
    return rows


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--N", type=int, default=W.CONFIGS[3].N)
    ap.add_argument("--reps", type=int, default=5)
    ap.add_argument("--eps", type=float, default=1e-4)
    a = ap.parse_args()
    rows = sweep(a.N, a.reps, a.eps)
    print(f"N = {a.N}, eps = {a.eps}; time = force launch + partial-sum reduction (CUDA events, best of {a.reps})")
    print("| n_act | kernel | S x sub | time, split [us] | interactions/s | TFLOP/s | time, S = 1 [us] | interactions/s | split speed-up |")
    print("|---|---|---|---|---|---|---|---|---|")
    names = {0: "lanes-over-i", 1: "lanes-over-j", 2: "lanes-over-i/32"}
    for r in rows:
        inter = r["n_act"] * (a.N - 1)
        print(f"| {r['n_act']} | {names[r['kernel']]} | {r['S']} x {r['sub']} | {r['split'] * 1e6:.1f} | {inter / r['split']:.3e} | "
              f"{inter / r['split'] * FLOP / 1e12:.2f} | {r['nosplit'] * 1e6:.1f} | {inter / r['nosplit']:.3e} | {r['nosplit'] / r['split']:.2f} |")


if __name__ == "__main__":
    main()
