"""BASELINE.json configs[2]: the block-time-step run (N = 262144 Plummer sphere, Kroupa-like masses, eps = 1e-4,
levels 2^-3 .. 2^-20 by the Aarseth criterion, 1/8 time unit), advanced with nb_run_blocks.

    python -m paper_1411_5234_b200.config3 [--N 262144] [--t-end 0.125] [--order 6] [--eta 0] [--profile-steps 1500]

Prints the run's totals (block steps, interactions, wall time, energy drift) and, from a second stretch driven one
step at a time, the device time per block step by active-set size.  PAPER.md:58 (block time steps)
(the small-active-set regime the j-split is for).
"""
from __future__ import annotations

import argparse
import time

import numpy as np

from . import binding as B
from . import workloads as W


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--N", type=int, default=None)
    ap.add_argument("--t-end", type=float, default=0.125)
    ap.add_argument("--order", type=int, default=6)
    ap.add_argument("--profile-steps", type=int, default=3000)
    ap.add_argument("--eta", type=float, default=0.0, help="accuracy parameter of the time-step criterion (0: the order's default)")
    a = ap.parse_args()
    import torch
    c, m, x, v = W.config_inputs(3, N=a.N)
    N = m.shape[0]
    dev = "cuda:0"
    g = B.System(torch.tensor(m, device=dev), torch.tensor(x, device=dev), torch.tensor(v, device=dev), c.eps,
                 host=False, device=0, order=a.order, eta=a.eta)
    K0, W0 = g.nb_energy()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    steps, t_last, sum_act = g.nb_run_blocks(a.t_end)
    torch.cuda.synchronize()
    el = time.perf_counter() - t0
    K1, W1 = g.nb_energy()
    inter = sum_act * (N - 1)
    print(f"N = {N}, order {a.order}, eta = {a.eta or 'default'}, eps = {c.eps}: {steps} block steps to t = {t_last}, {sum_act / N:.1f} steps per particle, "
          f"{inter:.4e} interactions in {el:.3f} s = {inter / el:.4e} interactions/s; dE/E = {(K1 + W1) / (K0 + W0) - 1:.3e}")
    if a.profile_steps <= 0:
        return
    # per-step cost from the device's own step log (nb_step_log): differences of the device clock between consecutive steps
    g.nb_run_blocks(1e30, a.profile_steps)
    na, tu = g.nb_step_log(a.profile_steps)
    rec = np.stack([na[1:], np.diff(tu)], axis=1)
    print(f"next {len(rec)} block steps in one nb_run_blocks call; cost per step = difference of the device clock (nb_step_log):")
    print("| n_act | steps | median us/step | min us/step | mean n_act | FP64-pipe floor us (106 cycles per pair) |")
    print("|---|---|---|---|---|---|")
    for lo, hi in ((1, 1), (2, 4), (5, 16), (17, 32), (33, 96), (97, 256), (257, 1024), (1025, 8192), (8193, N)):
        sel = (rec[:, 0] >= lo) & (rec[:, 0] <= hi)
        if sel.any():
            na_, us = rec[sel, 0], rec[sel, 1]
            floor = na_.mean() * (N - 1) * 106 / (148 * 4 * 32 * 1.965e9) * 1e6
            print(f"| {lo}..{hi} | {int(sel.sum())} | {np.median(us):.1f} | {us.min():.1f} | {na_.mean():.1f} | {floor:.1f} |")
    g.nb_free()


if __name__ == "__main__":
    main()
