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
    sizes = sorted({1 << k for k in range(0, N.bit_length())} | {3, 9, 17, 24, 96, 97, 300, 1000, 1536, 30720, 98304, N} & set(range(1, N + 1)))
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
        rec["S"], rec["kernel"], rec["units"] = p.n_split, p.kernel, p.n_units
        rows.append(rec)
    g.nb_set_max_split(0)
    g.nb_free()
    return rows


def svg_plot(rows, N, path):
    """The figure as a text file: TFLOP/s against n_act on log-log axes, j-split on and off (no plotting library needed)."""
    W_, H_, L, R, T, Bm = 760, 440, 70, 20, 30, 50
    xs = [r["n_act"] for r in rows]
    inter = lambda r, arm: r["n_act"] * (N - 1) / r[arm] * FLOP / 1e12
    ymin, ymax = 1e-3, 40.0
    X = lambda n: L + (W_ - L - R) * np.log10(n) / np.log10(max(xs))
    Y = lambda y: H_ - Bm - (H_ - T - Bm) * (np.log10(max(y, ymin)) - np.log10(ymin)) / (np.log10(ymax) - np.log10(ymin))
    out = [f'<svg xmlns="http://www.w3.org/2000/svg" width="{W_}" height="{H_}" font-family="sans-serif" font-size="11">',
           f'<rect width="{W_}" height="{H_}" fill="white"/>',
           f'<text x="{W_ / 2}" y="16" text-anchor="middle" font-size="13">nb_force on B200, N = {N}: FP64 TFLOP/s (86 flop per interaction) against active particles</text>']
    for k in range(0, int(np.log10(max(xs))) + 1):
        out.append(f'<line x1="{X(10 ** k):.1f}" y1="{T}" x2="{X(10 ** k):.1f}" y2="{H_ - Bm}" stroke="#ddd"/>')
        out.append(f'<text x="{X(10 ** k):.1f}" y="{H_ - Bm + 15}" text-anchor="middle">1e{k}</text>')
    for y in (1e-3, 1e-2, 1e-1, 1, 10, 37.2):
        out.append(f'<line x1="{L}" y1="{Y(y):.1f}" x2="{W_ - R}" y2="{Y(y):.1f}" stroke="{"#c88" if y == 37.2 else "#ddd"}"/>')
        out.append(f'<text x="{L - 6}" y="{Y(y) + 4:.1f}" text-anchor="end">{y:g}</text>')
    out.append(f'<text x="{W_ - R}" y="{Y(37.2) - 4:.1f}" text-anchor="end" fill="#a44">FP64 FMA peak 37.2</text>')
    for arm, col, name in (("split", "#1565c0", "j-split chosen by the cost model"), ("nosplit", "#e65100", "S = 1 (Bfactor off)")):
        pts = " ".join(f"{X(r['n_act']):.1f},{Y(inter(r, arm)):.1f}" for r in rows)
        out.append(f'<polyline points="{pts}" fill="none" stroke="{col}" stroke-width="1.6"/>')
        out += [f'<circle cx="{X(r["n_act"]):.1f}" cy="{Y(inter(r, arm)):.1f}" r="2.4" fill="{col}"/>' for r in rows]
    out.append(f'<text x="{L + 12}" y="{T + 14}" fill="#1565c0">j-split chosen by the cost model</text>')
    out.append(f'<text x="{L + 12}" y="{T + 28}" fill="#e65100">S = 1 ("Bfactor off")</text>')
    out.append(f'<text x="{W_ / 2}" y="{H_ - 12}" text-anchor="middle">active particles n_act (m of PAPER.md:58)</text>')
    out.append("</svg>")
    open(path, "w").write("\n".join(out) + "\n")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--N", type=int, default=W.CONFIGS[3].N)
    ap.add_argument("--reps", type=int, default=5)
    ap.add_argument("--eps", type=float, default=1e-4)
    ap.add_argument("--svg", default=None, help="also write the figure (an SVG text file) here")
    a = ap.parse_args()
    rows = sweep(a.N, a.reps, a.eps)
    print(f"N = {a.N}, eps = {a.eps}; time = force launch + partial-sum reduction (CUDA events, best of {a.reps})")
    print("| n_act | kernel | units x S | time, split [us] | interactions/s | TFLOP/s | of the FP64 issue bound | time, S = 1 [us] | interactions/s | split speed-up |")
    print("|---|---|---|---|---|---|---|---|---|---|")
    names = {0: "CTA tiles", 1: "warp units"}
    for r in rows:
        inter = r["n_act"] * (a.N - 1)
        bound = 148 * 4 * 32 / 106 * 1.965e9           # pairs/s at 53 FP64 instructions x 2 cycles per pair
        print(f"| {r['n_act']} | {names[r['kernel']]} | {r['units']} x {r['S']} | {r['split'] * 1e6:.1f} | {inter / r['split']:.3e} | "
              f"{inter / r['split'] * FLOP / 1e12:.2f} | {inter / r['split'] / bound:.3f} | {r['nosplit'] * 1e6:.1f} | {inter / r['nosplit']:.3e} | "
              f"{r['nosplit'] / r['split']:.2f} |")
    if a.svg:
        svg_plot(rows, a.N, a.svg)


if __name__ == "__main__":
    main()
