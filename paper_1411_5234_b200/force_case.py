"""One nb_force configuration, repeated: the case the ncu captures under profiles/ are taken on.

    python -m paper_1411_5234_b200.force_case --N 1048576 --n-act 8 [--reps 4] [--precision fp64|mixed] [--order 6]

Seeded Plummer sphere (config 4's recipe at size N, eps = 1e-4), one nb_predict, then `reps` calls of nb_force for the
same random active set (config 5's recipe).  Prints the launch plan and, per call, the device time of force kernel +
partial-sum reduction (CUDA events on the launch stream, nb_last_force_ms).
"""
from __future__ import annotations

import argparse

from . import binding as B
from . import workloads as W


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--N", type=int, default=W.CONFIGS[4].N)
    ap.add_argument("--n-act", type=int, default=8)
    ap.add_argument("--reps", type=int, default=4)
    ap.add_argument("--precision", default="fp64", choices=["fp64", "mixed"])
    ap.add_argument("--order", type=int, default=6)
    a = ap.parse_args()
    import torch
    m, x, v = W.plummer(a.N, W.BASE_SEED + 4, "equal")
    dev = "cuda:0"
    g = B.System(torch.tensor(m, device=dev), torch.tensor(x, device=dev), torch.tensor(v, device=dev), W.CONFIGS[4].eps, host=False,
                 order=a.order, precision=B.NB_PREC_MIXED if a.precision == "mixed" else B.NB_PREC_FP64)
    g.nb_predict(2.0 ** -10)
    idx = None if a.n_act == a.N else torch.tensor(W.config5_active(a.n_act, a.N) if a.n_act & (a.n_act - 1) == 0 else W.active_set(a.N, a.n_act, 5), device=dev)
    p = B.nb_plan_force(a.N, a.n_act, torch.cuda.get_device_properties(0).multi_processor_count)
    print(f"N = {a.N}, n_act = {a.n_act}, order {a.order}, {a.precision}: kernel {p.kernel} ({'CTA tiles' if p.kernel == 0 else 'warp units'}), "
          f"{p.n_units} units x S = {p.n_split} slices of {p.slice_tiles} tiles of {p.tile}, grid {p.grid}; "
          f"resident CTAs per SM: {g.nb_resident_ctas(p.kernel)}")
    inter = a.n_act * (a.N - 1)
    for r in range(a.reps):
        g.nb_force(idx, outputs=False)
        ms = g.nb_last_force_ms()
        print(f"  call {r}: {ms * 1e3:.1f} us, {inter / (ms * 1e-3):.4e} interactions/s")
    g.nb_free()


if __name__ == "__main__":
    main()
