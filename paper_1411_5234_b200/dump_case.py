"""Raw results of a fixed set of calls, for comparing two builds of libnb.so bit for bit.

    NB_LIB=/path/to/libnb_ptxas.so python -m paper_1411_5234_b200.dump_case OUT.npz

Seeded Plummer spheres (config 4's recipe at small sizes, eps = 1e-4 and eps = 0), orders 4, 6 and 8: nb_force for all particles
and for active sets of 1000, 37 and 1 particles (CTA tiles and warp units, with and without the self-pair mask), then 200
device-planned block steps (nb_run_blocks) at the 6th order.  tests/test_gpu_parity.py runs this once per build
(sass_sched.py's and ptxas's own) and compares the files.
"""
from __future__ import annotations

import sys

import numpy as np

from . import binding as B
from . import workloads as W


def main(path: str) -> None:
    import torch
    dev, out = "cuda:0", {}
    host = lambda t: t.cpu().numpy() if hasattr(t, "cpu") else np.asarray(t)
    for order in (6, 4, 8):
        for N, eps in ((20000, 1e-4), (4097, 0.0)):
            m, x, v = W.plummer(N, W.BASE_SEED + 4, "equal")
            g = B.System(torch.tensor(m, device=dev), torch.tensor(x, device=dev), torch.tensor(v, device=dev), eps, host=False, order=order)
            g.nb_predict(2.0 ** -10)
            for n_act in (N, 1000, 37, 1):
                idx = None if n_act == N else torch.tensor(W.active_set(N, n_act, 5), device=dev)
                for name, a in zip("ajsp", g.nb_force(idx)):
                    out[f"o{order}_N{N}_n{n_act}_{name}"] = host(a)
            if order == 6 and N == 20000:
                g.nb_run_blocks(2.0 ** -6, 200)
                for f in ("X", "V", "A", "DT"):
                    out[f"o{order}_N{N}_blocks_{f}"] = host(g.nb_get_state(f))
            g.nb_free()
    np.savez(path, **out)
    print(f"{len(out)} arrays, library {B.LIB_PATH}")


if __name__ == "__main__":
    main(sys.argv[1])
