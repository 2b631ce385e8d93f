"""The small case that is run under compute-sanitizer (memcheck, racecheck; one tool per call):

    compute-sanitizer --tool memcheck  python -m paper_1411_5234_b200.sanitize_case
    compute-sanitizer --tool racecheck python -m paper_1411_5234_b200.sanitize_case

Config 1 (N = 1024: startup, predict, force, 8 shared steps, energy) and 40 device-planned block steps plus 10 block
steps by separate calls of an N = 4096 Plummer sphere with Kroupa masses, so that every kernel of libnb.so runs: both
force shapes with their TMA / mbarrier staging, the work queue and its reset, predict-in-force, the one-kernel scheduler
with its last-block pass, the fused reduction + corrector, the CUDA-graph path, the index check and the mixed-precision
kernel.  Prints a one-line summary; the summaries under profiles/ are the sanitizer's own report of this run.
"""
from __future__ import annotations

import numpy as np

from . import binding as B
from . import workloads as W


def main():
    c, m, x, v = W.config_inputs(1)
    g = B.System(m, x, v, c.eps)
    g.nb_predict(0.0)
    g.nb_force()
    t = 0.0
    for _ in range(c.n_steps):
        t += c.dt
        g.nb_predict(t); g.nb_force(outputs=False); g.nb_corrector(None, c.dt)
    e1 = sum(g.nb_energy())
    g.nb_free()

    N = 4096
    m, x, v = W.plummer(N, 99, "kroupa")
    g = B.System(m, x, v, 1e-4)
    steps, t_last, n_sum = g.nb_run_blocks(1e30, 40)
    for _ in range(10):
        tn, n, act = g.nb_next_block()
        g.nb_predict(tn); g.nb_force(act, outputs=False); g.nb_corrector(act, 0.0)
    g.nb_predict(tn)
    for n_act in (1, 5, 17, 100, 300, 1024, N):             # warp units of every width, ragged and full CTA tiles
        idx = None if n_act == N else W.active_set(N, n_act, n_act)
        a = g.nb_force(idx)[0]
        assert np.isfinite(a).all()
    assert g.nb_check_indices(np.array([1, 2, 2], dtype=np.int32)) == B.NB_EINVAL
    na, tu = g.nb_step_log()
    g.nb_free()

    gm = B.System(m, x, v, 1e-4, precision=B.NB_PREC_MIXED)
    gm.nb_predict(2.0 ** -10)
    am = gm.nb_force()[0]
    gm.nb_free()
    for order in (4, 8):
        go = B.System(m[:600].copy(), x[:600].copy(), v[:600].copy(), 1e-3, order=order)
        go.nb_run_blocks(1e30, 8)
        go.nb_free()
    print(f"sanitize_case: config 1 energy {e1:.6f}; N = {N}: {steps} block steps to t = {t_last}, sum n_act {n_sum}, "
          f"log {na.size} entries; mixed |a| max {np.abs(am).max():.3e}")


if __name__ == "__main__":
    main()
