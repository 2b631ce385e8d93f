"""B200-native direct-summation N-body hot path (Hermite-6 acc+jerk+snap), arXiv:1411.5234.

The package holds the CUDA/C-ABI library (`csrc/` -> `libnb.so`), its thin ctypes binding
(`binding`) and the seeded input generators (`workloads`, no method arithmetic).  Nothing is
imported eagerly: `workloads` must stay importable without the CUDA library.
"""

__all__ = ["binding", "workloads", "build"]
