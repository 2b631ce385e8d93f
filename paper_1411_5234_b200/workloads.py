"""Seeded synthetic inputs shaped like the paper's runs (BASELINE.json configs).

This module serves BOTH the oracle and the CUDA path and therefore holds none of the
method's arithmetic: no forces, no predictor/corrector, no time steps — only initial
conditions, masses and active-index sets, all from numpy's PCG64 (`default_rng(seed)`).

Recipe: Plummer sphere by the Aarseth-Henon-Wielen sampling, Henon
units G = M = 1, E = -1/4 in expectation, centre of mass removed, no radial cut-off.
"""
from __future__ import annotations

import hashlib
from dataclasses import dataclass

import numpy as np

BASE_SEED = 14115234  # the arXiv id; config k uses BASE_SEED + k


@dataclass(frozen=True)
class Config:
    """One BASELINE.json config: sizes and parameters, no data."""
    index: int
    N: int
    eps: float
    masses: str          # "equal" | "kroupa"
    dt: float | None     # shared step (configs 1, 2); None = block time steps / single evaluation
    n_steps: int
    n_act: tuple = ()    # config 5 sweep

    @property
    def seed(self) -> int:
        return BASE_SEED + self.index


CONFIGS = {
    1: Config(1, 1024, 1e-3, "equal", 1.0 / 1024, 8),
    2: Config(2, 65536, 1e-4, "equal", 2.0 ** -12, 16),
    3: Config(3, 262144, 1e-4, "kroupa", None, 0),
    4: Config(4, 1048576, 1e-4, "equal", None, 0),
    5: Config(5, 1048576, 1e-4, "equal", None, 0, (1, 8, 64, 512, 4096, 32768)),
}


def equal_masses(N: int) -> np.ndarray:
    return np.full(N, 1.0 / N, dtype=np.float64)


def kroupa_masses(N: int, rng: np.random.Generator) -> np.ndarray:
    """Broken power law dN/dm ~ m^-1.3 on [0.1, 0.5), ~ m^-2.3 on [0.5, 100], continuous at 0.5,
    inverse-CDF sampled, then normalised to sum 1 (BASELINE.json configs[2])."""
    m_lo, m_br, m_hi = 0.1, 0.5, 100.0
    a1, a2 = 1.3, 2.3
    c2 = m_br ** (a2 - a1)                       # continuity at the break
    I1 = (m_lo ** (1 - a1) - m_br ** (1 - a1)) / (a1 - 1)
    I2 = c2 * (m_br ** (1 - a2) - m_hi ** (1 - a2)) / (a2 - 1)
    u = rng.random(N) * (I1 + I2)
    m = np.empty(N, dtype=np.float64)
    lo = u < I1
    m[lo] = (m_lo ** (1 - a1) - u[lo] * (a1 - 1)) ** (1.0 / (1 - a1))
    w = (u[~lo] - I1) / c2
    m[~lo] = (m_br ** (1 - a2) - w * (a2 - 1)) ** (1.0 / (1 - a2))
    return m / m.sum()


def plummer(N: int, seed: int, masses: str = "equal"):
    """Return (m[N], x[N,3], v[N,3]) float64, C-contiguous."""
    rng = np.random.default_rng(seed)
    m = equal_masses(N) if masses == "equal" else kroupa_masses(N, rng)

    tiny = 2.0 ** -53
    X1 = np.clip(rng.random(N), tiny, 1.0 - tiny)
    r = 1.0 / np.sqrt(X1 ** (-2.0 / 3.0) - 1.0)
    X2, X3 = rng.random(N), rng.random(N)
    z = (1.0 - 2.0 * X2) * r
    rxy = np.sqrt(np.maximum(r * r - z * z, 0.0))
    x = np.stack([rxy * np.cos(2 * np.pi * X3), rxy * np.sin(2 * np.pi * X3), z], axis=1)

    # speed fraction q = V / V_escape by von Neumann rejection on g(q) = q^2 (1 - q^2)^(7/2) < 0.1
    q = np.empty(N, dtype=np.float64)
    filled = 0
    while filled < N:
        need = N - filled
        X4 = rng.random(2 * need + 16)
        X5 = rng.random(2 * need + 16)
        ok = X4[0.1 * X5 < X4 * X4 * (1.0 - X4 * X4) ** 3.5]
        take = min(need, ok.size)
        q[filled:filled + take] = ok[:take]
        filled += take
    V = q * np.sqrt(2.0) * (1.0 + r * r) ** -0.25
    X6, X7 = rng.random(N), rng.random(N)
    vz = (1.0 - 2.0 * X6) * V
    vxy = np.sqrt(np.maximum(V * V - vz * vz, 0.0))
    v = np.stack([vxy * np.cos(2 * np.pi * X7), vxy * np.sin(2 * np.pi * X7), vz], axis=1)

    # Henon units
    x *= 3.0 * np.pi / 16.0
    v *= np.sqrt(16.0 / (3.0 * np.pi))
    # centre of mass at rest at the origin
    x -= (m[:, None] * x).sum(0) / m.sum()
    v -= (m[:, None] * v).sum(0) / m.sum()
    return m, np.ascontiguousarray(x), np.ascontiguousarray(v)


def config_inputs(index: int, N: int | None = None):
    """Inputs of BASELINE.json configs[index-1]; `N` overrides the size (reduced-N twins)."""
    c = CONFIGS[index]
    m, x, v = plummer(N or c.N, c.seed, c.masses)
    return c, m, x, v


def active_set(N: int, n_act: int, seed: int) -> np.ndarray:
    """Unique random indices, unsorted, int32 (config 5)."""
    rng = np.random.default_rng(seed)
    return rng.choice(N, size=n_act, replace=False).astype(np.int32)


def config5_active(n_act: int, N: int | None = None) -> np.ndarray:
    c = CONFIGS[5]
    rank = int(np.log2(n_act)) if n_act > 0 else 0
    return active_set(N or c.N, n_act, BASE_SEED + 50 + rank)


def sha256(*arrays: np.ndarray) -> str:
    h = hashlib.sha256()
    for a in arrays:
        h.update(np.ascontiguousarray(a).tobytes())
    return h.hexdigest()
