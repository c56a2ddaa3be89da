"""Seeded synthetic inputs shared by the tests, the oracle harness and bench.py.

This module holds NO arithmetic of the method (no force, jerk, potential,
predictor or integrator formula): it only draws the paper's workload -- "equal
mass particles of a Plummer sphere" in N-body units (Table 1
caption; L138 N-body units, Heggie & Mathieu) -- from a seed, plus the
block-step bookkeeping inputs (active i-sets, particle times) that the
BASELINE.json configs name.  Both the CUDA path and the oracle consume these
arrays; neither is imported here.

Recipe: textbook Aarseth-Henon-Wielen construction.
  radius      r = (X^(-2/3) - 1)^(-1/2),  X ~ U(0, 0.999)  (99.9 % mass cut)
  direction   isotropic
  speed       q by von Neumann rejection on g(q) = q^2 (1-q^2)^(7/2),
              v = q * sqrt(2) * (1 + r^2)^(-1/4)
  units       x *= 3*pi/16,  v *= sqrt(16/(3*pi))   (G = M = 1, E = -1/4)
  frame       centre-of-mass position and velocity removed
The draw order is fixed, so (seed, N) -> bit-identical arrays for one numpy.
"""
from __future__ import annotations

import numpy as np

MASS_CUT = 0.999

# BASELINE.json configs: (N, seed).  eps = 1/256 unless a config says eps = 0.
CONFIGS = {
    "C1": dict(N=1024, seed=1),
    "C2": dict(N=16384, seed=2),
    "C3": dict(N=131072, seed=3),
    "C4": dict(N=1048576, seed=4),
    "C5": dict(N=65536, seed=5),
}
EPS_PAPER = 1.0 / 256.0


def _isotropic(rng: np.random.Generator, n: int, length: np.ndarray) -> np.ndarray:
    cos_t = 1.0 - 2.0 * rng.random(n)
    phi = 2.0 * np.pi * rng.random(n)
    sin_t = np.sqrt(np.maximum(0.0, 1.0 - cos_t * cos_t))
    out = np.empty((n, 3), dtype=np.float64)
    out[:, 0] = length * sin_t * np.cos(phi)
    out[:, 1] = length * sin_t * np.sin(phi)
    out[:, 2] = length * cos_t
    return out


def plummer(n: int, seed: int):
    """Equal-mass Plummer sphere, N-body units.  Returns fp64 (m[n], x[n,3], v[n,3])."""
    if n < 1:
        raise ValueError("n must be >= 1")
    rng = np.random.default_rng(seed)
    X = MASS_CUT * (1.0 - rng.random(n))  # in (0, 0.999]
    r = 1.0 / np.sqrt(X ** (-2.0 / 3.0) - 1.0)
    x = _isotropic(rng, n, r)

    q = np.empty(n, dtype=np.float64)
    filled = 0
    while filled < n:
        need = n - filled
        cand = rng.random(3 * need + 64)
        y = rng.random(3 * need + 64)
        ok = cand[0.1 * y < cand * cand * (1.0 - cand * cand) ** 3.5][:need]
        q[filled:filled + ok.size] = ok
        filled += ok.size
    speed = q * np.sqrt(2.0) * (1.0 + r * r) ** (-0.25)
    v = _isotropic(rng, n, speed)

    x *= 3.0 * np.pi / 16.0
    v *= np.sqrt(16.0 / (3.0 * np.pi))
    x -= x.mean(axis=0)
    v -= v.mean(axis=0)
    m = np.full(n, 1.0 / n, dtype=np.float64)
    return m, x, v


def plummer_f32(n: int, seed: int):
    """plummer() rounded to fp32 (the paper's device precision).

    Asserts that no two particles share an fp32 position, so that "j != i by
    index" and "r_ij != 0" select the same pairs (reading R6).
    """
    m, x, v = plummer(n, seed)
    m32, x32, v32 = m.astype(np.float32), x.astype(np.float32), v.astype(np.float32)
    key = np.ascontiguousarray(x32).view(np.dtype((np.void, 12))).ravel()
    if np.unique(key).size != n:
        raise AssertionError("duplicate fp32 positions in seeded Plummer input")
    return m32, x32, v32


def config_inputs(name: str):
    c = CONFIGS[name]
    return plummer_f32(c["N"], c["seed"])


def active_block(n: int, n_i: int, seed: int) -> np.ndarray:
    """i-block "drawn uniformly without replacement" (BASELINE.json config 2)."""
    rng = np.random.default_rng([seed, n_i])
    return np.sort(rng.choice(n, size=n_i, replace=False)).astype(np.int32)


def particle_times(n: int, t: float, seed: int) -> np.ndarray:
    """Per-particle last-update times t_j = t - 2^-k, k in {7..12} (block-step mix)."""
    rng = np.random.default_rng([seed, 77])
    k = rng.integers(7, 13, size=n)
    return (t - 2.0 ** (-k.astype(np.float64))).astype(np.float64)


def gaussian_derivatives(n: int, seed: int, rms_a: float = 1.0, rms_j: float = 4.0):
    """Synthetic per-particle a, jerk (fp32) of given rms for predictor stress cases."""
    rng = np.random.default_rng([seed, 78])
    a = (rms_a / np.sqrt(3.0)) * rng.standard_normal((n, 3))
    j = (rms_j / np.sqrt(3.0)) * rng.standard_normal((n, 3))
    return a.astype(np.float32), j.astype(np.float32)
