"""ORACLE -- test infrastructure, not product code.

Plain, slow, fp64 CPU statement of what the hot path of arxiv 0707.0438
("kirin", Belleman, Bedorf & Portegies Zwart 2007) computes.  Only `tests/`,
`__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference`
legs may import this package.  It shares no code with
`paper_0707_0438_b200/` (the CUDA path) and imports nothing from it.

What is computed (citations are PAPER.md lines):

  direct summation of acceleration, jerk and potential for each active
  i-particle over all j-particles (L68 "The acceleration, its time derivative
  (jerk) and potential are computed by direct summation"; Eq. 1; inputs
  m, x, v / outputs a, jerk, pot L80-L83), with Plummer softening eps
  (L126, L132), self pair excluded (L96; j != i in Eq. 1), and for eps = 0
  zero-distance pairs skipped (L130-L132).

  the Hermite predictor for the j-particles (L68 "a predictor step that
  predicts a particle's position and velocity"; L428 GPU_set_ti).

With r = x_j - x_i, w = v_j - v_i, s = r.r + eps^2, G = 1:

    a_i    =  sum_{j != i}  m_j r s^(-3/2)
    jerk_i =  sum_{j != i}  m_j [ w s^(-3/2) - 3 (r.w) r s^(-5/2) ]
    pot_i  = -sum_{j != i}  m_j s^(-1/2)

Readings of silent / garbled passages (R1..R8):
  R1  Eq. 1 prints (r_i - r_j): taken as attractive, r = x_j - x_i.
  R2  softening is Plummer: r^2 -> r^2 + eps^2 in all three sums.
  R3  jerk (formula not printed, L68 cites Makino & Aarseth 1992) is the exact
      time derivative of the softened a along straight-line motion.
  R4  potential is per unit mass, negative, self term excluded (L96).
  R6  self pair recognised by INDEX; for eps = 0 additionally s == 0 skipped.
  R8  predictor is the Taylor series through the jerk:
      x_p = x + v dt + a dt^2/2 + jerk dt^3/6,  v_p = v + a dt + jerk dt^2/2.

Pins (tests/test_oracle_pins.py): two-body closed form, momentum sums, zero
force at the centre of symmetric lattices, jerk vs central finite difference
of a, a = -grad(pot) by finite difference, translation / boost / scaling
invariances, 50-digit mpmath brute force on N <= 48 (with duplicated positions
and eps = 0), predictor exactness on cubic trajectories.  No function here is
"parity unpinned".
"""
from __future__ import annotations

import numpy as np

_CHUNK_ELEMS = 1 << 22  # (i-chunk x N) fp64 temporaries per array


def _as64(a, shape_tail=()):
    a = np.asarray(a, dtype=np.float64)
    if shape_tail and a.shape[1:] != shape_tail:
        raise ValueError("bad shape")
    return a


def force(m, x, v, eps, i_index=None, want_jerk=True, xi=None, vi=None):
    """acc[n_i,3], jerk[n_i,3], pot[n_i] in fp64 (definition above).

    i_index[k] >= 0 : i-particle k is j-particle i_index[k]; that j is excluded
                      from its sums.  -1: external test particle (needs xi, vi).
    xi, vi          : optional explicit i-state overriding x[i_index], v[i_index].
    """
    m = _as64(m)
    x = _as64(x, (3,))
    n = m.shape[0]
    v = _as64(v, (3,)) if v is not None else np.zeros((n, 3))
    if i_index is None:
        i_index = np.arange(n)
    i_index = np.asarray(i_index, dtype=np.int64)
    n_i = i_index.shape[0]
    safe = np.where(i_index >= 0, i_index, 0)
    xi = x[safe] if xi is None else _as64(xi, (3,))
    vi = v[safe] if vi is None else _as64(vi, (3,))
    eps2 = float(eps) * float(eps)

    acc = np.zeros((n_i, 3))
    jrk = np.zeros((n_i, 3))
    pot = np.zeros(n_i)
    jj = np.arange(n)
    chunk = max(1, _CHUNK_ELEMS // max(n, 1))
    for lo in range(0, n_i, chunk):
        hi = min(n_i, lo + chunk)
        r = x[None, :, :] - xi[lo:hi, None, :]
        s = np.einsum("ijk,ijk->ij", r, r) + eps2
        skip = jj[None, :] == i_index[lo:hi, None]
        if eps2 == 0.0:
            skip |= s == 0.0
        s = np.where(skip, 1.0, s)
        mj = np.where(skip, 0.0, m[None, :])
        s_m12 = 1.0 / np.sqrt(s)
        s_m32 = s_m12 / s
        pot[lo:hi] = -np.sum(mj * s_m12, axis=1)
        acc[lo:hi] = np.sum((mj * s_m32)[:, :, None] * r, axis=1)
        if want_jerk:
            w = v[None, :, :] - vi[lo:hi, None, :]
            rw = np.einsum("ijk,ijk->ij", r, w)
            s_m52 = s_m32 / s
            jrk[lo:hi] = np.sum((mj * s_m32)[:, :, None] * w, axis=1) - 3.0 * np.sum(
                (mj * rw * s_m52)[:, :, None] * r, axis=1
            )
    return acc, jrk, pot


def nearest_neighbour(x, i_index=None, xi=None):
    """Index of, and squared distance to, the nearest j-particle of each i-particle (PAPER.md L128:
    "comparing the distance between each particle and all other particles ... maintain the particle
    with the minimum distance"), own entry excluded by index, fp64.  Reading R20: ties go to the
    lowest index; a particle with no other j gets index -1 and distance inf."""
    x = _as64(x, (3,))
    n = x.shape[0]
    if i_index is None:
        i_index = np.arange(n)
    idx = np.asarray(i_index, dtype=np.int64)
    xs = x[np.maximum(idx, 0)] if xi is None else _as64(xi, (3,))
    nn = np.full(idx.shape[0], -1, dtype=np.int64)
    r2min = np.full(idx.shape[0], np.inf)
    for k in range(idx.shape[0]):          # plain loop over i: one pass over j each
        d = x - xs[k]
        r2 = np.einsum("ij,ij->i", d, d)
        if idx[k] >= 0:
            r2[idx[k]] = np.inf
        if n > 0 and np.isfinite(r2).any():
            j = int(np.argmin(r2))         # argmin returns the first (lowest-index) minimum
            nn[k], r2min[k] = j, r2[j]
    return nn, r2min


def predict(t, tj, x, v, a, jerk):
    """Hermite predictor, R8: Taylor series through the jerk, fp64."""
    dt = (float(t) - _as64(tj))[:, None]
    x, v, a, jerk = _as64(x, (3,)), _as64(v, (3,)), _as64(a, (3,)), _as64(jerk, (3,))
    xp = x + v * dt + a * (dt * dt / 2.0) + jerk * (dt * dt * dt / 6.0)
    vp = v + a * dt + jerk * (dt * dt / 2.0)
    return xp, vp


def energy(m, x, v, eps):
    """Total energy E = sum 1/2 m v^2 + 1/2 sum m_i pot_i (softened), for PAPER.md Eq. 2 L142."""
    m = _as64(m)
    v = _as64(v, (3,))
    _, _, pot = force(m, x, v, eps, want_jerk=False)
    kin = 0.5 * np.sum(m * np.einsum("ij,ij->i", v, v))
    return kin + 0.5 * np.sum(m * pot)


def relative_energy_error(e_start, e_end):
    """PAPER.md Eq. 2 (L142): dE/E = (E_start - E_end) / E_start."""
    return (e_start - e_end) / e_start


def flops_per_second(k, n_i, n_j, seconds):
    """PAPER.md Eq. 3 (L178): P = k N^2 / t, k = 38 force only, k = 60 force+pot+jerk (L180)."""
    return k * float(n_i) * float(n_j) / seconds
