"""ORACLE -- test infrastructure, not product code.

fp64 statement of the host integrator that drives the force path: "4th order
predictor-corrector Hermite integrator with block time-steps" (PAPER.md L13,
L68, L74; scheme of Makino & Aarseth 1992 and McMillan & Aarseth 1993, which
the paper cites but does not print).  Forces come from oracle/nbody_oracle.py.
Pure numpy, O(N^2) per block step: small N only.

The paper prints none of the formulas, so every one below is a reading
(R15), written step by step in the order the scheme is run:

  predictor   x_p = x + v dt + a dt^2/2 + j dt^3/6 ; v_p = v + a dt + j dt^2/2   (R8)
  force       a1, j1 at (x_p, v_p) of ALL particles at the block time          (R7)
  corrector   a2 = [-6 (a0 - a1) - dt (4 j0 + 2 j1)] / dt^2
              a3 = [12 (a0 - a1) + 6 dt (j0 + j1)] / dt^3
              x1 = x_p + a2 dt^4/24 + a3 dt^5/120 ; v1 = v_p + a2 dt^3/6 + a3 dt^4/24
  time step   a2' = a2 + a3 dt  (a2 at the end of the step)
              dt_A = sqrt( eta (|a1| |a2'| + |j1|^2) / (|j1| |a3| + |a2'|^2) )   (Aarseth)
  block rule  steps are 2^-k <= dt_max; a step may halve repeatedly, may double only
              if dt_A >= 2 dt, 2 dt <= dt_max and the new time is a multiple of 2 dt
  first step  dt_0 = largest 2^-k <= min(eta_s |a| / |j|, dt_max), eta_s = eta/4

Pins (tests/test_hermite_oracle.py): Kepler two-body orbit (eps = 0) closes
after one period and conserves energy; global error falls ~16x when eta-driven
steps halve ("a decrease in the energy error of a factor of
2^4"); corrector reproduces a quintic-in-time trajectory exactly; block times
stay commensurate.
"""
from __future__ import annotations

import math

import numpy as np

from . import nbody_oracle as _force


def _norm(a):
    return np.sqrt(np.einsum("ij,ij->i", a, a))


def pow2_floor(dt):
    """Largest 2^-k (k integer, any sign) that is <= dt, elementwise."""
    dt = np.asarray(dt, dtype=np.float64)
    return np.exp2(np.floor(np.log2(dt)))


def initial_dt(a, j, eta, dt_max):
    na, nj = _norm(a), _norm(j)
    with np.errstate(divide="ignore", invalid="ignore"):
        raw = np.where(nj > 0.0, (eta / 4.0) * na / nj, dt_max)
    raw = np.where(raw > 0.0, raw, dt_max)
    return pow2_floor(np.minimum(raw, dt_max))


def correct(xp, vp, a0, j0, a1, j1, dt):
    """Hermite corrector; returns x1, v1, a2' (=a2 + a3 dt), a3."""
    dt = np.asarray(dt, dtype=np.float64)[:, None]
    a2 = (-6.0 * (a0 - a1) - dt * (4.0 * j0 + 2.0 * j1)) / (dt * dt)
    a3 = (12.0 * (a0 - a1) + 6.0 * dt * (j0 + j1)) / (dt * dt * dt)
    x1 = xp + a2 * (dt ** 4 / 24.0) + a3 * (dt ** 5 / 120.0)
    v1 = vp + a2 * (dt ** 3 / 6.0) + a3 * (dt ** 4 / 24.0)
    return x1, v1, a2 + a3 * dt, a3


def aarseth_dt(a1, j1, a2e, a3, eta):
    na, nj, n2, n3 = _norm(a1), _norm(j1), _norm(a2e), _norm(a3)
    num = na * n2 + nj * nj
    den = nj * n3 + n2 * n2
    with np.errstate(divide="ignore", invalid="ignore"):
        dt = np.sqrt(eta * num / den)
    return np.where((den > 0.0) & np.isfinite(dt) & (dt > 0.0), dt, np.inf)


def next_block_dt(dt_old, dt_want, t_new, dt_max):
    """Block rule: halve until <= dt_want; double at most once, only on even block boundaries."""
    out = np.array(dt_old, dtype=np.float64, copy=True)
    want = np.minimum(dt_want, dt_max)
    for k in range(out.shape[0]):
        d = out[k]
        if want[k] < d:
            while want[k] < d:
                d *= 0.5
        elif want[k] >= 2.0 * d and 2.0 * d <= dt_max and math.fmod(t_new, 2.0 * d) == 0.0:
            d *= 2.0
        out[k] = d
    return out


def evolve(m, x, v, eps, t_end, eta=0.01, dt_max=1.0 / 16.0, fixed_dt=None, force_fn=None):
    """Integrate from t = 0 to t_end (a multiple of dt_max, or of fixed_dt).

    fixed_dt: if given, every particle takes that constant step (shared-step
    Hermite; used by the convergence-order pin).  Returns a dict with the final
    fp64 state and counters.
    """
    f = force_fn or _force.force
    m = np.asarray(m, dtype=np.float64)
    x = np.array(x, dtype=np.float64)
    v = np.array(v, dtype=np.float64)
    n = m.shape[0]
    a, j, _ = f(m, x, v, eps)
    t = np.zeros(n)
    dt = np.full(n, fixed_dt) if fixed_dt is not None else initial_dt(a, j, eta, dt_max)
    steps = 0
    particle_steps = 0
    while True:
        t_new = float(np.min(t + dt))
        if t_new > t_end:
            break
        act = np.nonzero(t + dt == t_new)[0]
        xp, vp = _force.predict(t_new, t, x, v, a, j)
        a1, j1, _ = f(m, xp, vp, eps, i_index=act)
        x1, v1, a2e, a3 = correct(xp[act], vp[act], a[act], j[act], a1, j1, dt[act])
        x[act], v[act], a[act], j[act], t[act] = x1, v1, a1, j1, t_new
        if fixed_dt is None:
            dt[act] = next_block_dt(dt[act], aarseth_dt(a1, j1, a2e, a3, eta), t_new, dt_max)
        steps += 1
        particle_steps += act.size
        if t_new == t_end and np.all(t == t_end):
            break
    return dict(x=x, v=v, a=a, jerk=j, t=t, dt=dt, block_steps=steps, particle_steps=particle_steps)
