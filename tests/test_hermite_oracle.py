"""Pins for oracle/hermite_oracle.py (fp64 Hermite block-step integrator; readings R8, R15).

Closed forms and invariants only: quintic trajectories (corrector coefficients),
exponential acceleration history (Aarseth formula), Kepler orbit (whole scheme),
4th-order convergence, block-time commensurability.
"""
import numpy as np
import pytest

from oracle import hermite_oracle as ho
from oracle import nbody_oracle as no
from paper_0707_0438_b200 import inputs


def test_corrector_exact_on_quintic_trajectory():
    rng = np.random.default_rng(1)
    n = 9
    c = rng.standard_normal((6, n, 3))  # x(t) = sum_k c_k t^k
    fact = [1, 1, 2, 6, 24, 120]

    def deriv(order, t):
        out = np.zeros((n, 3))
        for k in range(order, 6):
            out += c[k] * (fact[k] / fact[k - order]) * t ** (k - order)
        return out

    t0 = 0.3
    dt = np.full(n, 0.25)
    t1 = t0 + 0.25
    x0, v0, a0, j0 = (deriv(k, t0) for k in range(4))
    a1, j1 = deriv(2, t1), deriv(3, t1)
    xp, vp = no.predict(t1, np.full(n, t0), x0, v0, a0, j0)
    x1, v1, a2e, a3 = ho.correct(xp, vp, a0, j0, a1, j1, dt)
    np.testing.assert_allclose(x1, deriv(0, t1), rtol=1e-12, atol=1e-13)
    np.testing.assert_allclose(v1, deriv(1, t1), rtol=1e-12, atol=1e-13)
    np.testing.assert_allclose(a2e, deriv(4, t1), rtol=1e-10, atol=1e-10)  # a^(2) at the END of the step
    np.testing.assert_allclose(a3, deriv(5, t1), rtol=1e-9, atol=1e-9)


def test_aarseth_step_closed_form():
    lam, eta = 3.0, 0.01
    c = np.array([[0.3, -0.4, 1.2]])
    dt = ho.aarseth_dt(c, lam * c, lam ** 2 * c, lam ** 3 * c, eta)
    np.testing.assert_allclose(dt, np.sqrt(eta) / lam, rtol=1e-14)


def test_block_rule():
    dt = np.array([1 / 64, 1 / 64, 1 / 64, 1 / 64, 1 / 16])
    want = np.array([1 / 500, 1 / 40, 1 / 70, 1.0, 1.0])
    # t_new = 3/64 is an odd multiple of 1/64: no doubling allowed
    out = ho.next_block_dt(dt, want, 3 / 64, 1 / 16)
    np.testing.assert_array_equal(out, [1 / 512, 1 / 64, 1 / 128, 1 / 64, 1 / 16])
    # t_new = 4/64: doubling allowed, once, and never beyond dt_max
    out = ho.next_block_dt(dt, want, 4 / 64, 1 / 16)
    np.testing.assert_array_equal(out, [1 / 512, 1 / 64, 1 / 128, 1 / 32, 1 / 16])  # 1/40 < 2/64: keeps
    np.testing.assert_array_equal(ho.pow2_floor([0.3, 0.25, 1 / 100]), [0.25, 0.25, 1 / 128])


def _kepler(e=0.5):
    """Two bodies, total mass 1, period exactly 1 (a = (2 pi)^(-2/3)); start at pericentre."""
    a = (2 * np.pi) ** (-2.0 / 3.0)
    m = np.array([0.6, 0.4])
    rp = a * (1 - e)
    vp = np.sqrt((1 + e) / (a * (1 - e)))
    x = np.array([[-m[1] * rp, 0, 0], [m[0] * rp, 0, 0]])
    v = np.array([[0, -m[1] * vp, 0], [0, m[0] * vp, 0]])
    return m, x, v


def test_kepler_orbit_closes_and_conserves_energy():
    m, x, v = _kepler()
    e0 = no.energy(m, x, v, 0.0)
    assert e0 == pytest.approx(-0.5 * m[0] * m[1] / (2 * np.pi) ** (-2.0 / 3.0), rel=1e-13)
    out = ho.evolve(m, x, v, 0.0, 1.0, eta=0.01, dt_max=1 / 16)
    assert np.all(out["t"] == 1.0)
    e1 = no.energy(m, out["x"], out["v"], 0.0)
    err = abs(no.relative_energy_error(e0, e1))
    assert err < 2e-6
    assert np.abs(out["x"] - x).max() < 1e-4  # one full period: back at the start
    assert np.abs(out["v"] - v).max() < 1e-3
    # eta/4 -> Aarseth steps halve -> error falls by about 2^4
    out4 = ho.evolve(m, x, v, 0.0, 1.0, eta=0.0025, dt_max=1 / 16)
    err4 = abs(no.relative_energy_error(e0, no.energy(m, out4["x"], out4["v"], 0.0)))
    assert err4 < err / 6.0
    assert out4["particle_steps"] > 1.5 * out["particle_steps"]


def test_fourth_order_convergence():
    """Halving a shared constant step divides the error by ~2^4."""
    m, x, v = _kepler(e=0.3)
    errs = []
    for dt in (1 / 128, 1 / 256, 1 / 512):
        out = ho.evolve(m, x, v, 0.0, 1.0, fixed_dt=dt)
        errs.append(np.abs(out["x"] - x).max())
    r1, r2 = errs[0] / errs[1], errs[1] / errs[2]
    assert 12.0 < r1 < 20.0 and 12.0 < r2 < 20.0, (errs, r1, r2)


def test_block_steps_commensurate_and_energy_small_plummer():
    m, x, v = inputs.plummer(128, 21)
    eps = inputs.EPS_PAPER
    e0 = no.energy(m, x, v, eps)
    out = ho.evolve(m, x, v, eps, 0.125, eta=0.01, dt_max=1 / 16)
    assert np.all(out["t"] == 0.125)
    k = np.log2(out["dt"])
    assert np.all(k == np.round(k)) and np.all(out["dt"] <= 1 / 16)
    assert np.all(np.mod(out["t"], out["dt"]) == 0.0)
    assert out["particle_steps"] > out["block_steps"] > 2
    e1 = no.energy(m, out["x"], out["v"], eps)
    assert abs(no.relative_energy_error(e0, e1)) < 1e-7


def test_initial_dt_hand_values():
    """Start-up step, reading R15 (PAPER.md L68, L74 print no formula): dt_0 = largest 2^-k <=
    min((eta / 4) |a| / |j|, dt_max).  Expected values worked by hand, not by the formula's code:
      |a| = 1, |j| = 8,  eta = 0.01: (0.01/4)/8 = 3.125e-4;  2^-12 = 2.44e-4 <= 3.125e-4 < 2^-11 = 4.88e-4
      |a| = 3, |j| = 0.5 (3-4-5 vectors): 0.0025 * 6 = 0.015;  2^-7 = 0.0078 <= 0.015 < 2^-6 = 0.0156
      |a| = 2, |j| = 0.01: 0.0025 * 200 = 0.5 > dt_max = 1/16  -> dt_max
      |j| = 0 -> dt_max;   |a| = 0 -> dt_max (a zero step is no step)
      exact power of two: |a| = 1, |j| = 0.64, eta = 0.01: 0.0025/0.64 = 2^-8 exactly -> 2^-8
    With eta/2 the first row gives 2^-11, with eta 2^-10: the pin tells the readings apart."""
    a = np.array([[1.0, 0, 0], [0, 1.8, 2.4], [0, 0, -2.0], [0.3, 0.1, 0.2], [0, 0, 0], [0, -1.0, 0]])
    j = np.array([[0, 8.0, 0], [0.3, 0, -0.4], [0.01, 0, 0], [0, 0, 0], [1.0, 2.0, 3.0], [0.64, 0, 0]])
    dt = ho.initial_dt(a, j, 0.01, 1 / 16)
    np.testing.assert_array_equal(dt, [2.0 ** -12, 2.0 ** -7, 1 / 16, 1 / 16, 1 / 16, 2.0 ** -8])
    # eta scales the step linearly: 4 eta -> two levels coarser, capped by dt_max
    dt4 = ho.initial_dt(a, j, 0.04, 1 / 16)
    np.testing.assert_array_equal(dt4, [2.0 ** -10, 2.0 ** -5, 1 / 16, 1 / 16, 1 / 16, 2.0 ** -6])
    # dt_max itself is not rounded by this function's caller contract: a power of two comes back as is
    np.testing.assert_array_equal(ho.initial_dt(a[:1], j[:1], 0.01, 2.0 ** -14), [2.0 ** -14])


def test_evolve_takes_the_start_up_step_first():
    """The integrator's first block time is the smallest start-up step (R15): circular two-body orbit
    with |a| / |j| known in closed form.  Bodies m1 = m2 = 1/2 at separation d = 1, eps = 0: each feels
    |a| = m / d^2 = 1/2; relative speed of a circular orbit v = sqrt(M/d) = 1, so |j| = m v / d^3 = 1/2
    (r.w = 0 on a circle).  (eta/4) |a|/|j| = 0.0025 -> 2^-9 = 0.00195 (2^-8 = 0.0039 is too large)."""
    m = np.array([0.5, 0.5])
    x = np.array([[-0.5, 0, 0], [0.5, 0, 0]])
    v = np.array([[0, -0.5, 0], [0, 0.5, 0]])
    seen = []

    def spy(m_, x_, v_, eps_, i_index=None):
        seen.append(None if i_index is None else len(i_index))
        return no.force(m_, x_, v_, eps_, i_index=i_index)

    out = ho.evolve(m, x, v, 0.0, 2.0 ** -9, eta=0.01, dt_max=2.0 ** -9, force_fn=spy)
    assert out["block_steps"] == 1 and np.all(out["t"] == 2.0 ** -9)
    a, jk, _ = no.force(m, x, v, 0.0)
    np.testing.assert_allclose(np.linalg.norm(a, axis=1), 0.5, rtol=1e-14)
    np.testing.assert_allclose(np.linalg.norm(jk, axis=1), 0.5, rtol=1e-14)
    np.testing.assert_array_equal(ho.initial_dt(a, jk, 0.01, 1 / 16), [2.0 ** -9, 2.0 ** -9])
    # to t = 1/16 with dt_max = 1/16: 32 steps of 2^-9 if the step never changed; the Aarseth step of a
    # circular orbit is sqrt(eta) / omega = 0.1 > dt_max, so the step doubles whenever the block rule allows
    # and may double only at times that are multiples of the doubled step.  By hand: 2^-9 to t = 2^-9 (odd:
    # no doubling), 2^-9 to 2^-8 (doubles), 2^-8 to 2^-7, 2^-7 to 2^-6, 2^-6 to 2^-5, 2^-5 to 2^-4: 6 steps.
    # (A start-up step of 2^-8 would give 5, of 2^-7 4.)
    out = ho.evolve(m, x, v, 0.0, 1 / 16, eta=0.01, dt_max=1 / 16)
    assert out["block_steps"] == 6 and out["particle_steps"] == 12
    np.testing.assert_array_equal(out["dt"], [2.0 ** -4, 2.0 ** -4])   # t = 2^-4 allows one more doubling
