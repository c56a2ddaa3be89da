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
