"""Seeded workload generator: determinism, units, structure."""
import numpy as np

from paper_0707_0438_b200 import inputs


def test_deterministic_and_distinct_seeds():
    a = inputs.plummer(1000, 3)
    b = inputs.plummer(1000, 3)
    c = inputs.plummer(1000, 4)
    for p, q in zip(a, b):
        assert np.array_equal(p, q)
    assert not np.array_equal(a[1], c[1])


def test_nbody_units_and_structure():
    m, x, v = inputs.plummer(20000, 1)
    assert m.sum() == 1.0 or abs(m.sum() - 1.0) < 1e-12
    assert np.abs((m[:, None] * x).sum(0)).max() < 1e-12
    assert np.abs((m[:, None] * v).sum(0)).max() < 1e-12
    r = np.sqrt((x ** 2).sum(1))
    assert abs(np.median(r) - 0.7686) < 0.02           # half-mass radius of the N-body-unit Plummer model
    assert r.max() < 23.5                              # 99.9 % mass cut at 38.7 a = 22.8 length units
    kin = 0.5 * np.sum(m * (v ** 2).sum(1))
    assert abs(kin - 0.25) < 0.01                      # T = 1/4 (virial, E = -1/4)
    b = 3 * np.pi / 16
    vesc2 = 2.0 / np.sqrt(r * r + b * b)
    assert np.all((v ** 2).sum(1) <= vesc2 * 1.02)     # bound: below the local escape speed (COM shift ~1e-2)


def test_fp32_cast_has_no_duplicates_and_blocks_are_unique():
    m, x, v = inputs.plummer_f32(4096, 2)
    assert m.dtype == x.dtype == v.dtype == np.float32
    for n_i in (1, 32, 256, 2048, 4096):
        idx = inputs.active_block(4096, n_i, 2)
        assert idx.dtype == np.int32 and idx.size == n_i and np.unique(idx).size == n_i
        assert idx.min() >= 0 and idx.max() < 4096
    tj = inputs.particle_times(100, 0.01, 2)
    assert np.all(tj < 0.01) and np.all(0.01 - tj <= 2.0 ** -7)
