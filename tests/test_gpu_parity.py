"""GPU parity: the CUDA path (through the C ABI, via the thin binding) against the fp64 oracle,
element by element on the same seeded inputs.  Tolerances: tests/parity.py (BASELINE.json).

Run on the B200 box:  python -m pytest tests -m gpu -x -q
"""
import numpy as np
import pytest

from paper_0707_0438_b200 import binding as nb
from paper_0707_0438_b200 import inputs
from parity import assert_parity, errors

pytestmark = pytest.mark.gpu

EPS = inputs.EPS_PAPER
FULL = nb.NBK_JERK | nb.NBK_POT


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu tests have no fallback")
    nb.load()
    return torch


class Ctx:
    def __init__(self, n_max, ni_max=None):
        self.h = nb.nbk_open(0, n_max, ni_max or n_max)

    def __enter__(self):
        return self.h

    def __exit__(self, *a):
        nb.nbk_close(self.h)


def gpu_force(ctx, m, x, v, eps, i_index=None, flags=FULL, xi=None, vi=None, n_i=None, load=True):
    n = m.shape[0]
    if load:
        nb.nbk_set_j_particles(ctx, None, None, m, x, v)
        nb.nbk_set_ti(ctx, 0.0)
    if n_i is None:
        n_i = n if i_index is None else len(i_index)
    nb.nbk_calc_firsthalf(ctx, n, n_i, i_index, xi, vi, np.float32(eps) ** 2, flags)
    return nb.nbk_calc_lasthalf(ctx, n_i)


# ----------------------------------------------------------------------------- config 1
@pytest.mark.parametrize("variant", [0x00, 0x01, 0x10, 0x11, 0x20, 0x21, 0x40, 0x41])
def test_c1_full_parity_all_kernel_forms(gpu, c_oracle, variant):
    """BASELINE config 1: N=1024, seed 1, eps=1/256, all i active; every inner-loop form
    (packed f32x2 / scalar) and every i-per-thread count the library can launch."""
    m, x, v = inputs.config_inputs("C1")
    ref = c_oracle.force(m, x, v, EPS)
    with Ctx(1024) as ctx:
        nb.nbk_set_variant(ctx, variant)
        got = gpu_force(ctx, m, x, v, EPS)
        shape = nb.nbk_last_launch(ctx)
    assert shape["launches"] >= 1 and shape["grid"] >= 1
    if variant >> 4:
        assert shape["i_per_thread"] == variant >> 4
    assert_parity(got, ref, what=f"C1 variant {variant:#x}")


@pytest.mark.parametrize("n,n_i", [(1, 1), (2, 2), (3, 1), (255, 255), (257, 100), (1000, 37),
                                   (1531, 1531), (4099, 513), (5000, 4999)])
def test_ragged_sizes(gpu, c_oracle, n, n_i):
    """Sizes that are not multiples of the j-tile (256) or the i-tile: ragged tails on both axes."""
    m, x, v = inputs.plummer_f32(n, seed=100 + n)
    idx = inputs.active_block(n, n_i, seed=7)
    ref = c_oracle.force(m, x, v, EPS, i_index=idx)
    with Ctx(n) as ctx:
        got = gpu_force(ctx, m, x, v, EPS, i_index=idx)
    if n == 1:
        assert np.all(got[0] == 0) and np.all(got[1] == 0) and abs(got[2][0]) < 1e-6
        return
    assert_parity(got, ref, what=f"n={n} n_i={n_i}")


def test_empty_inputs(gpu):
    m, x, v = inputs.plummer_f32(64, seed=3)
    with Ctx(64) as ctx:
        nb.nbk_set_j_particles(ctx, None, None, m, x, v)
        nb.nbk_set_ti(ctx, 0.0)
        nb.nbk_calc_firsthalf(ctx, 64, 0, np.zeros(0, np.int32), None, None, EPS ** 2, FULL)
        acc, jrk, pot = nb.nbk_calc_lasthalf(ctx, 0)
        assert acc.shape == (0, 3) and pot.shape == (0,)
        # n_j = 0: an external particle feels nothing
        xi = np.array([[0.1, 0.2, 0.3]], np.float32)
        nb.nbk_calc_firsthalf(ctx, 0, 1, np.array([-1], np.int32), xi, None, EPS ** 2, FULL)
        acc, jrk, pot = nb.nbk_calc_lasthalf(ctx, 1)
        assert np.all(acc == 0) and np.all(jrk == 0) and np.all(pot == 0)


def test_bad_calls_are_refused(gpu):
    m, x, v = inputs.plummer_f32(64, seed=3)
    with Ctx(64, 32) as ctx:
        nb.nbk_set_j_particles(ctx, None, None, m, x, v)
        with pytest.raises(nb.NbkError) as e:
            nb.nbk_calc_firsthalf(ctx, 64, 33, np.arange(33, dtype=np.int32), None, None, 0.0, FULL)
        assert e.value.status == nb.NBK_ERANGE
        with pytest.raises(nb.NbkError) as e:
            nb.nbk_calc_firsthalf(ctx, 64, 2, np.array([0, 64], np.int32), None, None, 0.0, FULL)
        assert e.value.status == nb.NBK_ERANGE
        with pytest.raises(nb.NbkError) as e:
            nb.nbk_calc_lasthalf(ctx, 5)
        assert e.value.status == nb.NBK_ESTATE
        with pytest.raises(nb.NbkError) as e:
            nb.nbk_set_j_particles(ctx, np.array([64], np.int32), None, m[:1], x[:1], v[:1])
        assert e.value.status == nb.NBK_ERANGE
