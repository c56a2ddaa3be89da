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
@pytest.mark.parametrize("variant", [0x00, 0x10, 0x20, 0x40, 0x100])
def test_c1_full_parity_all_kernel_forms(gpu, c_oracle, variant):
    """BASELINE config 1: N=1024, seed 1, eps=1/256, all i active; every i-per-thread count the
    library can launch, and the two-launch form of small blocks."""
    m, x, v = inputs.config_inputs("C1")
    ref = c_oracle.force(m, x, v, EPS)
    with Ctx(1024) as ctx:
        nb.nbk_set_variant(ctx, variant)
        got = gpu_force(ctx, m, x, v, EPS)
        shape = nb.nbk_last_launch(ctx)
    assert shape["launches"] >= 1 and shape["grid"] >= 1
    if (variant >> 4) & 15:
        assert shape["i_per_thread"] == (variant >> 4) & 15
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


def test_seeded_random_sizes_flags_and_kernel_forms(gpu, c_oracle):
    """300 seeded random cases over n, n_i (around the tile and warp boundaries), eps in {1/256, 0, 0.05},
    with and without jerk / nearest neighbour, every kernel form the library can be pinned to, indexed and
    external i-particles: every one inside the north_star tolerances."""
    rng = np.random.default_rng(20071107)
    sizes = [1, 2, 3, 5, 17, 63, 64, 65, 255, 256, 257, 1000, 1531, 2048, 4097]
    for case in range(300):
        n = int(rng.choice(sizes + [int(rng.integers(1, 6000))]))
        n_i = min(n, int(rng.choice([1, 2, 31, 32, 33, n, max(1, n // 2), int(rng.integers(1, n + 1))])))
        eps = float(rng.choice([EPS, 0.0, 0.05]))
        jerk = bool(rng.integers(0, 2))
        nn = jerk and rng.integers(0, 4) == 0
        flags = (nb.NBK_JERK if jerk else 0) | nb.NBK_POT | (nb.NBK_NN if nn else 0) | (nb.NBK_EPS0 if eps == 0.0 else 0)
        variant = int(rng.choice([0x00, 0x10, 0x20, 0x40, 0x100, 0x110]))
        m, x, v = inputs.plummer_f32(n, int(rng.integers(1, 1000)))
        idx = np.sort(rng.choice(n, size=n_i, replace=False)).astype(np.int32)
        xi = vi = None
        ii = idx
        if not nn and rng.integers(0, 5) == 0:   # external test particles beside the chosen ones
            xi = (x[idx] + np.float32(0.013)).astype(np.float32)
            vi = v[idx].copy()
            ii = np.full(n_i, -1, np.int32)
        what = f"case {case}: n={n} n_i={n_i} eps={eps} jerk={jerk} nn={nn} variant={variant:#x} external={xi is not None}"
        with Ctx(n) as ctx:
            nb.nbk_set_variant(ctx, variant)
            got = gpu_force(ctx, m, x, v, eps, i_index=ii, flags=flags, xi=xi, vi=vi, n_i=n_i)
            if nn:
                gi, gr2 = nb.nbk_get_neighbours(ctx, n_i)
        if n == 1 and xi is None:
            assert not np.any(got[0]) and not np.any(got[2]), what
            continue
        ref = c_oracle.force(m, x, v, eps, i_index=ii, want_jerk=jerk, xi=xi, vi=vi)
        e = errors(got, ref, jerk)
        assert np.all(np.isfinite(got[0])) and np.all(np.isfinite(got[2])), what
        assert e["acc_max"] <= 1e-4 and e["pot_max"] <= 1e-5, f"{what}: {e}"
        if jerk:
            assert e["jerk_p99"] <= 1e-3 and e["jerk_max"] <= 1e-2, f"{what}: {e}"
        if nn:
            ri, rr2 = c_oracle.nearest_neighbour(x, i_index=idx)
            assert np.all(np.abs(gr2 - rr2) <= 4e-6 * rr2 + 1e-12), what


def test_pinned_caller_arrays_take_the_direct_copy_path_same_bits(gpu, c_oracle):
    """Caller arrays in page-locked memory are copied by the DMA engine straight from / into them
    (no staging copy): same bits as with pageable arrays, also with addresses, times, a and jerk given."""
    n, t = 8192, 0.01
    m, x, v = inputs.plummer_f32(n, 6)
    a, k = inputs.gaussian_derivatives(n, 7)
    tj = inputs.particle_times(n, t, 8)
    addr = np.random.default_rng(9).permutation(n).astype(np.int32)
    keep = []

    def pin(arr):
        tt = gpu.from_numpy(np.ascontiguousarray(arr)).pin_memory()
        keep.append(tt)
        return tt.numpy()

    def run(pinned):
        f = pin if pinned else (lambda z: z)
        with Ctx(n) as ctx:
            nb.nbk_set_j_particles(ctx, f(addr), f(tj), f(m), f(x), f(v), f(a), f(k))
            nb.nbk_set_ti(ctx, t)
            nb.nbk_calc_firsthalf(ctx, n, n, None, None, None, np.float32(EPS) ** 2, FULL)
            if pinned:
                out = (pin(np.empty((n, 3), np.float32)), pin(np.empty((n, 3), np.float32)), pin(np.empty(n, np.float32)))
                got = nb.nbk_calc_lasthalf(ctx, n, out=out)
                assert got[0] is out[0] and got[2] is out[2]
            else:
                got = nb.nbk_calc_lasthalf(ctx, n)
            return tuple(np.array(g) for g in got)

    plain, direct = run(False), run(True)
    for p, d in zip(plain, direct):
        assert np.array_equal(p, d)
    # against the oracle: particle addr[q] holds input row q
    xs, vs, ms = np.empty_like(x), np.empty_like(v), np.empty_like(m)
    as_, ks, ts = np.empty_like(a), np.empty_like(k), np.empty_like(tj)
    xs[addr], vs[addr], ms[addr], as_[addr], ks[addr], ts[addr] = x, v, m, a, k, tj
    xp, vp = c_oracle.predict(t, ts, xs, vs, as_, ks)
    ref = c_oracle.force(ms, xp.astype(np.float32), vp.astype(np.float32), EPS)
    assert_parity(direct, ref, what="pinned direct path")
    with pytest.raises(ValueError):
        with Ctx(64) as ctx:
            gpu_force(ctx, m[:64], x[:64], v[:64], EPS)
            nb.nbk_calc_lasthalf(ctx, 64, out=(np.empty((64, 3)), np.empty((64, 3), np.float32), np.empty(64, np.float32)))
