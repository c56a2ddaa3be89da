"""GPU parity at BASELINE.json's configs C2-C5, in the launch shapes bench.py times, plus the
degenerate cases of the method.  Everything goes through the C ABI (via the thin binding); the
expected values come from oracle/ on the same seeded inputs.  Tolerances: tests/parity.py.

Run on the B200 box:  python -m pytest tests -m gpu -x -q
"""
import os

import numpy as np
import pytest

from paper_0707_0438_b200 import binding as nb
from paper_0707_0438_b200 import inputs
from parity import assert_parity, scalar_rel_err, vec_rel_err

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
    def __init__(self, n_max, ni_max=None, stream=0):
        self.h = nb.nbk_open(0, n_max, ni_max or n_max, stream)

    def __enter__(self):
        return self.h

    def __exit__(self, *a):
        nb.nbk_close(self.h)


# ----------------------------------------------------------------------------- config 2
@pytest.fixture(scope="module")
def c2(c_oracle):
    """N=16384, seed 2; per-particle a, jerk = the oracle's force at t_j = 0 rounded to fp32
    (DESIGN.md input recipe: 'seeded a and jerk'); prediction time t = 0.01."""
    m, x, v = inputs.config_inputs("C2")
    a, jk, _ = c_oracle.force(m, x, v, EPS)
    a32, j32 = a.astype(np.float32), jk.astype(np.float32)
    tj = np.zeros(m.shape[0])
    xp, vp = c_oracle.predict(0.01, tj, x, v, a32, j32)
    return dict(m=m, x=x, v=v, a=a32, jerk=j32, tj=tj, t=0.01, xp=xp, vp=vp)


def test_c2_predictor_matches_fp64_oracle(gpu, c2):
    """a3: device prediction vs fp64 oracle: one fp32 rounding of the fp64 result."""
    n = c2["m"].shape[0]
    with Ctx(n) as ctx:
        nb.nbk_set_j_particles(ctx, None, c2["tj"], c2["m"], c2["x"], c2["v"], c2["a"], c2["jerk"])
        nb.nbk_set_ti(ctx, c2["t"])
        nb.nbk_predict(ctx, n)
        gm, gx, gv = nb.nbk_get_predicted(ctx, n)
    assert np.array_equal(gm, c2["m"])
    # the device evaluates the same fp64 polynomial (possibly with FMA contraction) and rounds
    # once: at most 1 ulp of fp32 from the correctly rounded oracle value
    for got, ref in ((gx, c2["xp"]), (gv, c2["vp"])):
        ulp = np.spacing(np.abs(ref).astype(np.float32)).astype(np.float64)
        assert np.all(np.abs(got.astype(np.float64) - ref) <= 1.0 * ulp)
        assert np.mean(got == ref.astype(np.float32)) > 0.99


@pytest.mark.parametrize("n_i", [1, 32, 256, 2048, 16384])
def test_c2_block_step_sweep(gpu, c_oracle, c2, n_i):
    """a4-a7 for i-blocks 'drawn uniformly without replacement' after device prediction:
    (ii) kernel isolated: oracle on the GPU-predicted fp32 state; (iii) end to end: oracle
    prediction + oracle force in fp64."""
    n = c2["m"].shape[0]
    idx = inputs.active_block(n, n_i, seed=2)
    with Ctx(n) as ctx:
        nb.nbk_set_j_particles(ctx, None, c2["tj"], c2["m"], c2["x"], c2["v"], c2["a"], c2["jerk"])
        nb.nbk_set_ti(ctx, c2["t"])
        nb.nbk_calc_firsthalf(ctx, n, n_i, idx, None, None, np.float32(EPS) ** 2, FULL)
        got = nb.nbk_calc_lasthalf(ctx, n_i)
        shape = nb.nbk_last_launch(ctx)
        gm, gx, gv = nb.nbk_get_predicted(ctx, n)
    assert shape["launches"] == (1 if n_i <= 32 else 2) and shape["grid"] >= min(128, shape["sms"])
    ref_kernel = c_oracle.force(gm, gx, gv, EPS, i_index=idx)
    assert_parity(got, ref_kernel, what=f"C2 n_i={n_i} kernel-only")
    ref_e2e = c_oracle.force(c2["m"], c2["xp"], c2["vp"], EPS, i_index=idx)
    assert_parity(got, ref_e2e, what=f"C2 n_i={n_i} end-to-end")


def test_c2_stress_mixed_times_gaussian_derivatives(gpu, c_oracle):
    """Predictor stress: per-particle t_j = t - 2^-k (k in 7..12), Gaussian a, jerk of matched rms."""
    m, x, v = inputs.config_inputs("C2")
    n = m.shape[0]
    t = 0.01
    tj = inputs.particle_times(n, t, seed=2)
    a, jk = inputs.gaussian_derivatives(n, seed=2)
    xp, vp = c_oracle.predict(t, tj, x, v, a, jk)
    idx = inputs.active_block(n, 2048, seed=3)
    with Ctx(n) as ctx:
        nb.nbk_set_j_particles(ctx, None, tj, m, x, v, a, jk)
        nb.nbk_set_ti(ctx, t)
        nb.nbk_calc_firsthalf(ctx, n, 2048, idx, None, None, np.float32(EPS) ** 2, FULL)
        got = nb.nbk_calc_lasthalf(ctx, 2048)
        gm, gx, gv = nb.nbk_get_predicted(ctx, n)
    ulp = np.spacing(np.abs(xp).astype(np.float32)).astype(np.float64)
    assert np.all(np.abs(gx.astype(np.float64) - xp) <= ulp)
    assert_parity(got, c_oracle.force(m, xp, vp, EPS, i_index=idx), what="C2 stress")


# ----------------------------------------------------------------------------- config 3
@pytest.mark.parametrize("eps", [EPS, 0.0])
def test_c3_headline_full_parity(gpu, c_oracle, eps):
    """N=131072 seed 3, all i active, eps=1/256 and eps=0 (self pair excluded): every particle
    against the C oracle (1.7e10 pairs), in the launch shape bench.py times."""
    m, x, v = inputs.config_inputs("C3")
    n = m.shape[0]
    with Ctx(n) as ctx:
        nb.nbk_set_j_particles(ctx, None, None, m, x, v)
        nb.nbk_set_ti(ctx, 0.0)
        nb.nbk_calc_firsthalf(ctx, n, n, None, None, None, np.float32(eps) ** 2, FULL)
        got = nb.nbk_calc_lasthalf(ctx, n)
        shape = nb.nbk_last_launch(ctx)
    assert shape["grid"] == shape["sms"] and shape["i_per_thread"] == 4
    ref = c_oracle.force(m, x, v, eps)
    e = assert_parity(got, ref, what=f"C3 eps={eps}")
    # momentum: sum m a = 0 for the exact sums; the GPU's is bounded by its per-particle error
    p = np.abs((m[:, None].astype(np.float64) * got[0]).sum(axis=0)).max()
    assert p < 1e-6, p
    print(f"C3 eps={eps}: {e}")


# ----------------------------------------------------------------------------- config 4
def test_c4_million_acc_pot_only_sampled(gpu, c_oracle):
    """N=1048576 seed 4: acc+pot without jerk for all i; oracle on a seeded 1024-particle subset."""
    m, x, v = inputs.config_inputs("C4")
    n = m.shape[0]
    with Ctx(n) as ctx:
        nb.nbk_set_j_particles(ctx, None, None, m, x, None)
        nb.nbk_set_ti(ctx, 0.0)
        nb.nbk_calc_firsthalf(ctx, n, n, None, None, None, np.float32(EPS) ** 2, nb.NBK_POT)
        acc, jrk, pot = nb.nbk_calc_lasthalf(ctx, n)
    assert np.all(jrk == 0.0)
    assert np.all(np.isfinite(acc)) and np.all(np.isfinite(pot)) and np.all(pot < 0.0)
    sub = inputs.active_block(n, 1024, seed=4)
    racc, _, rpot = c_oracle.force(m, x, v, EPS, i_index=sub, want_jerk=False)
    assert_parity((acc[sub], None, pot[sub]), (racc, None, rpot), jerk=False, what="C4 subset")
    # a property that holds at any size: W = 1/2 sum m pot ~ -1/2 for the Plummer model in N-body
    # units (softening and the 99.9 % mass cut move it by a few per cent)
    w = 0.5 * np.sum(m.astype(np.float64) * pot)
    assert -0.52 < w < -0.45, w


# ----------------------------------------------------------------------------- config 5
def _energy(c_oracle, m, x, v, eps):
    _, _, pot = c_oracle.force(m, x, v, eps, want_jerk=False)
    return 0.5 * np.sum(m * np.sum(v * v, axis=1)) + 0.5 * np.sum(m * pot)


def test_c5_hermite_energy_conservation(gpu, c_oracle):
    """N=65536 seed 5 integrated to t=1 with the host Hermite driver (eta=0.01, dt_max=1/16),
    device predictor + force per block step: |dE/E| < 1e-6 (BASELINE.json north_star), energy
    by the fp64 oracle at both ends (Eq. 2)."""
    m, x, v = inputs.plummer(inputs.CONFIGS["C5"]["N"], inputs.CONFIGS["C5"]["seed"])
    n = m.shape[0]
    e0 = _energy(c_oracle, m, x, v, EPS)
    with Ctx(n) as ctx:
        st = nb.nbk_hermite_evolve(ctx, m, x, v, EPS, 1.0, eta=0.01, dt_max=1.0 / 16.0)
    e1 = _energy(c_oracle, m, x, v, EPS)
    de = abs((e0 - e1) / e0)
    print(f"C5: dE/E={de:.3e} block_steps={st['block_steps']} particle_steps={st['particle_steps']} "
          f"wall={st['wall_seconds']:.2f}s gpu_calls={st['gpu_call_seconds']:.2f}s "
          f"interactions={st['interactions']:.3e}")
    assert st["t_reached"] == 1.0
    assert abs(e0 + 0.25) < 0.01
    assert de < 1e-6, de


def test_hermite_small_n_follows_the_fp64_oracle_integrator(gpu):
    """N=256 to t=0.25: the GPU-driven run and oracle/hermite_oracle.py (same scheme, fp64 forces)
    take the same block steps at first and end with nearby states and equal energy drift scale."""
    from oracle import hermite_oracle, nbody_oracle
    m, x, v = inputs.plummer(256, seed=11)
    ref = hermite_oracle.evolve(m, x, v, EPS, 0.25)
    gx, gv = x.copy(), v.copy()
    with Ctx(256) as ctx:
        st = nb.nbk_hermite_evolve(ctx, m, gx, gv, EPS, 0.25)
    assert st["t_reached"] == 0.25
    # fp32 forces perturb step choices slightly: counts agree to a few per cent
    assert abs(st["particle_steps"] - ref["particle_steps"]) <= 0.05 * ref["particle_steps"]
    e0 = nbody_oracle.energy(m, x, v, EPS)
    assert abs((nbody_oracle.energy(m, gx, gv, EPS) - e0) / e0) < 1e-6
    assert abs((nbody_oracle.energy(m, ref["x"], ref["v"], EPS) - e0) / e0) < 1e-6
    # chaotic divergence over 0.25 time units is tiny: positions agree to ~1e-5 typical
    assert np.median(np.linalg.norm(gx - ref["x"], axis=1)) < 1e-4


# ----------------------------------------------------------------------------- degenerate cases
def test_repeat_runs_are_bitwise_identical(gpu):
    """Reading R11: fixed work split and fixed-order reductions => same bits run to run."""
    m, x, v = inputs.plummer_f32(5000, seed=9)
    idx = inputs.active_block(5000, 777, seed=1)
    with Ctx(5000) as ctx:
        nb.nbk_set_j_particles(ctx, None, None, m, x, v)
        nb.nbk_set_ti(ctx, 0.0)
        outs = []
        for _ in range(3):
            nb.nbk_calc_firsthalf(ctx, 5000, 777, idx, None, None, np.float32(EPS) ** 2, FULL)
            outs.append(nb.nbk_calc_lasthalf(ctx, 777))
    for o in outs[1:]:
        for a, b in zip(outs[0], o):
            assert np.array_equal(a, b)


@pytest.mark.parametrize("eps", [EPS, 0.0])
def test_duplicate_positions(gpu, c_oracle, eps):
    """Reading R6: a coincident j != i adds -m_j/eps to pot and nothing to acc, jerk for eps > 0;
    for eps = 0 the zero-distance pair contributes nothing at all."""
    m, x, v = inputs.plummer_f32(300, seed=21)
    x[17] = x[250]
    x[100] = x[101]
    v[100] = v[101]
    ref = c_oracle.force(m, x, v, eps)
    with Ctx(300) as ctx:
        nb.nbk_set_j_particles(ctx, None, None, m, x, v)
        nb.nbk_set_ti(ctx, 0.0)
        nb.nbk_calc_firsthalf(ctx, 300, 300, None, None, None, np.float32(eps) ** 2, FULL)
        got = nb.nbk_calc_lasthalf(ctx, 300)
    assert_parity(got, ref, what=f"duplicates eps={eps}")


def test_external_test_particles_and_explicit_i_state(gpu, c_oracle):
    """i_index = -1: external particle, no j left out; i_index >= 0 with xi/vi given: the explicit
    state is used and the own j entry is still left out by index."""
    m, x, v = inputs.plummer_f32(1000, seed=31)
    rng = np.random.default_rng(5)
    n_i = 70
    idx = np.full(n_i, -1, np.int32)
    idx[::2] = rng.choice(1000, size=idx[::2].size, replace=False)
    xi = (0.5 * rng.standard_normal((n_i, 3))).astype(np.float32)
    vi = (0.5 * rng.standard_normal((n_i, 3))).astype(np.float32)
    ref = c_oracle.force(m, x, v, EPS, i_index=idx, xi=xi, vi=vi)
    with Ctx(1000) as ctx:
        nb.nbk_set_j_particles(ctx, None, None, m, x, v)
        nb.nbk_set_ti(ctx, 0.0)
        nb.nbk_calc_firsthalf(ctx, 1000, n_i, idx, xi, vi, np.float32(EPS) ** 2, FULL)
        got = nb.nbk_calc_lasthalf(ctx, n_i)
    assert_parity(got, ref, what="external / explicit i-state")


def test_heavy_particle_self_potential_is_excluded_exactly(gpu, c_oracle):
    """A particle holding half the mass with tiny softening: m_i/eps = 5e5 |pot|.  Adding and
    subtracting its self term in fp32 would lose the potential; exclusion by index does not."""
    m, x, v = inputs.plummer_f32(513, seed=41)
    m = m.copy()
    m[300] = 0.5
    eps = 1e-6
    ref = c_oracle.force(m, x, v, eps)
    with Ctx(513) as ctx:
        nb.nbk_set_j_particles(ctx, None, None, m, x, v)
        nb.nbk_set_ti(ctx, 0.0)
        nb.nbk_calc_firsthalf(ctx, 513, 513, None, None, None, np.float32(eps) ** 2, FULL)
        got = nb.nbk_calc_lasthalf(ctx, 513)
    assert_parity(got, ref, what="heavy particle")


def test_scatter_by_address_f64_and_j_subset(gpu, c_oracle):
    """a1 with addresses (set_j in two shuffled batches, fp64 entry point) and n_j < loaded n:
    only j in [0, n_j) act."""
    m, x, v = inputs.plummer(2000, seed=51)
    perm = np.random.default_rng(6).permutation(2000).astype(np.int32)
    with Ctx(2000) as ctx:
        for part in (perm[:700], perm[700:]):
            nb.nbk_set_j_particles_f64(ctx, part, None, m[part], x[part], v[part])
        nb.nbk_set_ti(ctx, 0.0)
        nb.nbk_calc_firsthalf(ctx, 1500, 1500, None, None, None, np.float32(EPS) ** 2, FULL)
        got = nb.nbk_calc_lasthalf(ctx, 1500)
        gm, gx, gv = nb.nbk_get_predicted(ctx, 1500)
    assert np.array_equal(gx, x[:1500].astype(np.float32))
    ref = c_oracle.force(gm, gx, gv, EPS)
    assert_parity(got, ref, what="scatter + subset")


def test_device_pointer_entry_points_on_a_torch_stream(gpu, c_oracle):
    """_dev variants with torch tensors on a torch stream (PyTorch only owns memory and stream)."""
    torch = gpu
    m, x, v = inputs.plummer_f32(3000, seed=61)
    ref = c_oracle.force(m, x, v, EPS)
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        dm, dx, dv = (torch.from_numpy(t).cuda() for t in (m, x, v))
        acc = torch.empty((3000, 3), dtype=torch.float32, device="cuda")
        jrk = torch.empty_like(acc)
        pot = torch.empty(3000, dtype=torch.float32, device="cuda")
    stream.synchronize()
    with Ctx(3000, stream=stream.cuda_stream) as ctx:
        nb.nbk_set_j_particles_dev(ctx, 3000, 0, 0, dm.data_ptr(), dx.data_ptr(), dv.data_ptr())
        nb.nbk_set_ti(ctx, 0.0)
        nb.nbk_calc_firsthalf_dev(ctx, 3000, 3000, 0, 0, 0, np.float32(EPS) ** 2, FULL)
        nb.nbk_calc_lasthalf_dev(ctx, 3000, acc.data_ptr(), jrk.data_ptr(), pot.data_ptr())
        nb.nbk_sync(ctx)
        got = (acc.cpu().numpy(), jrk.cpu().numpy(), pot.cpu().numpy())
    assert_parity(got, ref, what="device entry points")


def test_errors_do_not_depend_on_which_kernel_shape_ran(gpu, c_oracle):
    """Same 4099 x 4099 problem through every i-per-thread shape: each within tolerance of the
    oracle and within fp32 round-off of one another."""
    m, x, v = inputs.plummer_f32(4099, seed=71)
    ref = c_oracle.force(m, x, v, EPS)
    res = []
    with Ctx(4099) as ctx:
        nb.nbk_set_j_particles(ctx, None, None, m, x, v)
        nb.nbk_set_ti(ctx, 0.0)
        for variant in (0x10, 0x20, 0x40, 0x00):
            nb.nbk_set_variant(ctx, variant)
            nb.nbk_calc_firsthalf(ctx, 4099, 4099, None, None, None, np.float32(EPS) ** 2, FULL)
            res.append(nb.nbk_calc_lasthalf(ctx, 4099))
            assert_parity(res[-1], ref, what=f"variant {variant:#x}")
    for r in res[1:]:
        assert np.percentile(vec_rel_err(r[0], res[0][0]), 99) < 5e-6
        assert scalar_rel_err(r[2], res[0][2]).max() < 2e-6


@pytest.mark.parametrize("n_i", [1, 5, 32])
def test_small_block_one_launch_path_matches_two_kernel_path(gpu, c_oracle, n_i):
    """Blocks of <= 32 i-particles are reduced by the force kernel's last CTA (one launch, indices in
    the launch parameters, results in mapped host memory).  Same sums as force + reduce kernels."""
    m, x, v = inputs.plummer_f32(6000, seed=81)
    idx = inputs.active_block(6000, n_i, seed=4)
    ref = c_oracle.force(m, x, v, EPS, i_index=idx)
    with Ctx(6000) as ctx:
        nb.nbk_set_j_particles(ctx, None, None, m, x, v)
        nb.nbk_set_ti(ctx, 0.0)
        out = {}
        for variant in (0x000, 0x100):
            nb.nbk_set_variant(ctx, variant)
            runs = []
            for _ in range(3):
                nb.nbk_calc_firsthalf(ctx, 6000, n_i, idx, None, None, np.float32(EPS) ** 2, FULL)
                runs.append(nb.nbk_calc_lasthalf(ctx, n_i))
            assert nb.nbk_last_launch(ctx)["launches"] == (1 if variant == 0 else 2)
            for r in runs[1:]:
                assert all(np.array_equal(a, b) for a, b in zip(runs[0], r))
            out[variant] = runs[0]
            assert_parity(runs[0], ref, what=f"small block n_i={n_i} variant {variant:#x}")
        # identity index (i_index = NULL) through the same path
        nb.nbk_set_variant(ctx, 0)
        nb.nbk_calc_firsthalf(ctx, 6000, n_i, None, None, None, np.float32(EPS) ** 2, FULL)
        ident = nb.nbk_calc_lasthalf(ctx, n_i)
    assert np.abs(out[0][0] - out[0x100][0]).max() <= 2e-6 * np.abs(ref[0]).max()
    assert scalar_rel_err(out[0][2], out[0x100][2]).max() < 1e-6
    assert_parity(ident, c_oracle.force(m, x, v, EPS, i_index=np.arange(n_i)), what="identity small block")


def test_set_j_of_a_few_particles_rides_in_the_launch(gpu):
    """n <= 16 particles go through the parameter-space scatter; the stored state must equal what the
    staged path stores (read back through the predictor at dt = 0)."""
    m, x, v = inputs.plummer(500, seed=91)
    with Ctx(500) as ctx:
        nb.nbk_set_j_particles_f64(ctx, None, None, m, x, v)
        addr = np.array([499, 3, 250, 17, 0], np.int32)
        x2 = x[addr] + 0.125
        v2 = v[addr] * 0.5
        nb.nbk_set_j_particles_f64(ctx, addr, np.full(5, 0.25), m[addr] * 2, x2, v2)
        nb.nbk_set_ti(ctx, 0.25)
        nb.nbk_predict(ctx, 500)
        gm, gx, gv = nb.nbk_get_predicted(ctx, 500)
    ex, ev, em = x.copy(), v.copy(), m.copy()
    ex[addr], ev[addr], em[addr] = x2, v2, m[addr] * 2
    # untouched particles have t_j = 0, v != 0: they moved by v * 0.25; touched ones (t_j = t) did not
    rest = np.setdiff1d(np.arange(500), addr)
    assert np.array_equal(gx[addr], ex[addr].astype(np.float32))
    assert np.array_equal(gv[addr], ev[addr].astype(np.float32))
    assert np.array_equal(gm, em.astype(np.float32))
    assert np.array_equal(gx[rest], (x[rest] + v[rest].astype(np.float32).astype(np.float64) * 0.25).astype(np.float32))


# ----------------------------------------------------------------------------- nearest neighbour
def _check_nn(got_nn, got_r2, ref_nn, ref_r2, x, idx, xi=None, what=""):
    """Index bit-exact where the answer is unique in fp32; where the GPU picked another j, that j
    must be as near as the true neighbour to within fp32 rounding of the squared distance."""
    got_nn = np.asarray(got_nn, np.int64)
    same = got_nn == ref_nn
    xs = x[np.maximum(idx, 0)].astype(np.float64) if xi is None else xi.astype(np.float64)
    bad = np.nonzero(~same)[0]
    for k in bad:
        assert got_nn[k] >= 0 and got_nn[k] != idx[k], f"{what}: invalid neighbour for i={k}"
        d = x[got_nn[k]].astype(np.float64) - xs[k]
        r2 = float(d @ d)
        assert r2 <= ref_r2[k] * (1 + 1e-6) + 1e-12, f"{what}: i={k} got j={got_nn[k]} r2={r2} ref {ref_r2[k]}"
    assert bad.size <= max(2, 1e-4 * same.size), f"{what}: {bad.size} near-ties of {same.size}"
    fin = np.isfinite(ref_r2)
    assert np.allclose(got_r2[fin], ref_r2[fin], rtol=2e-6, atol=1e-12), what
    return bad.size


@pytest.mark.parametrize("n,n_i,eps", [(1024, 1024, EPS), (4099, 777, EPS), (4099, 4099, 0.0),
                                       (6000, 1, EPS), (6000, 5, EPS), (6000, 32, 0.0), (300, 300, EPS)])
def test_nearest_neighbour_matches_oracle(gpu, c_oracle, n, n_i, eps):
    """SURVEY 8(f)-2 / PAPER.md L126-L128: neighbour index and distance from the force kernel, every
    launch shape (one-launch small blocks, split-j, full), plus: the forces do not change."""
    m, x, v = inputs.plummer_f32(n, seed=200 + n)
    if n == 300:                       # duplicates: the twin is the neighbour at distance 0
        x[17] = x[250]
        x[100] = x[101]
    idx = inputs.active_block(n, n_i, seed=9)
    ref_nn, ref_r2 = c_oracle.nearest_neighbour(x, i_index=idx)
    with Ctx(n) as ctx:
        nb.nbk_set_j_particles(ctx, None, None, m, x, v)
        nb.nbk_set_ti(ctx, 0.0)
        nb.nbk_calc_firsthalf(ctx, n, n_i, idx, None, None, np.float32(eps) ** 2, FULL)
        plain = nb.nbk_calc_lasthalf(ctx, n_i)
        nb.nbk_calc_firsthalf(ctx, n, n_i, idx, None, None, np.float32(eps) ** 2, FULL | nb.NBK_NN)
        withnn = nb.nbk_calc_lasthalf(ctx, n_i)
        nn, r2 = nb.nbk_get_neighbours(ctx, n_i)
        with pytest.raises(nb.NbkError):
            nb.nbk_calc_firsthalf(ctx, n, n_i, idx, None, None, np.float32(eps) ** 2, nb.NBK_POT | nb.NBK_NN)
    if n_i > 32:
        for a, b in zip(plain, withnn):
            assert np.array_equal(a, b)
    else:   # small blocks: the plain call is the one-launch kernel, the neighbour search rides in the tiled one.
        # Different summation orders, so not the same bits: each form must sit within a few fp32 ulps of the
        # fp64 oracle sum (ulp of the vector's norm; measured on a B200: acc <= 0.86, jerk <= 4.2, pot <= 0.51), hence within a
        # few ulps of the other.
        ref = c_oracle.force(m, x, v, eps, i_index=idx)
        ulp = 2.0 ** -23
        for name, got in (("one-launch", plain), ("tiled+nn", withnn)):
            ea = vec_rel_err(got[0], ref[0]).max() / ulp
            ej = vec_rel_err(got[1], ref[1]).max() / ulp
            ep = scalar_rel_err(got[2], ref[2]).max() / ulp
            print(f"nn small block n_i={n_i} eps={eps} {name}: acc {ea:.2f} jerk {ej:.2f} pot {ep:.2f} ulp")
            assert ea <= 4.0 and ej <= 16.0 and ep <= 2.0, (name, ea, ej, ep)
    _check_nn(nn, r2, ref_nn, ref_r2, x, idx, what=f"nn n={n} n_i={n_i} eps={eps}")
    if n == 300:
        pos = {int(i): k for k, i in enumerate(idx)}
        assert nn[pos[17]] == 250 and nn[pos[250]] == 17 and nn[pos[100]] == 101 and r2[pos[100]] == 0.0


def test_nearest_neighbour_external_particles_and_j_subset(gpu, c_oracle):
    m, x, v = inputs.plummer_f32(3000, seed=231)
    rng = np.random.default_rng(3)
    n_i, n_j = 90, 2500
    idx = np.full(n_i, -1, np.int32)
    idx[::3] = rng.choice(n_j, size=idx[::3].size, replace=False)
    xi = (0.4 * rng.standard_normal((n_i, 3))).astype(np.float32)
    ref_nn, ref_r2 = c_oracle.nearest_neighbour(x[:n_j], i_index=idx, xi=xi)
    with Ctx(3000) as ctx:
        nb.nbk_set_j_particles(ctx, None, None, m, x, v)
        nb.nbk_set_ti(ctx, 0.0)
        nb.nbk_calc_firsthalf(ctx, n_j, n_i, idx, xi, None, np.float32(EPS) ** 2, FULL | nb.NBK_NN)
        nb.nbk_calc_lasthalf(ctx, n_i)
        nn, r2 = nb.nbk_get_neighbours(ctx, n_i)
    assert nn.max() < n_j
    _check_nn(nn, r2, ref_nn, ref_r2, x, idx, xi=xi, what="nn external")


def test_nearest_neighbour_c3_full(gpu, c_oracle):
    """N = 131072, all i, in the launch shape of the headline run."""
    m, x, v = inputs.config_inputs("C3")
    n = m.shape[0]
    ref_nn, ref_r2 = c_oracle.nearest_neighbour(x)
    with Ctx(n) as ctx:
        nb.nbk_set_j_particles(ctx, None, None, m, x, v)
        nb.nbk_set_ti(ctx, 0.0)
        nb.nbk_calc_firsthalf(ctx, n, n, None, None, None, np.float32(EPS) ** 2, FULL | nb.NBK_NN)
        nb.nbk_calc_lasthalf(ctx, n)
        nn, r2 = nb.nbk_get_neighbours(ctx, n)
        assert nb.nbk_last_launch(ctx)["launches"] == 3
    nbad = _check_nn(nn, r2, ref_nn, ref_r2, x, np.arange(n), what="nn C3")
    print(f"C3 nearest neighbour: {nbad} fp32 near-ties of {n}")


# ----------------------------------------------------------------------------- device-resident integrator
def test_device_resident_hermite_small_n_matches_host_driver_and_oracle(gpu):
    """the block-step loop on the device (scheduler from level counts, predictor +
    selection, device-planned force, fp64 corrector) against the host driver and the fp64 oracle
    integrator: same scheme => same step counts to a few per cent, nearby end states, same energy."""
    from oracle import hermite_oracle, nbody_oracle
    m, x, v = inputs.plummer(256, seed=11)
    ref = hermite_oracle.evolve(m, x, v, EPS, 0.25)
    hx, hv = x.copy(), v.copy()
    dx, dv = x.copy(), v.copy()
    with Ctx(256) as ctx:
        sh = nb.nbk_hermite_evolve(ctx, m, hx, hv, EPS, 0.25)
        sd = nb.nbk_hermite_evolve_dev(ctx, m, dx, dv, EPS, 0.25)
    assert sd["t_reached"] == 0.25
    assert abs(sd["particle_steps"] - ref["particle_steps"]) <= 0.05 * ref["particle_steps"]
    assert abs(sd["particle_steps"] - sh["particle_steps"]) <= 0.02 * sh["particle_steps"]
    assert sum(sd["ni_histogram"]) == sd["block_steps"]
    e0 = nbody_oracle.energy(m, x, v, EPS)
    assert abs((nbody_oracle.energy(m, dx, dv, EPS) - e0) / e0) < 1e-6
    assert np.median(np.linalg.norm(dx - ref["x"], axis=1)) < 1e-4
    assert np.median(np.linalg.norm(dx - hx, axis=1)) < 1e-4


def test_device_resident_hermite_c5_energy(gpu, c_oracle):
    """C5 on the device-resident loop: N=65536 to t=1, |dE/E| < 1e-6, same block-step statistics
    as the host-driven run to within the sensitivity of step choices to fp32 force round-off."""
    m, x, v = inputs.plummer(inputs.CONFIGS["C5"]["N"], inputs.CONFIGS["C5"]["seed"])
    n = m.shape[0]
    e0 = _energy(c_oracle, m, x, v, EPS)
    with Ctx(n) as ctx:
        st = nb.nbk_hermite_evolve_dev(ctx, m, x, v, EPS, 1.0, eta=0.01, dt_max=1.0 / 16.0)
    e1 = _energy(c_oracle, m, x, v, EPS)
    de = abs((e0 - e1) / e0)
    print(f"C5 device-resident: dE/E={de:.3e} block_steps={st['block_steps']} "
          f"particle_steps={st['particle_steps']} wall={st['wall_seconds']:.2f}s "
          f"interactions={st['interactions']:.3e}")
    assert st["t_reached"] == 1.0
    assert de < 1e-6, de
    assert 0.9 * 62748 < st["block_steps"] < 1.1 * 62748


def test_device_resident_hermite_is_repeatable(gpu):
    """The order in which due particles are collected is not fixed (atomic cursor), but each
    particle's sums do not depend on its slot: two runs end in bit-identical states."""
    m, x, v = inputs.plummer(3000, seed=17)
    outs = []
    with Ctx(3000) as ctx:
        for _ in range(2):
            gx, gv = x.copy(), v.copy()
            st = nb.nbk_hermite_evolve_dev(ctx, m, gx, gv, EPS, 0.125)
            outs.append((gx, gv, st["block_steps"], st["particle_steps"]))
    assert outs[0][2:] == outs[1][2:]
    assert np.array_equal(outs[0][0], outs[1][0]) and np.array_equal(outs[0][1], outs[1][1])


@pytest.mark.parametrize("n_i", [1, 7, 32, 33, 200, 1531])
def test_every_kernel_form_flag_and_block_size(gpu, c_oracle, n_i):
    """Matrix: block sizes on both sides of the one-launch limit x {acc+jerk+pot, acc+pot, +NN, eps=0}
    x {planner's choice, I pinned to 1/2/4, scalar loop, two-kernel path}; prediction active.
    Every combination against the oracle on the device-predicted state."""
    n = 1531
    m, x, v = inputs.plummer_f32(n, seed=7)
    a0, j0 = (0.1 * v).astype(np.float32), (0.01 * v).astype(np.float32)
    idx = inputs.active_block(n, n_i, seed=3)
    with Ctx(n) as ctx:
        nb.nbk_set_j_particles(ctx, None, np.zeros(n), m, x, v, a0, j0)
        nb.nbk_set_ti(ctx, 0.01)
        nb.nbk_predict(ctx, n)
        gm, gx, gv = nb.nbk_get_predicted(ctx, n)
        refs = {eps: c_oracle.force(gm, gx, gv, eps, i_index=idx) for eps in (EPS, 0.0)}
        ref_nn, ref_r2 = c_oracle.nearest_neighbour(gx, i_index=idx)
        for flags in (FULL, nb.NBK_POT, FULL | nb.NBK_NN, FULL | nb.NBK_EPS0):
            eps = 0.0 if flags & nb.NBK_EPS0 else EPS
            jerk = bool(flags & nb.NBK_JERK)
            for variant in (0x000, 0x010, 0x020, 0x040, 0x110, 0x100):
                nb.nbk_set_variant(ctx, variant)
                nb.nbk_calc_firsthalf(ctx, n, n_i, idx, None, None, np.float32(eps) ** 2, flags)
                got = nb.nbk_calc_lasthalf(ctx, n_i)
                assert_parity(got, refs[eps], jerk=jerk, what=f"n_i={n_i} flags={flags} variant={variant:#x}")
                if not jerk:
                    assert np.all(got[1] == 0)
                if flags & nb.NBK_NN:
                    nn, r2 = nb.nbk_get_neighbours(ctx, n_i)
                    _check_nn(nn, r2, ref_nn, ref_r2, gx, idx, what=f"nn n_i={n_i} variant={variant:#x}")


# ----------------------------------------------------------------------------- batched acc + pot calls
def _batch_problem(seed, n_groups, ni_range, nj_range, with_empty=False):
    """Treecode-shaped synthetic batch: per group a clump of i-particles and an interaction list of
    'cells' (masses, positions) around it; the group's own particles are part of their list."""
    rng = np.random.default_rng(seed)
    ni = rng.integers(ni_range[0], ni_range[1] + 1, n_groups)
    nj = rng.integers(nj_range[0], nj_range[1] + 1, n_groups)
    if with_empty:
        ni[3] = 0
        nj[5] = 0
        nj[6] = 1
    io = np.concatenate([[0], np.cumsum(ni)]).astype(np.int64)
    jo = np.concatenate([[0], np.cumsum(nj)]).astype(np.int64)
    xi = np.empty((io[-1], 3), np.float32)
    xj = np.empty((jo[-1], 3), np.float32)
    mj = rng.uniform(0.5, 2.0, jo[-1]).astype(np.float32) / 1000.0
    for g in range(n_groups):
        centre = rng.standard_normal(3)
        xi[io[g]:io[g + 1]] = (centre + 0.05 * rng.standard_normal((ni[g], 3))).astype(np.float32)
        lst = centre + rng.standard_normal((nj[g], 3)) * rng.uniform(0.05, 2.0, (nj[g], 1))
        k = min(ni[g], nj[g])
        lst[:k] = xi[io[g]:io[g] + k]          # own particles sit in their own list
        xj[jo[g]:jo[g + 1]] = lst.astype(np.float32)
    return io, jo, xi, mj, xj


def _batch_oracle(c_oracle, io, jo, xi, mj, xj, eps):
    acc = np.zeros((io[-1], 3))
    pot = np.zeros(io[-1])
    for g in range(io.shape[0] - 1):
        a, b, c, d = io[g], io[g + 1], jo[g], jo[g + 1]
        if b > a and d > c:
            ra, _, rp = c_oracle.force(mj[c:d], xj[c:d], None, eps, i_index=np.full(b - a, -1),
                                       want_jerk=False, xi=xi[a:b])
            acc[a:b], pot[a:b] = ra, rp
    return acc, pot


@pytest.mark.parametrize("shape", [dict(n_groups=40, ni_range=(1, 90), nj_range=(1, 700)),
                                   dict(n_groups=300, ni_range=(8, 300), nj_range=(100, 2500)),
                                   dict(n_groups=7, ni_range=(400, 1500), nj_range=(3000, 9000)),
                                   dict(n_groups=1, ni_range=(5, 5), nj_range=(3, 3))])
@pytest.mark.parametrize("eps", [EPS, 0.0])
def test_batched_calls_match_oracle(gpu, c_oracle, shape, eps):
    """many (i-group, interaction list) problems of irregular sizes in one launch,
    acc + pot only, against the oracle group by group (external i-particles, nothing excluded by
    index; eps = 0 skips the zero-distance own entries).  Includes empty groups and empty lists."""
    io, jo, xi, mj, xj = _batch_problem(5 + shape["n_groups"], with_empty=shape["n_groups"] >= 40, **shape)
    racc, rpot = _batch_oracle(c_oracle, io, jo, xi, mj, xj, eps)
    with Ctx(64) as ctx:
        flags = nb.NBK_POT | (nb.NBK_EPS0 if eps == 0.0 else 0)
        outs = [nb.nbk_calc_batch(ctx, io, xi, jo, mj, xj, np.float32(eps) ** 2, flags) for _ in range(2)]
        with pytest.raises(nb.NbkError):
            nb.nbk_calc_batch(ctx, io, xi, jo, mj, xj, 0.0, nb.NBK_JERK)
    acc, pot = outs[0]
    assert np.array_equal(acc, outs[1][0]) and np.array_equal(pot, outs[1][1])
    live = np.abs(rpot) > 0
    assert np.all(acc[~live] == 0) and np.all(pot[~live] == 0)
    assert_parity((acc[live], None, pot[live]), (racc[live], None, rpot[live]), jerk=False, what=f"batch {shape}")


def test_batched_calls_device_pointers(gpu, c_oracle):
    torch = gpu
    io, jo, xi, mj, xj = _batch_problem(77, 120, (16, 200), (200, 1500))
    racc, rpot = _batch_oracle(c_oracle, io, jo, xi, mj, xj, EPS)
    dxi, dmj, dxj = (torch.from_numpy(t).cuda() for t in (xi, mj, xj))
    acc = torch.empty((io[-1], 3), dtype=torch.float32, device="cuda")
    pot = torch.empty(io[-1], dtype=torch.float32, device="cuda")
    torch.cuda.synchronize()
    with Ctx(64) as ctx:
        nb.nbk_calc_batch_dev(ctx, io, dxi.data_ptr(), jo, dmj.data_ptr(), dxj.data_ptr(), np.float32(EPS) ** 2,
                              nb.NBK_POT, acc.data_ptr(), pot.data_ptr())
    assert_parity((acc.cpu().numpy(), None, pot.cpu().numpy()), (racc, None, rpot), jerk=False, what="batch dev")


def test_caller_owned_workspace_and_double_readback(gpu, c_oracle):
    """nbk_open_ws: every device buffer of the context lives in one torch tensor the caller owns
    (PyTorch is the allocator); nbk_calc_lasthalf_f64 returns the same fp32 results widened."""
    torch = gpu
    n = 5000
    m, x, v = inputs.plummer_f32(n, seed=301)
    need = nb.nbk_workspace_bytes(0, n, n)
    assert need > 0
    ws = torch.empty(need, dtype=torch.uint8, device="cuda")
    assert ws.data_ptr() % 256 == 0
    with pytest.raises(nb.NbkError):
        nb.nbk_open_ws(0, n, n, 0, ws.data_ptr(), need - 1)
    ctx = nb.nbk_open_ws(0, n, n, 0, ws.data_ptr(), need)
    try:
        nb.nbk_set_j_particles(ctx, None, None, m, x, v)
        nb.nbk_set_ti(ctx, 0.0)
        nb.nbk_calc_firsthalf(ctx, n, n, None, None, None, np.float32(EPS) ** 2, FULL | nb.NBK_NN)
        got = nb.nbk_calc_lasthalf(ctx, n)
        got64 = nb.nbk_calc_lasthalf_f64(ctx, n)
        nn, r2 = nb.nbk_get_neighbours(ctx, n)
    finally:
        nb.nbk_close(ctx)
    ws.zero_()          # still the caller's: close did not free it
    torch.cuda.synchronize()
    assert_parity(got, c_oracle.force(m, x, v, EPS), what="workspace ctx")
    for a, b in zip(got, got64):
        assert b.dtype == np.float64 and np.array_equal(a.astype(np.float64), b)
    ref_nn, ref_r2 = c_oracle.nearest_neighbour(x)
    _check_nn(nn, r2, ref_nn, ref_r2, x, np.arange(n), what="workspace ctx nn")


# ----------------------------------------------------------------------------- round-2 additions
def test_set_j_dev_with_addresses_times_and_derivatives(gpu, c_oracle):
    """a1 for a device-resident caller (PAPER.md L427 GPU_set_j_particle: address, time, mass, x, v,
    a, jerk): nbk_set_j_particles_dev with DEVICE addr, tj, a, jerk in two shuffled batches, then the
    device predictor (a3) and a force block: predicted state and forces against the oracle."""
    torch = gpu
    n = 5000
    m, x, v = inputs.plummer_f32(n, seed=91)
    t = 0.01
    tj = inputs.particle_times(n, t, seed=9)
    a, jk = inputs.gaussian_derivatives(n, seed=9)
    a, jk = a.astype(np.float32), jk.astype(np.float32)
    perm = np.random.default_rng(12).permutation(n).astype(np.int32)
    xp, vp = c_oracle.predict(t, tj, x, v, a, jk)
    idx = inputs.active_block(n, 777, seed=4)
    keep = []
    with Ctx(n) as ctx:
        for part in (perm[:1803], perm[1803:]):
            dev = [torch.from_numpy(np.ascontiguousarray(arr[part])).cuda() for arr in (tj, m, x, v, a, jk)]
            dad = torch.from_numpy(part.copy()).cuda()
            keep += dev + [dad]
            torch.cuda.synchronize()
            nb.nbk_set_j_particles_dev(ctx, part.shape[0], dad.data_ptr(), *[d.data_ptr() for d in dev])
        nb.nbk_set_ti(ctx, t)
        nb.nbk_calc_firsthalf(ctx, n, 777, idx, None, None, np.float32(EPS) ** 2, FULL)
        got = nb.nbk_calc_lasthalf(ctx, 777)
        gm, gx, gv = nb.nbk_get_predicted(ctx, n)
    assert np.array_equal(gm, m)
    for g, ref in ((gx, xp), (gv, vp)):
        ulp = np.spacing(np.abs(ref).astype(np.float32)).astype(np.float64)
        assert np.all(np.abs(g.astype(np.float64) - ref) <= ulp)
        assert np.mean(g == ref.astype(np.float32)) > 0.99
    assert_parity(got, c_oracle.force(m, xp, vp, EPS, i_index=idx), what="set_j_dev addr/tj/a/jerk")


@pytest.mark.parametrize("driver", ["host", "dev"])
def test_hermite_start_up_step_closed_form(gpu, driver):
    """Reading R15's start-up step dt_0 = largest 2^-k <= (eta/4)|a|/|j| through the C ABI, on a case
    with a closed form (same as tests/test_hermite_oracle.py): equal masses 1/2 on a circular orbit of
    separation 1, eps = 0: |a| = |j| = 1/2, (0.01/4) -> 2^-9.  The Aarseth step of a circle (0.1) exceeds
    dt_max = 1/16, so the step doubles whenever the block rule allows: 2^-9, 2^-9, 2^-8, 2^-7, 2^-6,
    2^-5 reach t = 1/16 in exactly 6 block steps of 2 particles (5 if dt_0 were 2^-8, 4 if 2^-7)."""
    m = np.array([0.5, 0.5])
    x0 = np.array([[-0.5, 0, 0], [0.5, 0, 0]])
    v0 = np.array([[0, -0.5, 0], [0, 0.5, 0]])
    fn = nb.nbk_hermite_evolve if driver == "host" else nb.nbk_hermite_evolve_dev
    with Ctx(64) as ctx:
        x, v = x0.copy(), v0.copy()
        st = fn(ctx, m, x, v, 0.0, 1.0 / 16.0, eta=0.01, dt_max=1.0 / 16.0)
        assert st["t_reached"] == 1.0 / 16.0
        assert st["block_steps"] == 6 and st["particle_steps"] == 12
        assert sum(st["ni_histogram"]) == 6
        # one step of dt_max = 2^-9 lands exactly on t_end = 2^-9
        x, v = x0.copy(), v0.copy()
        st = fn(ctx, m, x, v, 0.0, 2.0 ** -9, eta=0.01, dt_max=2.0 ** -9)
        assert st["block_steps"] == 1 and st["particle_steps"] == 2
    # the orbit: after t the pair has turned by the angle t (omega = 1)
    ang = 2.0 ** -9
    np.testing.assert_allclose(x[1], [0.5 * np.cos(ang), 0.5 * np.sin(ang), 0.0], atol=1e-9)


@pytest.mark.parametrize("driver", ["host", "dev"])
def test_hermite_drivers_refuse_dt_max_of_two_or_more(gpu, driver):
    """dt_max in [2^-48, 2): the level lists are indexed from 2^0 (include/nbk.h); 2 and above, and
    non-positive or NaN values, are NBK_EINVAL in both drivers (no out-of-range level)."""
    m, x, v = inputs.plummer(64, seed=5)
    fn = nb.nbk_hermite_evolve if driver == "host" else nb.nbk_hermite_evolve_dev
    with Ctx(64) as ctx:
        for bad in (2.0, 4.0, 1024.0, 0.0, -1.0, float("nan"), 2.0 ** -60):
            with pytest.raises(nb.NbkError) as e:
                fn(ctx, m, x.copy(), v.copy(), EPS, 1024.0 if bad > 2 else 2.0, eta=0.01, dt_max=bad)
            assert e.value.status == nb.NBK_EINVAL, bad
        st = fn(ctx, m, x.copy(), v.copy(), EPS, 1.0, eta=0.01, dt_max=1.9)   # rounds down to 2^0
        assert st["t_reached"] == 1.0 and st["block_steps"] > 16


@pytest.mark.parametrize("n,n_i", [(1024, 1024), (300, 7)])
def test_subnormal_softening_is_zero_softening(gpu, c_oracle, n, n_i):
    """The kernels flush subnormals (.ftz): eps = 1e-20 (eps^2 = 1e-40, a subnormal fp32) must act as
    eps = 0 -- own entry and zero-distance pairs skipped -- not produce NaN."""
    m, x, v = inputs.plummer_f32(n, seed=33)
    x[5] = x[9]                                    # a coincident pair besides the own entries
    idx = inputs.active_block(n, n_i, seed=1) if n_i < n else None
    if idx is not None:
        idx[0] = 5
        idx = np.unique(idx).astype(np.int32)
        n_i = idx.shape[0]
    eps2 = np.float32(1e-40)
    assert 0 < eps2 < np.finfo(np.float32).tiny
    ref = c_oracle.force(m, x, v, 0.0, i_index=idx)
    with Ctx(n) as ctx:
        nb.nbk_set_j_particles(ctx, None, None, m, x, v)
        nb.nbk_set_ti(ctx, 0.0)
        nb.nbk_calc_firsthalf(ctx, n, n_i, idx, None, None, eps2, FULL)
        got = nb.nbk_calc_lasthalf(ctx, n_i)
    assert all(np.isfinite(g).all() for g in got)
    assert_parity(got, ref, what="subnormal eps2")


@pytest.mark.parametrize("eps", [EPS, 0.0])
def test_device_resident_paths_agree(gpu, monkeypatch, eps):
    """nbk_hermite_evolve_dev by its three routes -- every step through the chain of launches
    (NBK_STEPS_MAX_ACT=0: what runs for n > 131072), steps of <= 4 particles in the persistent stepping
    kernel (lanes over j), steps of <= 1024 (lanes over i too) -- against the host driver: same scheme,
    so the same step counts to a few per cent, nearby end states, the same energy; each route bitwise
    repeatable.  eps = 0 takes the guarded pair loops (hd_steps_kernel<true>, EPS0 force kernels)."""
    from oracle import nbody_oracle
    m, x, v = inputs.plummer(1500, seed=23)
    e0 = nbody_oracle.energy(m, x, v, eps)
    with Ctx(1500) as ctx:
        hx, hv = x.copy(), v.copy()
        sh = nb.nbk_hermite_evolve(ctx, m, hx, hv, eps, 0.125)
        for max_act in ("0", "4", "1024"):
            monkeypatch.setenv("NBK_STEPS_MAX_ACT", max_act)
            runs = []
            for _ in range(2):
                gx, gv = x.copy(), v.copy()
                st = nb.nbk_hermite_evolve_dev(ctx, m, gx, gv, eps, 0.125)
                runs.append((gx, gv, st))
            assert np.array_equal(runs[0][0], runs[1][0]) and np.array_equal(runs[0][1], runs[1][1]), max_act
            gx, gv, st = runs[0]
            assert st["t_reached"] == 0.125
            assert sum(st["ni_histogram"]) == st["block_steps"]
            assert abs(st["particle_steps"] - sh["particle_steps"]) <= 0.03 * sh["particle_steps"], max_act
            assert abs((nbody_oracle.energy(m, gx, gv, eps) - e0) / e0) < 1e-6, max_act
            assert np.median(np.linalg.norm(gx - hx, axis=1)) < 1e-4, max_act


@pytest.mark.parametrize("n", [40000, 70001])
def test_device_resident_stepping_kernel_at_bench_sizes(gpu, c_oracle, monkeypatch, n):
    """The stepping kernel at the sizes the C5 number is measured at, which the N = 1500 test above never
    reaches: a j-chunk of several hundred particles per CTA (multi-block loop over 256-particle blocks),
    more than one 16-byte vector of level bytes per thread in the due-list scan (n > 65536: more than four),
    and due lists of 513..1024 particles that take the three-round split of the tiled pair sums.  Integrated
    to t = 1/16 with all steps of <= 1024 particles in hd_steps_kernel, twice (bitwise repeatable), against the
    launch-chain route and the host driver: same particle steps to 0.1 %, nearby end states, energy."""
    m, x, v = inputs.plummer(n, seed=77)
    t_end = 1.0 / 16.0
    e0 = _energy(c_oracle, m, x, v, EPS)
    with Ctx(n) as ctx:
        hx, hv = x.copy(), v.copy()
        sh = nb.nbk_hermite_evolve(ctx, m, hx, hv, EPS, t_end)
        out = {}
        for max_act in ("1024", "0"):
            monkeypatch.setenv("NBK_STEPS_MAX_ACT", max_act)
            runs = []
            for _ in range(2 if max_act == "1024" else 1):
                gx, gv = x.copy(), v.copy()
                st = nb.nbk_hermite_evolve_dev(ctx, m, gx, gv, EPS, t_end)
                runs.append((gx, gv, st))
            if len(runs) == 2:
                assert np.array_equal(runs[0][0], runs[1][0]) and np.array_equal(runs[0][1], runs[1][1])
                assert runs[0][2]["particle_steps"] == runs[1][2]["particle_steps"]
            out[max_act] = runs[0]
    gx, gv, st = out["1024"]
    cx, cv, sc = out["0"]
    hist = st["ni_histogram"]
    assert sum(hist[:10]) > 100 and hist[9] > 0, hist        # steps the stepping kernel takes, incl. 512..1023
    for what, (ox, ov, so) in (("launch chain", (cx, cv, sc)), ("host driver", (hx, hv, sh))):
        dx = np.linalg.norm(gx - ox, axis=1)
        print(f"n={n} stepping kernel vs {what}: particle_steps {st['particle_steps']} / {so['particle_steps']}, "
              f"block_steps {st['block_steps']} / {so['block_steps']}, |dx| median {np.median(dx):.2e} "
              f"p99 {np.percentile(dx, 99):.2e} max {dx.max():.2e}")
        assert st["t_reached"] == so["t_reached"] == t_end
        # measured: particle steps within 1.1e-4 relative, |dx| median <= 9.2e-12, p99 <= 4.1e-11
        assert abs(st["particle_steps"] - so["particle_steps"]) <= 1e-3 * so["particle_steps"], what
        assert np.median(dx) < 1e-10 and np.percentile(dx, 99) < 1e-9, what
    e1 = _energy(c_oracle, m, gx, gv, EPS)
    assert abs((e1 - e0) / e0) < 1e-6


def test_device_resident_reports_its_launch_form_and_validates_the_knob(gpu, monkeypatch):
    """nbk_last_launch after nbk_hermite_evolve_dev says whether the persistent stepping kernel ran and how it
    was captured (2: cooperative launch, 1: plain launch, 0: not used), so a silent fall-back from the
    cooperative form is visible; NBK_STEPS_MAX_ACT must be a whole number in 0..1024."""
    m, x, v = inputs.plummer(600, seed=3)
    with Ctx(600) as ctx:
        monkeypatch.setenv("NBK_STEPS_MAX_ACT", "1024")
        nb.nbk_hermite_evolve_dev(ctx, m, x.copy(), v.copy(), EPS, 1.0 / 64.0, dt_max=1.0 / 64.0)
        shape = nb.nbk_last_launch(ctx)
        assert shape["launches"] == 2, shape          # the B200 box captures the cooperative form
        assert shape["grid"] == shape["sms"] and shape["threads"] == 512 and shape["j_tile"] == 1024
        monkeypatch.setenv("NBK_STEPS_MAX_ACT", "0")
        nb.nbk_hermite_evolve_dev(ctx, m, x.copy(), v.copy(), EPS, 1.0 / 64.0, dt_max=1.0 / 64.0)
        shape = nb.nbk_last_launch(ctx)
        assert shape["launches"] == 0 and shape["grid"] == 0, shape
        for bad in ("-1", "1025", "12x", "", "4.5"):
            monkeypatch.setenv("NBK_STEPS_MAX_ACT", bad)
            with pytest.raises(nb.NbkError) as e:
                nb.nbk_hermite_evolve_dev(ctx, m, x.copy(), v.copy(), EPS, 1.0 / 64.0, dt_max=1.0 / 64.0)
            assert e.value.status == nb.NBK_EINVAL, bad


_PDL_SCRIPT = """
import sys, numpy as np
sys.path.insert(0, {root!r})
from paper_0707_0438_b200 import binding as nb, inputs
m, x, v = inputs.plummer_f32(3000, seed=8)
ctx = nb.nbk_open(0, 3000, 3000)
out = []
nb.nbk_set_j_particles(ctx, None, None, m, x, v)
for n_i, t in ((3000, 0.0), (200, 0.01), (7, 0.02)):
    nb.nbk_set_ti(ctx, t)
    idx = inputs.active_block(3000, n_i, seed=n_i)
    nb.nbk_calc_firsthalf(ctx, 3000, n_i, idx, None, None, np.float32(1 / 256) ** 2, 3)
    out += list(nb.nbk_calc_lasthalf(ctx, n_i))
md, xd, vd = inputs.plummer(400, seed=9)
nb.nbk_hermite_evolve_dev(ctx, md, xd, vd, 1 / 256, 1 / 32, dt_max=1 / 32)
nb.nbk_close(ctx)
np.savez({path!r}, *out, xd, vd)
"""


def test_programmatic_dependent_launch_switch_changes_no_bits(gpu, tmp_path):
    """NBK_PDL=0 (read once per process, csrc/nbk_api.cu) launches the block-step kernel chain without the
    programmatic-dependent-launch attribute: griddepcontrol.wait / launch_dependents then do nothing and the
    stream orders the kernels fully.  Same kernels, same data, so the same bits as with the attribute on -- a
    kernel that touched global memory before its pdl_wait would differ with it on.  Two child processes."""
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    res = {}
    for pdl in ("1", "0"):
        path = str(tmp_path / f"pdl{pdl}.npz")
        env = dict(os.environ, NBK_PDL=pdl)
        env.pop("NBK_STEPS_MAX_ACT", None)
        subprocess.run([sys.executable, "-c", _PDL_SCRIPT.format(root=root, path=path)], check=True, env=env,
                       timeout=600)
        with np.load(path) as z:
            res[pdl] = [z[k] for k in z.files]
    assert len(res["1"]) == len(res["0"]) == 11
    for a, b in zip(res["1"], res["0"]):
        assert np.array_equal(a, b)


def test_stepping_kernel_200_repeats_bitwise(gpu, monkeypatch):
    """hd_steps_kernel hands partial rows and per-particle flags from CTA to CTA through global memory
    (tagged 8-byte words, st.relaxed / ld.acquire, no grid barrier) -- traffic compute-sanitizer's racecheck
    does not look at (it checks shared memory only; profiles/r03_sanitizer.md).  A missed wait would show as a
    run that read a stale row: 200 runs of N = 1500 to t = 1/32 (~400 block steps each) must all end in the
    bits of the first, for eps > 0 and eps = 0."""
    m, x, v = inputs.plummer(1500, seed=23)
    monkeypatch.setenv("NBK_STEPS_MAX_ACT", "1024")
    with Ctx(1500) as ctx:
        for eps in (EPS, 0.0):
            first = None
            for rep in range(200):
                gx, gv = x.copy(), v.copy()
                st = nb.nbk_hermite_evolve_dev(ctx, m, gx, gv, eps, 1.0 / 32.0, dt_max=1.0 / 32.0)
                if first is None:
                    first = (gx, gv, st["block_steps"], st["particle_steps"])
                    assert st["t_reached"] == 1.0 / 32.0 and st["block_steps"] > 100
                    continue
                assert (st["block_steps"], st["particle_steps"]) == first[2:], (eps, rep)
                assert np.array_equal(gx, first[0]) and np.array_equal(gv, first[1]), (eps, rep)


def test_batched_calls_small_groups_split_lanes(gpu, c_oracle):
    """Batched calls with the lanes of a warp split 2 and 4 ways over each j-tile (mean group size
    12-23 and below 12): every group against the oracle, bitwise repeatable."""
    for ni_range, slices in (((6, 30), 2), ((2, 12), 4)):
        io, jo, xi, mj, xj = _batch_problem(31 + slices, 500, ni_range, (40, 900))
        racc, rpot = _batch_oracle(c_oracle, io, jo, xi, mj, xj, EPS)
        with Ctx(64) as ctx:
            outs = [nb.nbk_calc_batch(ctx, io, xi, jo, mj, xj, np.float32(EPS) ** 2, nb.NBK_POT) for _ in range(2)]
            assert nb.nbk_last_launch(ctx)["j_split_warps"] == slices
        assert np.array_equal(outs[0][0], outs[1][0]) and np.array_equal(outs[0][1], outs[1][1])
        assert_parity((outs[0][0], None, outs[0][1]), (racc, None, rpot), jerk=False, what=f"batch slices={slices}")


@pytest.mark.parametrize("n_i", [1, 3, 4, 5, 17, 32])
def test_small_block_kernel_one_launch_predict_force_reduce(gpu, c_oracle, n_i):
    """Blocks of <= 32 particles of the j-set are ONE launch (small_block_kernel): every CTA predicts its own
    j-particles and the i-particles from the raw state, sums, the last CTA reduces (PAPER.md L78, L256,
    L112-L118).  Against the oracle on the oracle-predicted state, with and without jerk, eps > 0 and 0;
    the predicted arrays it leaves behind are the predictor kernel's bits; a set_j of a few particles before
    the call rides in the launch; device index arrays; bitwise repeatable."""
    torch = gpu
    n = 7001
    m, x, v = inputs.plummer_f32(n, seed=61)
    t = 0.0078125
    tj = inputs.particle_times(n, t, seed=5)
    a, jk = inputs.gaussian_derivatives(n, seed=5)
    a, jk = a.astype(np.float32), jk.astype(np.float32)
    idx = inputs.active_block(n, n_i, seed=8)
    with Ctx(n) as ctx:
        nb.nbk_set_j_particles(ctx, None, tj, m, x, v, a, jk)
        # a few corrected particles just before the block step: new state for the first min(n_i, 8) of the block
        k = min(n_i, 8)
        upd = idx[:k]
        x2, v2 = x.copy(), v.copy()
        x2[upd] += np.float32(1e-3)
        v2[upd] *= np.float32(1.01)
        tj2 = tj.copy()
        tj2[upd] = t - 2.0 ** -9
        nb.nbk_set_j_particles(ctx, upd, tj2[upd], m[upd], x2[upd], v2[upd], a[upd], jk[upd])
        xp, vp = c_oracle.predict(t, tj2, x2, v2, a, jk)
        nb.nbk_set_ti(ctx, t)
        for flags, eps in ((FULL, EPS), (nb.NBK_POT, EPS), (FULL | nb.NBK_EPS0, 0.0)):
            jerk = bool(flags & nb.NBK_JERK)
            ref = c_oracle.force(m, xp, vp, eps, i_index=idx, want_jerk=jerk)
            runs = []
            for _ in range(2):
                nb.nbk_calc_firsthalf(ctx, n, n_i, idx, None, None, np.float32(eps) ** 2, flags)
                runs.append(nb.nbk_calc_lasthalf(ctx, n_i))
            shape = nb.nbk_last_launch(ctx)
            assert shape["launches"] == 1 and shape["threads"] == 512 and shape["j_split_warps"] == 16
            assert all(np.array_equal(p, q) for p, q in zip(*runs))
            assert_parity(runs[0], ref, jerk=jerk, what=f"small block n_i={n_i} flags={flags}")
            if not jerk:
                assert np.all(runs[0][1] == 0)
        gm, gx, gv = nb.nbk_get_predicted(ctx, n)          # left behind by the one-launch kernel
        nb.nbk_set_ti(ctx, t + 1.0)
        nb.nbk_set_ti(ctx, t)
        nb.nbk_predict(ctx, n)                              # the predictor kernel proper
        pm, px, pv = nb.nbk_get_predicted(ctx, n)
        assert np.array_equal(gm, pm) and np.array_equal(gx, px) and np.array_equal(gv, pv)
        # device index array through the _dev entry point, results read back on the device
        didx = torch.from_numpy(idx).cuda()
        out = [torch.empty((n_i, 3), dtype=torch.float32, device="cuda") for _ in range(2)]
        out.append(torch.empty(n_i, dtype=torch.float32, device="cuda"))
        torch.cuda.synchronize()
        nb.nbk_calc_firsthalf_dev(ctx, n, n_i, didx.data_ptr(), 0, 0, np.float32(EPS) ** 2, FULL)
        nb.nbk_calc_lasthalf_dev(ctx, n_i, *[o.data_ptr() for o in out])
        nb.nbk_sync(ctx)
        assert nb.nbk_last_launch(ctx)["launches"] == 1
    ref = c_oracle.force(m, xp, vp, EPS, i_index=idx)
    assert_parity(tuple(o.cpu().numpy() for o in out), ref, what=f"small block dev n_i={n_i}")
