"""Pins for the fp64 oracle (numpy and C forms) against what the paper and the
mathematics fix -- never against the CUDA path and never against itself.

Each pin is chosen so a plausible mistake fails it: a wrong sign (two-body,
a = -grad pot), a dropped or mis-scaled jerk term (finite difference of a),
wrong softening placement (a = -grad pot, scalings), a transposed operand or
wrong index (brute force, antisymmetry), self term not excluded (lattice
potential, duplicate-position cases).
"""
import os

import mpmath
import numpy as np
import pytest

from oracle import nbody_oracle as py_oracle
from paper_0707_0438_b200 import inputs

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


@pytest.fixture(params=["numpy", "c"])
def oracle(request, c_oracle):
    return py_oracle if request.param == "numpy" else c_oracle


def _rand(n, seed, scale_v=0.7):
    rng = np.random.default_rng(seed)
    m = rng.uniform(0.2, 1.5, n) / n
    x = rng.standard_normal((n, 3))
    v = scale_v * rng.standard_normal((n, 3))
    return m, x, v


# --- 1. two-body closed form (SURVEY 8(c) pin 1; Eq. 1 L41 with reading R1, R2) ---
@pytest.mark.parametrize("eps", [0.0, 1.0 / 256.0, 0.3])
def test_two_body_closed_form(oracle, eps):
    m = np.array([0.7, 0.3])
    x = np.array([[0.1, -0.2, 0.05], [0.9, 0.4, -0.35]])
    v = np.array([[0.0, 0.3, -0.1], [-0.2, -0.5, 0.25]])
    d = x[1] - x[0]
    u = v[1] - v[0]
    s = d @ d + eps * eps
    a1 = m[1] * d * s ** -1.5
    j1 = m[1] * (u * s ** -1.5 - 3.0 * (d @ u) * d * s ** -2.5)
    p1 = -m[1] * s ** -0.5
    acc, jrk, pot = oracle.force(m, x, v, eps)
    np.testing.assert_allclose(acc[0], a1, rtol=1e-14)
    np.testing.assert_allclose(jrk[0], j1, rtol=1e-13)
    np.testing.assert_allclose(pot[0], p1, rtol=1e-14)
    # particle 2 by antisymmetry: m1 a1 = -m2 a2, same for the jerk
    np.testing.assert_allclose(m[1] * acc[1], -m[0] * acc[0], rtol=1e-14)
    np.testing.assert_allclose(m[1] * jrk[1], -m[0] * jrk[0], rtol=1e-13)
    np.testing.assert_allclose(pot[1], -m[0] * s ** -0.5, rtol=1e-14)
    # attraction: particle 0 is pulled towards particle 1, potential negative
    assert acc[0] @ d > 0 and pot[0] < 0


# --- 2. momentum: sum m a = 0 and sum m jerk = 0 to fp64 round-off (pin 2) ---
@pytest.mark.parametrize("eps", [1.0 / 256.0, 0.05])
def test_momentum_sums_vanish(oracle, eps):
    m, x, v = inputs.plummer(512, 11)
    acc, jrk, _ = oracle.force(m, x, v, eps)
    scale_a = np.sum(m[:, None] * np.abs(acc))
    scale_j = np.sum(m[:, None] * np.abs(jrk))
    assert np.abs((m[:, None] * acc).sum(0)).max() < 1e-13 * scale_a
    assert np.abs((m[:, None] * jrk).sum(0)).max() < 1e-12 * scale_j


# --- 3. symmetric lattice: zero force / jerk at the centre, closed-form potential (pin 3) ---
def test_lattice_centre(oracle):
    g = np.arange(-2, 3, dtype=np.float64)
    pts = np.array([[a, b, c] for a in g for b in g for c in g if (a, b, c) != (0, 0, 0)])
    n = pts.shape[0]
    omega = np.array([0.3, -0.2, 0.5])
    vel = np.cross(omega, pts) + 0.4 * pts  # point-symmetric: v(-x) = -v(x)
    m = np.full(n + 1, 1.0 / (n + 1))
    x = np.vstack([np.zeros((1, 3)), pts])
    v = np.vstack([np.zeros((1, 3)), vel])
    eps = 0.1
    acc, jrk, pot = oracle.force(m, x, v, eps, i_index=np.array([0]))
    assert np.abs(acc).max() < 1e-15 and np.abs(jrk).max() < 1e-15
    expect = -np.sum(m[1:] / np.sqrt((pts ** 2).sum(1) + eps * eps))
    np.testing.assert_allclose(pot[0], expect, rtol=1e-14)


# --- 4. jerk = d(acc)/dt along straight-line motion (pin 4; reading R3) ---
@pytest.mark.parametrize("eps", [0.0, 1.0 / 256.0])
def test_jerk_matches_finite_difference_of_acc(oracle, eps):
    m, x, v = _rand(40, 5)
    _, jrk, _ = oracle.force(m, x, v, eps)
    h = 1e-5
    ap, _, _ = oracle.force(m, x + h * v, v, eps)
    am, _, _ = oracle.force(m, x - h * v, v, eps)
    fd = (ap - am) / (2 * h)
    np.testing.assert_allclose(jrk, fd, rtol=2e-7, atol=1e-8 * np.abs(jrk).max())


# --- 5. acc = -grad_i pot (pin 5; readings R2, R4: same softened s in both sums) ---
@pytest.mark.parametrize("eps", [1.0 / 256.0, 0.2])
def test_acc_is_minus_gradient_of_potential(oracle, eps):
    m, x, v = _rand(30, 6)
    acc, _, _ = oracle.force(m, x, v, eps)
    h = 1e-6
    for i in (0, 7, 29):
        for d in range(3):
            xp, xm = x.copy(), x.copy()
            xp[i, d] += h
            xm[i, d] -= h
            pp = oracle.force(m, xp, v, eps, i_index=np.array([i]))[2][0]
            pm = oracle.force(m, xm, v, eps, i_index=np.array([i]))[2][0]
            assert abs(acc[i, d] + (pp - pm) / (2 * h)) < 1e-8 * max(1.0, abs(acc[i, d]))


# --- 6. invariances and scalings (pin 6) ---
def test_invariances_and_scalings(oracle):
    m, x, v = _rand(64, 7)
    eps = 0.03
    a0, j0, p0 = oracle.force(m, x, v, eps)
    a, j, p = oracle.force(m, x + np.array([3.0, -1.0, 2.0]), v + np.array([0.5, 0.1, -0.7]), eps)
    np.testing.assert_allclose(a, a0, rtol=1e-11, atol=1e-14)
    np.testing.assert_allclose(j, j0, rtol=1e-10, atol=1e-13)
    np.testing.assert_allclose(p, p0, rtol=1e-12)
    a, j, p = oracle.force(2.5 * m, x, v, eps)
    np.testing.assert_allclose(a, 2.5 * a0, rtol=1e-13)
    np.testing.assert_allclose(j, 2.5 * j0, rtol=1e-13, atol=1e-15)
    np.testing.assert_allclose(p, 2.5 * p0, rtol=1e-13)
    lam, mu = 1.7, 0.6
    a, j, p = oracle.force(m, lam * x, mu * v, lam * eps)
    np.testing.assert_allclose(a, a0 / lam ** 2, rtol=1e-12)
    np.testing.assert_allclose(j, mu * j0 / lam ** 3, rtol=1e-11, atol=1e-14)
    np.testing.assert_allclose(p, p0 / lam, rtol=1e-12)


# --- 7. brute force, 50 digits, N <= 48, incl. duplicated positions and eps = 0 (pin 7; R6) ---
def _mp_force(m, x, v, eps, i):
    mpmath.mp.dps = 50
    M = [mpmath.mpf(float(t)) for t in m]
    X = [[mpmath.mpf(float(c)) for c in r] for r in x]
    V = [[mpmath.mpf(float(c)) for c in r] for r in v]
    e2 = mpmath.mpf(float(eps)) ** 2
    a = [mpmath.mpf(0)] * 3
    jk = [mpmath.mpf(0)] * 3
    p = mpmath.mpf(0)
    for j in range(len(M)):
        if j == i:
            continue
        r = [X[j][d] - X[i][d] for d in range(3)]
        w = [V[j][d] - V[i][d] for d in range(3)]
        s = r[0] ** 2 + r[1] ** 2 + r[2] ** 2 + e2
        if e2 == 0 and s == 0:
            continue
        rw = r[0] * w[0] + r[1] * w[1] + r[2] * w[2]
        p -= M[j] / mpmath.sqrt(s)
        for d in range(3):
            a[d] += M[j] * r[d] / s ** mpmath.mpf(1.5)
            jk[d] += M[j] * (w[d] / s ** mpmath.mpf(1.5) - 3 * rw * r[d] / s ** mpmath.mpf(2.5))
    return [float(t) for t in a], [float(t) for t in jk], float(p)


@pytest.mark.parametrize("eps,dup", [(1.0 / 256.0, False), (0.0, False), (1.0 / 256.0, True), (0.0, True)])
def test_brute_force_mpmath(oracle, eps, dup):
    m, x, v = _rand(48, 8)
    if dup:  # particle 5 sits exactly on particle 3 (distinct index, zero distance)
        x[5] = x[3]
    acc, jrk, pot = oracle.force(m, x, v, eps)
    for i in (0, 3, 5, 47):
        a, jk, p = _mp_force(m, x, v, eps, i)
        np.testing.assert_allclose(acc[i], a, rtol=1e-12, atol=1e-15)
        np.testing.assert_allclose(jrk[i], jk, rtol=1e-11, atol=1e-14)
        np.testing.assert_allclose(pot[i], p, rtol=1e-13)
    assert np.isfinite(acc).all() and np.isfinite(jrk).all() and np.isfinite(pot).all()


def test_duplicate_position_softened_adds_only_potential(oracle):
    """R6: for eps > 0 a coincident j != i adds -m_j/eps to pot and nothing to acc, jerk (w != 0 allowed)."""
    m, x, v = _rand(20, 9)
    eps = 1.0 / 256.0
    a0, j0, p0 = oracle.force(m, x, v, eps, i_index=np.array([4]))
    m2 = np.append(m, 0.123)
    x2 = np.vstack([x, x[4]])
    v2 = np.vstack([v, v[4]])  # same velocity: the pair contributes no jerk either
    a1, j1, p1 = oracle.force(m2, x2, v2, eps, i_index=np.array([4]))
    np.testing.assert_allclose(a1, a0, rtol=1e-15)
    np.testing.assert_allclose(j1, j0, rtol=1e-15)
    np.testing.assert_allclose(p1, p0 - 0.123 / eps, rtol=1e-14)


def test_external_test_particle_and_subset(oracle):
    """i_index = -1 is an external test particle (no j excluded); a subset equals rows of the full result."""
    m, x, v = _rand(33, 10)
    eps = 0.01
    full = oracle.force(m, x, v, eps)
    idx = np.array([31, 2, 17])
    sub = oracle.force(m, x, v, eps, i_index=idx)
    for f, s in zip(full, sub):
        np.testing.assert_allclose(s, f[idx], rtol=1e-13)
    xi = np.array([[0.3, 0.1, -0.2]])
    vi = np.array([[0.0, 0.2, 0.1]])
    ext = oracle.force(m, x, v, eps, i_index=np.array([-1]), xi=xi, vi=vi)
    m2, x2, v2 = np.append(m, 0.0), np.vstack([x, xi]), np.vstack([v, vi])
    ref = oracle.force(m2, x2, v2, eps, i_index=np.array([33]))
    for e, r in zip(ext, ref):
        np.testing.assert_allclose(e, r, rtol=1e-13)


# --- 8. continuum check: radial acceleration ~ -M(r)/r^2 for the Plummer model (pin 8, loose) ---
def test_plummer_continuum_profile(c_oracle):
    m, x, v = inputs.plummer(8192, 12)
    idx = np.arange(0, 8192, 8)
    acc, _, pot = c_oracle.force(m, x, v, 0.0, i_index=idx, want_jerk=False)
    r = np.sqrt((x[idx] ** 2).sum(1))
    b = 3 * np.pi / 16
    a_rad = np.einsum("ij,ij->i", acc, x[idx]) / r
    model = -(r ** 3 / (r * r + b * b) ** 1.5) / (r * r)
    sel = (r > 0.3) & (r < 3.0)
    assert abs(np.median(a_rad[sel] / model[sel]) - 1.0) < 0.05
    phi_model = -1.0 / np.sqrt(r * r + b * b)
    assert abs(np.median(pot[sel] / phi_model[sel]) - 1.0) < 0.05


# --- 9. predictor (pin 9; reading R8) ---
def test_predictor_exact_on_cubic_and_identity_at_dt0(oracle):
    rng = np.random.default_rng(3)
    n = 17
    x0, v0, a0, j0 = (rng.standard_normal((n, 3)) for _ in range(4))
    tj = rng.uniform(0.0, 0.5, n)
    t = 0.75
    dt = (t - tj)[:, None]
    xs = x0 + dt * (v0 + dt * (a0 / 2 + dt * j0 / 6))  # Horner form of the same cubic
    vs = v0 + dt * (a0 + dt * j0 / 2)
    xp, vp = oracle.predict(t, tj, x0, v0, a0, j0)
    np.testing.assert_allclose(xp, xs, rtol=1e-14, atol=1e-15)
    np.testing.assert_allclose(vp, vs, rtol=1e-14, atol=1e-15)
    xp, vp = oracle.predict(0.25, np.full(n, 0.25), x0, v0, a0, j0)
    assert np.array_equal(xp, x0) and np.array_equal(vp, v0)
    # derivative consistency: d x_p / dt = v_p
    h = 1e-6
    xa, _ = oracle.predict(t + h, tj, x0, v0, a0, j0)
    xb, _ = oracle.predict(t - h, tj, x0, v0, a0, j0)
    _, vm = oracle.predict(t, tj, x0, v0, a0, j0)
    np.testing.assert_allclose((xa - xb) / (2 * h), vm, rtol=1e-8, atol=1e-9)


# --- numpy form == C form on a Plummer input (two independent writings of the definition) ---
def test_numpy_and_c_forms_agree(c_oracle):
    m, x, v = inputs.plummer_f32(1024, 1)
    idx = inputs.active_block(1024, 100, 1)
    for eps in (0.0, inputs.EPS_PAPER):
        a, j, p = py_oracle.force(m, x, v, eps, i_index=idx)
        a2, j2, p2 = c_oracle.force(m, x, v, eps, i_index=idx)
        np.testing.assert_allclose(a2, a, rtol=1e-12, atol=1e-14)
        np.testing.assert_allclose(j2, j, rtol=1e-10, atol=1e-11)
        np.testing.assert_allclose(p2, p, rtol=1e-13)


# --- energy and the paper's reporting conventions ---
def test_plummer_energy_is_minus_quarter():
    """N-body units: E = -1/4 in expectation; virial ratio 2T/|W| ~ 1 (pin 17)."""
    m, x, v = inputs.plummer(2048, 13)
    e = py_oracle.energy(m, x, v, 0.0)
    kin = 0.5 * np.sum(m * (v ** 2).sum(1))
    assert abs(e + 0.25) < 0.02
    assert abs(2 * kin / (kin - e) - 1.0) < 0.08
    assert py_oracle.relative_energy_error(-0.25, -0.25 * (1 + 1e-6)) == pytest.approx(-1e-6, rel=1e-6)


@pytest.mark.parametrize("fname,k", [("paper_table4_force_pot_jerk.txt", 60), ("paper_table3_force_only.txt", 38)])
def test_flop_convention_reproduces_paper_tables(fname, k):
    """Eq. 3 (L178) with the printed times reproduces the printed GFLOP/s (Tables 3, 4) to print precision."""
    rows = np.loadtxt(os.path.join(GOLDEN, fname))
    for n, t, gf in rows:
        got = py_oracle.flops_per_second(k, n, n, t) / 1e9
        # times are printed to 2-7 significant digits (worst case 0.000090 s: half a unit in the last
        # place is 0.6 %; the printed speed deviates by up to 0.8 % from the printed time)
        assert abs(got / gf - 1.0) < 0.01, (n, got, gf)


# --- nearest neighbour (reading R20) -----------------------------------------
def test_nearest_neighbour_on_a_line_and_lattice(oracle):
    """Closed cases: points on a line at 0, 1, 3, 7, 15 (gaps double) => nn = 1, 0, 1, 2, 3;
    a simple cubic lattice => every nearest distance is the spacing, and ties go to the lowest index."""
    x = np.zeros((5, 3))
    x[:, 0] = [0.0, 1.0, 3.0, 7.0, 15.0]
    nn, r2 = oracle.nearest_neighbour(x)
    assert list(nn) == [1, 0, 1, 2, 3]
    assert np.allclose(r2, [1.0, 1.0, 4.0, 16.0, 64.0], rtol=0, atol=0)
    g = np.arange(4.0)
    lat = np.array([[a, b, c] for a in g for b in g for c in g]) * 0.5      # index = 16a + 4b + c
    nn, r2 = oracle.nearest_neighbour(lat)
    assert np.all(r2 == 0.25)
    for i, (a, b, c) in enumerate([(a, b, c) for a in range(4) for b in range(4) for c in range(4)]):
        cand = [16 * aa + 4 * bb + cc for aa, bb, cc in
                [(a - 1, b, c), (a, b - 1, c), (a, b, c - 1), (a, b, c + 1), (a, b + 1, c), (a + 1, b, c)]
                if 0 <= aa < 4 and 0 <= bb < 4 and 0 <= cc < 4]
        assert nn[i] == min(cand)


def test_nearest_neighbour_brute_force_subset_external_and_degenerate(oracle):
    rng = np.random.default_rng(12)
    x = rng.standard_normal((57, 3))
    idx = np.array([5, 56, 0, 33])
    nn, r2 = oracle.nearest_neighbour(x, i_index=idx)
    for k, i in enumerate(idx):
        best, bj = None, -1
        for j in range(57):
            if j == i:
                continue
            d = sum((x[j, c] - x[i, c]) ** 2 for c in range(3))
            if best is None or d < best:
                best, bj = d, j
        assert nn[k] == bj and abs(r2[k] - best) <= 1e-15 * best
    # external particle: nothing excluded; a j at the same place is the neighbour at distance 0
    nn, r2 = oracle.nearest_neighbour(x, i_index=np.array([-1]), xi=x[7:8])
    assert nn[0] == 7 and r2[0] == 0.0
    # mutual pairs: the closest pair of the set are each other's neighbours
    nn, r2 = oracle.nearest_neighbour(x)
    i = int(np.argmin(r2))
    assert nn[nn[i]] == i
    # translation invariance of the index, and a lone particle has none
    nn2, _ = oracle.nearest_neighbour(x + 3.0)
    assert np.array_equal(nn, nn2)
    nn1, r1 = oracle.nearest_neighbour(x[:1])
    assert nn1[0] == -1 and np.isinf(r1[0])


# --- the numpy form's i-chunk loop (more than _CHUNK_ELEMS pair temporaries): several chunks ---
def test_numpy_form_across_i_chunks():
    """n_i * N > 4 M pairs makes nbody_oracle.force walk several i-chunks.  Pins that a chunk's rows
    land in the right slots: momentum sums over ALL i vanish (a shifted or dropped chunk breaks the
    pairwise cancellation), and the rows on both sides of every chunk boundary equal a scalar loop
    written from the definition (Eq. 1)."""
    n = 3000
    m, x, v = _rand(n, 77)
    eps = 1.0 / 256.0
    chunk = py_oracle._CHUNK_ELEMS // n
    assert n > 2 * chunk                      # three chunks
    acc, jrk, pot = py_oracle.force(m, x, v, eps)
    assert np.abs((m[:, None] * acc).sum(0)).max() < 1e-13 * np.sum(m[:, None] * np.abs(acc))
    assert np.abs((m[:, None] * jrk).sum(0)).max() < 1e-12 * np.sum(m[:, None] * np.abs(jrk))
    for i in (0, chunk - 1, chunk, 2 * chunk - 1, 2 * chunk, n - 1):
        a, jk, p = np.zeros(3), np.zeros(3), 0.0
        for j in range(n):
            if j == i:
                continue
            r, w = x[j] - x[i], v[j] - v[i]
            s = r @ r + eps * eps
            a += m[j] * r * s ** -1.5
            jk += m[j] * (w * s ** -1.5 - 3.0 * (r @ w) * r * s ** -2.5)
            p -= m[j] * s ** -0.5
        np.testing.assert_allclose(acc[i], a, rtol=1e-11)
        np.testing.assert_allclose(jrk[i], jk, rtol=1e-10, atol=1e-12 * np.abs(jk).max())
        np.testing.assert_allclose(pot[i], p, rtol=1e-12)
    # an i-subset that straddles a chunk boundary of its own (n_i = 1500 > chunk) with a permutation
    idx = np.random.default_rng(3).permutation(n)[:1500]
    acc_s, jrk_s, pot_s = py_oracle.force(m, x, v, eps, i_index=idx)
    np.testing.assert_array_equal(acc_s, acc[idx])
    np.testing.assert_array_equal(pot_s, pot[idx])
