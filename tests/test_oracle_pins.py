"""Pins for the CPU oracle (oracle/nbody_oracle.c): each test checks it against something the paper
or the mathematics fixes *independently of the oracle's own formula* -- closed forms, exact rational
brute force written separately, invariances, energy integrals, special limits.  A plausible mistake
(dropped term, wrong sign or index, eps vs eps^2, transposed operand, wrong half-kick) fails at least
one of them.  CPU only.

Pin numbering follows SURVEY.md section 8.1.3 (P1..P12).
"""
import math
import os
from fractions import Fraction

import mpmath
import numpy as np
import pytest

import oracle
from paper_astro_ph_0703100_b200 import workloads as wl

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _one(xi, xj, mj, eps2):
    acc, pot = oracle.force(np.asarray(xi, dtype=np.float64).reshape(-1, 3),
                            np.asarray(xj, dtype=np.float64).reshape(-1, 3),
                            np.asarray(mj, dtype=np.float64).reshape(-1), eps2)
    return acc, pot


# ----------------------------------------------------------------------------- P1
def _golden_rows():
    rows = []
    with open(os.path.join(GOLDEN, "two_body_exact.txt")) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            rows.append([Fraction(tok) for tok in line.split()])
    return rows


@pytest.mark.parametrize("row", _golden_rows())
@pytest.mark.parametrize("offset", [(0.0, 0.0, 0.0), (0.5, -2.0, 4.0)])
def test_p1_two_body_exact_rationals(row, offset):
    """Eq. (1): a = m d / (d.d + eps2)^(3/2), phi = -m / (d.d + eps2)^(1/2), exact cases."""
    dx, dy, dz, eps2, m, s = row
    assert dx * dx + dy * dy + dz * dz + eps2 == s * s      # the fixture row is self-consistent
    o = np.array(offset)
    xi = o
    xj = o + np.array([float(dx), float(dy), float(dz)])
    acc, pot = _one(xi, xj, [float(m)], float(eps2))
    want_a = [float(m * d / s ** 3) for d in (dx, dy, dz)]
    want_p = float(-m / s)
    np.testing.assert_allclose(acc[0], want_a, rtol=4e-16, atol=0)
    np.testing.assert_allclose(pot[0], want_p, rtol=4e-16, atol=0)
    # and the reaction on j from i is equal and opposite per unit mass product
    acc_j, pot_j = _one(xj, xi, [float(m)], float(eps2))
    np.testing.assert_allclose(acc_j[0], [-a for a in want_a], rtol=4e-16, atol=0)
    np.testing.assert_allclose(pot_j[0], want_p, rtol=4e-16, atol=0)


def test_p1_eps2_is_epsilon_squared_not_epsilon():
    """the argument is eps2.  d = (3,0,0): eps2 = 16 -> r = 5; eps = 16 would give r = sqrt(265)."""
    acc, pot = _one([0, 0, 0], [3, 0, 0], [1.0], 16.0)
    assert acc[0, 0] == pytest.approx(3.0 / 125.0, rel=1e-15)
    assert pot[0] == pytest.approx(-0.2, rel=1e-15)


# ----------------------------------------------------------------------------- P2
def test_p2_coincident_pairs_contribute_nothing():
    # same point, any eps (including 0): a = 0, phi = 0, no NaN
    for eps2 in (0.0, 1e-4, 1.0):
        acc, pot = _one([1.5, -2.0, 0.25], [1.5, -2.0, 0.25], [3.0], eps2)
        assert np.all(acc == 0.0) and pot[0] == 0.0
    # duplicated j-particles at the i position are all skipped; a distinct one is not
    xj = np.array([[1, 1, 1], [1, 1, 1], [4, 1, 1]], dtype=np.float64)
    acc, pot = _one([1, 1, 1], xj, [5.0, 7.0, 2.0], 16.0)
    np.testing.assert_allclose(acc[0], [2.0 * 3.0 / 125.0, 0, 0], rtol=1e-15)
    assert pot[0] == pytest.approx(-2.0 / 5.0, rel=1e-15)


def test_p2_subset_each_i_skips_exactly_its_own_copy():
    """C2 shape: i = subset of j.  phi_masked = phi_unmasked + m_i/eps, and the unmasked sum is obtained
    here by moving the i-particle's own copy out of the j-set and adding the self term by hand."""
    w = wl.subset_workload(512, 16, 1.0 / 128, seed=11)
    xj = w.x_j.astype(np.float64)
    mj = w.m_j.astype(np.float64)
    eps2 = float(w.eps2)
    acc, pot = oracle.force(xj[w.i_index], xj, mj, eps2)
    for k, idx in enumerate(w.i_index):
        keep = np.ones(len(xj), dtype=bool)
        keep[idx] = False
        a2, p2 = oracle.force(xj[idx:idx + 1], xj[keep], mj[keep], eps2)
        np.testing.assert_allclose(acc[k], a2[0], rtol=1e-13)
        assert pot[k] == pytest.approx(p2[0], rel=1e-13)


# ----------------------------------------------------------------------------- P3
@pytest.mark.parametrize("seed", [0, 5])
def test_p3_momentum_antisymmetry(seed):
    rng = np.random.default_rng(seed)
    n = 257
    x = rng.normal(size=(n, 3))
    m = rng.uniform(0.1, 2.0, size=n)
    acc, _ = oracle.force(x, x, m, 1e-3)
    net = np.linalg.norm((m[:, None] * acc).sum(axis=0))
    scale = (m * np.linalg.norm(acc, axis=1)).sum()
    assert net <= 1e-13 * scale


# ----------------------------------------------------------------------------- P4
def test_p4_axis_permutation_and_sign_flip_exact():
    rng = np.random.default_rng(1)
    n = 64
    x = rng.normal(size=(n, 3))
    m = rng.uniform(0.5, 1.5, size=n)
    acc, pot = oracle.force(x, x, m, 0.01)
    perm = [2, 0, 1]
    sign = np.array([1.0, -1.0, -1.0])
    x2 = x[:, perm] * sign
    acc2, pot2 = oracle.force(x2, x2, m, 0.01)
    # d.d is summed in a different order after a permutation, so allow rounding-level differences
    np.testing.assert_allclose(acc2, acc[:, perm] * sign, rtol=1e-12, atol=1e-15)
    np.testing.assert_allclose(pot2, pot, rtol=1e-13)
    # pure sign flip: bitwise equal
    x3 = x * sign
    acc3, pot3 = oracle.force(x3, x3, m, 0.01)
    assert np.array_equal(acc3, acc * sign) and np.array_equal(pot3, pot)


def test_p4_translation_exact_on_dyadic_grid():
    rng = np.random.default_rng(2)
    n = 48
    x = rng.integers(-512, 512, size=(n, 3)).astype(np.float64) / 64.0   # dyadic grid
    m = rng.integers(1, 16, size=n).astype(np.float64) / 16.0
    acc, pot = oracle.force(x, x, m, 2.0 ** -8)
    shift = np.array([1024.0, -256.0, 4096.0])
    acc2, pot2 = oracle.force(x + shift, x + shift, m, 2.0 ** -8)
    assert np.array_equal(acc, acc2) and np.array_equal(pot, pot2)


def test_p4_general_rotation_and_translation():
    rng = np.random.default_rng(3)
    n = 100
    x = rng.normal(size=(n, 3))
    m = rng.uniform(0.5, 1.5, size=n)
    q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
    t = np.array([0.3, -1.7, 2.2])
    acc, pot = oracle.force(x, x, m, 0.02)
    x2 = x @ q.T + t
    acc2, pot2 = oracle.force(x2, x2, m, 0.02)
    np.testing.assert_allclose(acc2, acc @ q.T, rtol=0, atol=1e-12 * np.abs(acc).max())
    np.testing.assert_allclose(pot2, pot, rtol=1e-12)


# ----------------------------------------------------------------------------- P5
def _plummer_truncated_W():
    """W_T = -(1/M_T^2) int_0^10 M(r) M'(r) / r dr for M(r) = r^3 (1+r^2)^(-3/2), by quadrature (mpmath)."""
    M = lambda r: r ** 3 * (1 + r * r) ** mpmath.mpf(-1.5)
    dM = lambda r: 3 * r * r * (1 + r * r) ** mpmath.mpf(-2.5)
    integral = mpmath.quad(lambda r: M(r) * dM(r) / r, [0, 1, 10])
    return float(-integral / M(mpmath.mpf(10)) ** 2)


def test_p5_plummer_potential_energy_closed_form():
    """Untruncated Plummer: W = -3 pi G M^2 / (32 a) (BASELINE.json north_star).  The configs truncate at
    10a and keep m = 1/N, which gives W_T = -0.302443 by the integral above; softening adds ~ +0.138 eps^2."""
    assert _plummer_truncated_W() == pytest.approx(-0.302443, abs=2e-6)
    # the untruncated limit of the same integral is -3 pi / 32
    M = lambda r: r ** 3 * (1 + r * r) ** mpmath.mpf(-1.5)
    dM = lambda r: 3 * r * r * (1 + r * r) ** mpmath.mpf(-2.5)
    w_inf = -mpmath.quad(lambda r: M(r) * dM(r) / r, [0, 1, 10, mpmath.inf])
    assert float(w_inf) == pytest.approx(-3 * math.pi / 32, rel=1e-10)

    n = 8192
    vals = []
    for seed in (100, 101, 102):
        w = wl.plummer_workload(n, 1.0 / 256, seed=seed)
        _, pot = oracle.force(w.x_j, w.x_j, w.m_j, w.eps2)
        vals.append(0.5 * float(np.sum(w.m_j.astype(np.float64) * pot)))
    expect = _plummer_truncated_W() * (1.0 - 1.0 / n) + 0.138 * float(w.eps2)
    sigma = 0.5 / math.sqrt(n) * abs(expect)
    for v in vals:
        assert abs(v - expect) <= 3.0 * sigma, (v, expect)
    assert abs(np.mean(vals) - expect) <= 3.0 * sigma / math.sqrt(len(vals))


# ----------------------------------------------------------------------------- P6
def _brute_force_mp(xi, xj, mj, eps2):
    """Independent evaluator: exact rational differences and r^2, 50-digit square root; loops over
    components outermost -- a different structure from the oracle on purpose."""
    mpmath.mp.dps = 50
    n_i, n_j = len(xi), len(xj)
    out_a = [[mpmath.mpf(0)] * 3 for _ in range(n_i)]
    out_p = [mpmath.mpf(0)] * n_i
    for i in range(n_i):
        for j in range(n_j):
            d = [Fraction(float(xj[j][c])) - Fraction(float(xi[i][c])) for c in range(3)]
            if all(c == 0 for c in d):
                continue
            r2 = sum(c * c for c in d) + Fraction(float(eps2))
            r = mpmath.sqrt(mpmath.mpf(r2.numerator) / mpmath.mpf(r2.denominator))
            mm = mpmath.mpf(float(mj[j]))
            out_p[i] -= mm / r
            for c in range(3):
                out_a[i][c] += mm * (mpmath.mpf(d[c].numerator) / mpmath.mpf(d[c].denominator)) / r ** 3
    return (np.array([[float(v) for v in row] for row in out_a]), np.array([float(v) for v in out_p]))


@pytest.mark.parametrize("n,eps2,seed", [(2, 0.0, 0), (3, 0.25, 1), (5, 1e-3, 2), (8, 0.0, 3), (8, 1.0 / 4096, 4)])
def test_p6_brute_force_small_n(n, eps2, seed):
    rng = np.random.default_rng(seed)
    x = rng.normal(size=(n, 3))
    m = rng.uniform(0.1, 3.0, size=n)
    acc, pot = oracle.force(x, x, m, eps2)
    ref_a, ref_p = _brute_force_mp(x, x, m, eps2)
    np.testing.assert_allclose(acc, ref_a, rtol=1e-13, atol=1e-13 * np.abs(ref_a).max())
    np.testing.assert_allclose(pot, ref_p, rtol=1e-13)


def test_p6_brute_force_separate_i_and_j_sets_float32_entry():
    rng = np.random.default_rng(9)
    xi = rng.normal(size=(3, 3)).astype(np.float32)
    xj = rng.normal(size=(7, 3)).astype(np.float32)
    mj = rng.uniform(0.1, 3.0, size=7).astype(np.float32)
    xj[2] = xi[1]                                    # one coincident pair
    eps2 = np.float32(1.0 / 1024)
    acc, pot = oracle.force(xi, xj, mj, eps2)
    ref_a, ref_p = _brute_force_mp(xi, xj, mj, eps2)
    np.testing.assert_allclose(acc, ref_a, rtol=1e-13, atol=1e-13 * np.abs(ref_a).max())
    np.testing.assert_allclose(pot, ref_p, rtol=1e-13)


# ----------------------------------------------------------------------------- P7
def test_p7_uniform_sphere_energy_and_radial_field():
    """Uniform ball radius R, masses independent of position: E[1/r12] = 6/(5R), so
    E[W] = -(3/5) (1 - sum m_i^2) / R; and the mean radial acceleration at radius r is -M r / R^3."""
    n = 8192
    vals, expects = [], []
    for seed in (200, 201, 202):
        w = wl.uniform_sphere_workload(n, 1.0 / 1024, seed=seed)
        m = w.m_j.astype(np.float64)
        acc, pot = oracle.force(w.x_j, w.x_j, w.m_j, w.eps2)
        vals.append(0.5 * float(np.sum(m * pot)))
        expects.append(-0.6 * (1.0 - float(np.sum(m * m))))
    for v, e in zip(vals, expects):
        assert abs(v / e - 1.0) < 0.03, (v, e)
    assert abs(np.mean(vals) / np.mean(expects) - 1.0) < 0.02
    # radial field (last seed): regress a_r on r over the bulk
    x = w.x_j.astype(np.float64)
    r = np.linalg.norm(x, axis=1)
    a_r = np.einsum("ij,ij->i", acc, x) / r
    sel = (r > 0.3) & (r < 0.95)
    slope = np.sum(a_r[sel] * r[sel]) / np.sum(r[sel] ** 2)
    assert slope == pytest.approx(-1.0, abs=0.05)


# ----------------------------------------------------------------------------- P8
def test_p8_large_softening_limit():
    rng = np.random.default_rng(4)
    n = 200
    x = rng.uniform(-1, 1, size=(n, 3))
    m = rng.uniform(0.5, 1.5, size=n)
    eps2 = 1e6 * 12.0
    eps = math.sqrt(eps2)
    acc, pot = oracle.force(x, x, m, eps2)
    M = m.sum()
    # the i-particle skips itself: exclude its own mass from the monopole
    for i in (0, 17, n - 1):
        Mi = M - m[i]
        xcm = (m[:, None] * x).sum(axis=0) - m[i] * x[i]
        want = (xcm - Mi * x[i]) / eps ** 3
        np.testing.assert_allclose(acc[i], want, rtol=1e-5)
        assert pot[i] == pytest.approx(-Mi / eps, rel=1e-6)


# ----------------------------------------------------------------------------- P9
def test_p9_regular_figures():
    s, m, eps2 = 2.0, 1.5, 0.25
    tri = np.array([[0, 0, 0], [s, 0, 0], [s / 2, s * math.sqrt(3) / 2, 0]])
    acc, pot = oracle.force(tri, tri, np.full(3, m), eps2)
    centroid = tri.mean(axis=0)
    mag = math.sqrt(3) * m * s / (s * s + eps2) ** 1.5
    for i in range(3):
        assert np.linalg.norm(acc[i]) == pytest.approx(mag, rel=1e-14)
        to_c = centroid - tri[i]
        cosang = np.dot(acc[i], to_c) / (np.linalg.norm(acc[i]) * np.linalg.norm(to_c))
        assert cosang == pytest.approx(1.0, abs=1e-14)
        assert pot[i] == pytest.approx(-2 * m / math.sqrt(s * s + eps2), rel=1e-14)
    # probe at the centre of a cube of equal masses feels nothing; phi = -8 m / sqrt(3 h^2 + eps2)
    h = 1.0
    cube = np.array([[sx, sy, sz] for sx in (-h, h) for sy in (-h, h) for sz in (-h, h)], dtype=np.float64)
    acc, pot = oracle.force(np.zeros((1, 3)), cube, np.full(8, m), eps2)
    assert np.all(np.abs(acc) <= 1e-16)
    assert pot[0] == pytest.approx(-8 * m / math.sqrt(3 * h * h + eps2), rel=1e-15)


# ----------------------------------------------------------------------------- P12 (leapfrog)
def _binary(d=1.0, m=0.5, eps2=0.01):
    x = np.array([[-d / 2, 0, 0], [d / 2, 0, 0]], dtype=np.float64)
    speed = math.sqrt(m * d * d / (2.0 * (d * d + eps2) ** 1.5))
    v = np.array([[0, -speed, 0], [0, speed, 0]], dtype=np.float64)
    omega = math.sqrt(2.0 * m / (d * d + eps2) ** 1.5)
    return x, v, np.array([m, m]), omega


def _energy64(x, v, m, eps2):
    _, pot = oracle.force(x, x, m, eps2)
    return 0.5 * np.sum(m * np.sum(v * v, axis=1)) + 0.5 * np.sum(m * pot)


def test_p12_softened_circular_binary_stays_circular():
    eps2 = 0.01
    x, v, m, omega = _binary(eps2=eps2)
    period = 2 * math.pi / omega
    n_steps = 2000
    dt = period / n_steps
    e0 = _energy64(x, v, m, eps2)
    x1, v1, _, _ = oracle.leapfrog_kdk(x, v, m, eps2, dt, n_steps)
    # after one period the bodies are back (phase error O(dt^2)), radius preserved
    assert np.linalg.norm(x1[0]) == pytest.approx(0.5, rel=1e-5)
    np.testing.assert_allclose(x1, x, atol=2e-5)
    assert abs(_energy64(x1, v1, m, eps2) - e0) <= 1e-9 * abs(e0)
    # momentum conserved to round-off
    assert np.linalg.norm((m[:, None] * v1).sum(axis=0)) <= 1e-15


def test_p12_dt_squared_convergence():
    """Second order: the phase error after a fixed time scales as dt^2 (halving dt divides it by ~4)."""
    eps2 = 0.01
    x, v, m, omega = _binary(eps2=eps2)
    period = 2 * math.pi / omega

    def phase_error(n_steps):
        x1, _, _, _ = oracle.leapfrog_kdk(x, v, m, eps2, period / n_steps, n_steps)
        return np.linalg.norm(x1 - x)

    e_coarse, e_fine = phase_error(100), phase_error(200)
    assert 3.6 < e_coarse / e_fine < 4.4

    # eccentric orbit: the energy error at a fixed time also scales as dt^2
    v_ecc = v * 0.6
    e0 = _energy64(x, v_ecc, m, eps2)

    def energy_error(n_steps):
        x1, v1, _, _ = oracle.leapfrog_kdk(x, v_ecc, m, eps2, 1.0 / n_steps, n_steps)
        return abs(_energy64(x1, v1, m, eps2) - e0)

    r = energy_error(64) / energy_error(128)
    assert 3.0 < r < 5.0


def test_p12_time_reversal():
    rng = np.random.default_rng(7)
    n = 16
    x = rng.normal(size=(n, 3))
    v = 0.3 * rng.normal(size=(n, 3))
    m = rng.uniform(0.5, 1.5, size=n) / n
    eps2, dt, steps = 0.05, 1.0 / 64, 50
    x1, v1, _, _ = oracle.leapfrog_kdk(x, v, m, eps2, dt, steps)
    x2, v2, _, _ = oracle.leapfrog_kdk(x1, -v1, m, eps2, dt, steps)
    np.testing.assert_allclose(x2, x, atol=1e-11)
    np.testing.assert_allclose(-v2, v, atol=1e-11)


def test_p12_single_step_by_hand():
    """One KDK step written out with numpy from forces of the (pinned) force oracle: pins the half-kick
    placement and that dt (not dt/2, not dt^2) multiplies v in the drift."""
    rng = np.random.default_rng(8)
    n = 5
    x = rng.normal(size=(n, 3))
    v = rng.normal(size=(n, 3))
    m = rng.uniform(0.5, 1.5, size=n)
    eps2, dt = 0.1, 0.03125
    a0, _ = oracle.force(x, x, m, eps2)
    vh = v + a0 * (dt / 2)
    xn = x + vh * dt
    a1, p1 = oracle.force(xn, xn, m, eps2)
    vn = vh + a1 * (dt / 2)
    x1, v1, acc1, pot1 = oracle.leapfrog_kdk(x, v, m, eps2, dt, 1)
    np.testing.assert_allclose(x1, xn, rtol=1e-15, atol=1e-15)
    np.testing.assert_allclose(v1, vn, rtol=1e-15, atol=1e-15)
    np.testing.assert_allclose(acc1, a1, rtol=1e-15)
    np.testing.assert_allclose(pot1, p1, rtol=1e-15)
    # zero steps: state untouched, a and phi of the initial state returned
    x0, v0, acc0, _ = oracle.leapfrog_kdk(x, v, m, eps2, dt, 0)
    assert np.array_equal(x0, x) and np.array_equal(v0, v)
    np.testing.assert_allclose(acc0, a0, rtol=1e-15)


def test_energy_entry_matches_hand_sum():
    w = wl.plummer_workload(300, 1.0 / 64, seed=5, with_velocities=True)
    T, W, E = oracle.energy(w.x_j, w.v, w.m_j, w.eps2)
    m = w.m_j.astype(np.float64)
    _, pot = oracle.force(w.x_j, w.x_j, w.m_j, w.eps2)
    assert T == pytest.approx(0.5 * np.sum(m * np.sum(w.v.astype(np.float64) ** 2, axis=1)), rel=1e-14)
    assert W == pytest.approx(0.5 * np.sum(m * pot), rel=1e-14)
    assert E == pytest.approx(T + W, rel=1e-15)


def test_edge_sizes():
    x = np.zeros((0, 3))
    acc, pot = oracle.force(x, np.ones((4, 3)), np.ones(4), 0.1)
    assert acc.shape == (0, 3) and pot.shape == (0,)
    acc, pot = oracle.force(np.ones((3, 3)), x, np.zeros(0), 0.1)
    assert np.all(acc == 0) and np.all(pot == 0)
    with pytest.raises(ValueError):
        oracle.force(np.ones((1, 3)), np.ones((1, 3)), np.ones(1), -1.0)


def test_error_metric_eq3():
    """Eq. (3), on a case worked by hand."""
    ref = np.array([[3.0, 4.0, 0.0], [0.0, 0.0, 2.0]])
    tst = np.array([[3.0, 4.0, 0.5], [0.0, 0.0, 2.0]])
    e = oracle.error_metrics(tst, ref, np.array([-1.0, -2.2]), np.array([-1.0, -2.0]))
    assert e["acc_max"] == pytest.approx(0.1)
    assert e["acc_rms"] == pytest.approx(0.1 / math.sqrt(2))
    assert e["pot_max"] == pytest.approx(0.1)


def test_f2_batched_entry_is_one_force_call_per_sub_problem():
    """oracle.force_batched against the mpmath brute force, sub-problem by sub-problem (tiny), incl. empty ones."""
    rng = np.random.default_rng(4)
    x_i = rng.normal(size=(7, 3)); x_j = rng.normal(size=(12, 3)); m_j = rng.uniform(0.5, 1.5, 12)
    x_j[2] = x_i[1]                                   # a coincident pair inside sub-problem 0
    i_off = np.array([0, 3, 3, 6]); j_off = np.array([0, 5, 9, 12])
    acc, pot = oracle.force_batched(i_off, j_off, x_i, x_j, m_j, 0.01)
    for b in range(3):
        i0, i1, j0, j1 = i_off[b], i_off[b + 1], j_off[b], j_off[b + 1]
        if i1 > i0:
            ra, rp = _brute_force_mp(x_i[i0:i1], x_j[j0:j1], m_j[j0:j1], 0.01)
            np.testing.assert_allclose(acc[i0:i1], ra, rtol=1e-13, atol=1e-15)
            np.testing.assert_allclose(pot[i0:i1], rp, rtol=1e-13)
    assert not acc[6].any() and pot[6] == 0.0         # outside every sub-problem


# ----------------------------------------------------------------------------- row f3: eps2 per i-particle
def test_f3_constant_array_reproduces_the_scalar_entry_bitwise():
    rng = np.random.default_rng(11)
    x = rng.normal(size=(60, 3)); m = rng.uniform(0.5, 1.5, 60)
    a0, p0 = oracle.force(x[:17], x, m, 0.03)
    a1, p1 = oracle.force_eps_i(x[:17], np.full(17, 0.03), x, m)
    assert np.array_equal(a0, a1) and np.array_equal(p0, p1)


def test_f3_two_body_exact_with_a_different_eps2_per_i():
    """Golden rows (d, eps2, m, s) of two_body_exact.txt, all i-particles in ONE call, each with its own eps2."""
    rows = _golden_rows()
    xj = np.array([[10.0, -20.0, 5.0]])                       # one j-particle; i-particle k sits at xj - d_k
    xi = np.array([[10.0 - float(r[0]), -20.0 - float(r[1]), 5.0 - float(r[2])] for r in rows])
    e2 = np.array([float(r[3]) for r in rows])
    m = float(rows[0][4])
    acc, pot = oracle.force_eps_i(xi, e2, xj, np.array([m]))
    for k, r in enumerate(rows):
        d, s = r[:3], r[5]
        exact = [float(Fraction(m) * c / s ** 3) for c in d]
        np.testing.assert_allclose(acc[k], exact, rtol=1e-14, atol=1e-17)
        assert pot[k] == pytest.approx(float(-Fraction(m) / s), rel=1e-14)


def test_f3_brute_force_random_eps2_per_i():
    rng = np.random.default_rng(12)
    x = rng.normal(size=(7, 3)); m = rng.uniform(0.5, 1.5, 7)
    e2 = np.array([0.0, 1e-4, 0.01, 0.25, 1.0, 0.0, 3.0])
    acc, pot = oracle.force_eps_i(x, e2, x, m)
    for i in range(7):
        ra, rp = _brute_force_mp(x[i:i + 1], x, m, e2[i])
        np.testing.assert_allclose(acc[i], ra[0], rtol=1e-13, atol=1e-15)
        np.testing.assert_allclose(pot[i], rp[0], rtol=1e-13)
    with pytest.raises(ValueError):
        oracle.force_eps_i(x, -e2 - 1.0, x, m)


# ----------------------------------------------------------------------------- P13: a = -grad(phi), Gauss, Newton
def test_p13_acceleration_is_minus_the_gradient_of_the_potential():
    """Eq. (1) and the potential of Fig. A.4 must be consistent: a_i = -d phi / d r_i for a probe (an i-particle that
    is not in the j-set).  Central differences of the oracle's OWN phi, Richardson-extrapolated."""
    rng = np.random.default_rng(21)
    xj = rng.normal(size=(50, 3)); mj = rng.uniform(0.5, 1.5, 50)
    probes = rng.normal(size=(6, 3)) * 1.5
    for eps2 in (0.0, 0.05):
        acc, _ = oracle.force(probes, xj, mj, eps2)
        grad = np.zeros_like(acc)
        for c in range(3):
            for h, wgt in ((1e-3, 4.0 / 3.0), (2e-3, -1.0 / 3.0)):
                e = np.zeros(3); e[c] = h
                _, pp = oracle.force(probes + e, xj, mj, eps2)
                _, pm = oracle.force(probes - e, xj, mj, eps2)
                grad[:, c] += wgt * (pp - pm) / (2 * h)
        np.testing.assert_allclose(acc, -grad, rtol=2e-7, atol=1e-9)


def test_p13_newton_shell_theorem_and_gauss_flux():
    """A thin spherical shell of mass M (many equal points on a sphere of radius R, eps = 0): no force inside,
    M / r^2 toward the centre outside; phi = -M / R inside (Newton's theorems, to the sampling error of the shell)."""
    n, R, M = 20000, 1.0, 1.0
    k = np.arange(n) + 0.5                                   # Fibonacci sphere: quasi-uniform points
    z = 1 - 2 * k / n; phi = np.pi * (1 + 5 ** 0.5) * k
    shell = R * np.stack([np.sqrt(1 - z * z) * np.cos(phi), np.sqrt(1 - z * z) * np.sin(phi), z], 1)
    m = np.full(n, M / n)
    inside = np.array([[0.0, 0.0, 0.0], [0.3, -0.2, 0.1], [0.0, 0.5, 0.0]])
    outside = np.array([[2.0, 0.0, 0.0], [0.0, -3.0, 4.0]])
    a_in, p_in = oracle.force(inside, shell, m, 0.0)
    a_out, p_out = oracle.force(outside, shell, m, 0.0)
    assert np.abs(a_in).max() < 2e-4 and np.abs(p_in + M / R).max() < 1e-5
    r = np.linalg.norm(outside, axis=1)
    np.testing.assert_allclose(a_out, -M * outside / r[:, None] ** 3, rtol=1e-5, atol=1e-6)
    np.testing.assert_allclose(p_out, -M / r, rtol=1e-6)


def test_p13_mass_linearity_and_superposition():
    rng = np.random.default_rng(22)
    xi = rng.normal(size=(9, 3)); xj = rng.normal(size=(40, 3)); mj = rng.uniform(0.5, 1.5, 40)
    a, p = oracle.force(xi, xj, mj, 0.02)
    a2, p2 = oracle.force(xi, xj, 3.5 * mj, 0.02)
    np.testing.assert_allclose(a2, 3.5 * a, rtol=1e-14); np.testing.assert_allclose(p2, 3.5 * p, rtol=1e-14)
    aa, pa = oracle.force(xi, xj[:17], mj[:17], 0.02)
    ab, pb = oracle.force(xi, xj[17:], mj[17:], 0.02)
    np.testing.assert_allclose(aa + ab, a, rtol=1e-13, atol=1e-15); np.testing.assert_allclose(pa + pb, p, rtol=1e-13)
    perm = rng.permutation(40)                               # the order of the j-particles does not matter (to rounding)
    a3, p3 = oracle.force(xi, xj[perm], mj[perm], 0.02)
    np.testing.assert_allclose(a3, a, rtol=1e-13, atol=1e-15); np.testing.assert_allclose(p3, p, rtol=1e-13)


# ----------------------------------------------------------------------------- lj (row f3, reading R19)
def _lj_rows(x, sigma, eps):
    x = np.asarray(x, dtype=np.float64).reshape(-1, 3)
    n = x.shape[0]
    return np.concatenate([x, np.broadcast_to(np.asarray(sigma, dtype=np.float64) / 2.0, (n,)).reshape(n, 1),
                           np.sqrt(np.broadcast_to(np.asarray(eps, dtype=np.float64), (n,))).reshape(n, 1)], axis=1)


def test_lj_two_body_closed_forms():
    """12-6 Lennard-Jones, one pair on the x-axis: zero force and U = -eps at the minimum r = 2^(1/6) sigma; U = 0 and a
    repulsion of 24 eps / sigma at r = sigma; at r = 2 sigma the exact rationals U = 4 eps (2^-12 - 2^-6) and
    |F| = 24 eps (2^-6 - 2^-11) / (2 sigma), attractive.  The force is the one ON the i-particle."""
    sigma, eps = 1.5, 0.7
    i = _lj_rows([[0.0, 0.0, 0.0]], sigma, eps)
    for r, f_expect, u_expect in (
            (2.0 ** (1.0 / 6.0) * sigma, 0.0, -eps),
            (sigma, -24.0 * eps / sigma, 0.0),                                  # pushed away from j: toward -x
            (2.0 * sigma, float(Fraction(24) * Fraction(7, 10) * (Fraction(1, 64) - Fraction(2, 4096)) / 3), None)):
        out = oracle.lennard_jones(i, _lj_rows([[r, 0.0, 0.0]], sigma, eps))
        assert abs(out[0, 0] - f_expect) <= 1e-13 * max(1.0, abs(f_expect)), (r, out)
        assert out[0, 1] == 0.0 and out[0, 2] == 0.0
        if u_expect is not None:
            assert abs(out[0, 3] - u_expect) <= 1e-14
    u2 = oracle.lennard_jones(i, _lj_rows([[0.0, 0.0, -2.0 * sigma]], sigma, eps))
    assert abs(u2[0, 3] - 4 * eps * (2.0 ** -12 - 2.0 ** -6)) <= 1e-16
    assert u2[0, 2] < 0.0 and u2[0, 0] == 0.0                                   # attracted toward j at -z


def test_lj_mixing_rule_third_law_and_coincident_pairs():
    rng = np.random.default_rng(31)
    n = 40
    x = rng.uniform(0.0, 6.0, (n, 3))
    sig = rng.uniform(0.8, 1.2, n); eps = rng.uniform(0.5, 2.0, n)
    rows = _lj_rows(x, sig, eps)
    out = oracle.lennard_jones(rows, rows)                                     # the self pair adds nothing (R1)
    assert np.all(np.isfinite(out))
    # Lorentz-Berthelot: the pair (a, b) is a single-species pair with sigma = (sig_a + sig_b) / 2, eps = sqrt(eps_a eps_b)
    a, b = 3, 17
    pair = oracle.lennard_jones(rows[a:a + 1], rows[b:b + 1])
    s, e = 0.5 * (sig[a] + sig[b]), math.sqrt(eps[a] * eps[b])
    same = oracle.lennard_jones(_lj_rows(x[a], s, e), _lj_rows(x[b], s, e))
    np.testing.assert_allclose(pair, same, rtol=1e-14)
    # Newton's third law: the forces of a closed system sum to zero; U is symmetric, so sum_i U_i = 2 E_total
    scale = np.abs(out[:, :3]).sum()
    assert np.abs(out[:, :3].sum(axis=0)).max() <= 1e-13 * scale
    # a duplicate of particle 0 elsewhere in the j-list: skipped for i = 0, felt by everybody else
    rows2 = np.concatenate([rows, rows[:1]])
    out2 = oracle.lennard_jones(rows, rows2)
    np.testing.assert_array_equal(out2[0], out[0])
    assert np.all(out2[1:, 3] != out[1:, 3])


def test_lj_force_is_minus_gradient_of_total_energy_and_python_loop():
    rng = np.random.default_rng(32)
    n = 12
    g = np.stack(np.meshgrid(*[np.arange(3.0)] * 3, indexing="ij"), -1).reshape(-1, 3)[:n] * 1.3
    x = g + rng.uniform(-0.1, 0.1, (n, 3))
    sig = rng.uniform(0.9, 1.1, n); eps = rng.uniform(0.5, 1.5, n)

    def energy(xx):
        r = _lj_rows(xx, sig, eps)
        return 0.5 * oracle.lennard_jones(r, r)[:, 3].sum()

    out = oracle.lennard_jones(_lj_rows(x, sig, eps), _lj_rows(x, sig, eps))
    h = 1e-5
    for i in (0, 5, 11):
        for c in range(3):
            xp, xm = x.copy(), x.copy()
            xp[i, c] += h; xm[i, c] -= h
            np.testing.assert_allclose(out[i, c], -(energy(xp) - energy(xm)) / (2 * h), rtol=2e-7, atol=1e-8)
    # the definition written out as a pure-Python double loop (F on i points from j to i when repulsive)
    for i in range(n):
        f = [0.0, 0.0, 0.0]; u = 0.0
        for j in range(n):
            if j == i:
                continue
            d = [x[i][c] - x[j][c] for c in range(3)]
            r = math.sqrt(sum(v * v for v in d))
            s = 0.5 * (sig[i] + sig[j]); e = math.sqrt(eps[i] * eps[j])
            dudr = 4 * e * (-12 * s ** 12 / r ** 13 + 6 * s ** 6 / r ** 7)
            for c in range(3):
                f[c] += -dudr * d[c] / r
            u += 4 * e * ((s / r) ** 12 - (s / r) ** 6)
        np.testing.assert_allclose(out[i, :3], f, rtol=1e-11, atol=1e-12)
        assert abs(out[i, 3] - u) <= 1e-12 * max(1.0, abs(u))
