"""Pins of the force + jerk + potential oracle (row f1; Fig. A.4) -- CPU only.

Each pin is independent of oracle_force_jerk's own arithmetic: exact rationals worked from the
statements of Fig. A.4, the time derivative of the separately pinned acceleration oracle, an
arbitrary-precision brute force written from the textbook formula, and invariances.
"""
import os
from fractions import Fraction

import mpmath
import numpy as np
import pytest

import oracle

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "hermite_two_body_exact.txt")


def _rows():
    rows = []
    with open(GOLDEN) as f:
        for line in f:
            line = line.strip()
            if line and not line.startswith("#"):
                rows.append(tuple(Fraction(t) for t in line.split()))
    return rows


@pytest.mark.parametrize("row", _rows())
def test_h1_two_body_exact_rationals(row):
    dx, dy, dz, ux, uy, uz, eps2, m, s = row
    assert dx * dx + dy * dy + dz * dz + eps2 == s * s              # the fixture is self-consistent
    d, dv = (dx, dy, dz), (ux, uy, uz)
    ddv = sum(a * b for a, b in zip(d, dv))
    a_exact = [m * c / s ** 3 for c in d]
    j_exact = [m * w / s ** 3 - 3 * m * ddv * c / s ** 5 for c, w in zip(d, dv)]
    for off, voff in (((0, 0, 0), (0, 0, 0)), ((1.5, -2.0, 0.25), (0.5, 0.25, -1.0))):
        xi = np.array([off], dtype=np.float64); vi = np.array([voff], dtype=np.float64)
        xj = xi + np.array([[float(c) for c in d]]); vj = vi + np.array([[float(c) for c in dv]])
        acc, jerk, pot = oracle.force_jerk(xi, vi, xj, vj, np.array([float(m)]), float(eps2))
        np.testing.assert_allclose(acc[0], [float(c) for c in a_exact], rtol=1e-15, atol=1e-18)
        np.testing.assert_allclose(jerk[0], [float(c) for c in j_exact], rtol=4e-15, atol=1e-17)
        assert pot[0] == pytest.approx(float(-m / s), rel=1e-15)


def _random_system(n, seed, dtype=np.float64):
    rng = np.random.default_rng(seed)
    x = rng.normal(size=(n, 3)).astype(dtype)
    v = rng.normal(size=(n, 3)).astype(dtype)
    m = rng.uniform(0.5, 1.5, n).astype(dtype)
    return x, v, m


@pytest.mark.parametrize("seed,eps2", [(0, 0.01), (1, 0.0), (2, 1.0)])
def test_h2_jerk_is_the_time_derivative_of_the_pinned_acceleration(seed, eps2):
    """jerk_i = d a_i / dt along x(t) = x + v t: central difference of oracle.force (pinned by test_oracle_pins)."""
    x, v, m = _random_system(40, seed)
    xi, vi = x[:13] + 0.0, v[:13] + 0.0                  # i-set is a subset: exercises the coincident rule too
    acc, jerk, pot = oracle.force_jerk(xi, vi, x, v, m, eps2)
    a0, p0 = oracle.force(xi, x, m, eps2)
    np.testing.assert_allclose(acc, a0, rtol=1e-14, atol=1e-15)       # same a and phi as the force-only oracle
    np.testing.assert_allclose(pot, p0, rtol=1e-14)
    h = 1e-4
    ap, _ = oracle.force(xi + h * vi, x + h * v, m, eps2)
    am, _ = oracle.force(xi - h * vi, x - h * v, m, eps2)
    fd = (ap - am) / (2 * h)
    scale = np.linalg.norm(jerk, axis=1).max()
    assert np.abs(fd - jerk).max() <= 3e-6 * scale                    # O(h^2) truncation + 1e-16/h roundoff
    # Richardson: the error shrinks 4x when h halves -> it is truncation of the right derivative, not a wrong term
    h2 = 2e-4
    ap2, _ = oracle.force(xi + h2 * vi, x + h2 * v, m, eps2)
    am2, _ = oracle.force(xi - h2 * vi, x - h2 * v, m, eps2)
    rich = (4 * fd - (ap2 - am2) / (2 * h2)) / 3
    assert np.abs(rich - jerk).max() <= 2e-9 * scale


def _brute_mp(xi, vi, xj, vj, mj, eps2):
    """Independent evaluator: mpmath, 40 digits, textbook formula d/dt [m d / r^3] -- not the Fig. A.4 statement order."""
    mpmath.mp.dps = 40
    out_a, out_j, out_p = [], [], []
    for a in range(len(xi)):
        A = [mpmath.mpf(0)] * 3; J = [mpmath.mpf(0)] * 3; P = mpmath.mpf(0)
        for b in range(len(xj)):
            d = [mpmath.mpf(float(xj[b][c])) - mpmath.mpf(float(xi[a][c])) for c in range(3)]
            if all(c == 0 for c in d):
                continue
            w = [mpmath.mpf(float(vj[b][c])) - mpmath.mpf(float(vi[a][c])) for c in range(3)]
            r = mpmath.sqrt(sum(c * c for c in d) + mpmath.mpf(float(eps2)))
            rdot = sum(c * e for c, e in zip(d, w)) / r                # d r / dt
            mm = mpmath.mpf(float(mj[b]))
            for c in range(3):
                A[c] += mm * d[c] / r ** 3
                J[c] += mm * (w[c] / r ** 3 - 3 * d[c] * rdot / r ** 4)
            P -= mm / r
        out_a.append([float(c) for c in A]); out_j.append([float(c) for c in J]); out_p.append(float(P))
    return np.array(out_a), np.array(out_j), np.array(out_p)


@pytest.mark.parametrize("n,eps2,seed", [(2, 0.0, 0), (3, 0.25, 1), (6, 1e-4, 2), (5, 0.0, 3)])
def test_h3_brute_force_small_n(n, eps2, seed):
    x, v, m = _random_system(n, seed)
    acc, jerk, pot = oracle.force_jerk(x, v, x, v, m, eps2)
    ra, rj, rp = _brute_mp(x, v, x, v, m, eps2)
    np.testing.assert_allclose(acc, ra, rtol=1e-13, atol=1e-15)
    np.testing.assert_allclose(jerk, rj, rtol=1e-12, atol=1e-14)
    np.testing.assert_allclose(pot, rp, rtol=1e-13)


def test_h3_float32_entry_promotes_exactly():
    x, v, m = _random_system(7, 5, np.float32)
    xi, vi = x[:3].copy(), v[:3].copy() + np.float32(0.5)             # same positions, other velocities: still coincident
    acc, jerk, pot = oracle.force_jerk(xi, vi, x, v, m, np.float32(0.01))
    ra, rj, rp = _brute_mp(xi, vi, x, v, m, np.float32(0.01))
    np.testing.assert_allclose(acc, ra, rtol=1e-13, atol=1e-15)
    np.testing.assert_allclose(jerk, rj, rtol=1e-12, atol=1e-14)
    np.testing.assert_allclose(pot, rp, rtol=1e-13)


def test_h4_momentum_antisymmetry_and_galilean_invariance():
    x, v, m = _random_system(200, 7)
    acc, jerk, pot = oracle.force_jerk(x, v, x, v, m, 0.01)
    for arr in (acc, jerk):                                           # sum_i m_i jerk_i = d/dt sum m a = 0
        tot = (m[:, None] * arr).sum(0)
        assert np.linalg.norm(tot) <= 1e-13 * (m[:, None] * np.abs(arr)).sum()
    boost = np.array([3.0, -1.0, 0.5])
    acc2, jerk2, pot2 = oracle.force_jerk(x, v + boost, x, v + boost, m, 0.01)
    np.testing.assert_allclose(jerk2, jerk, rtol=1e-11, atol=1e-12)   # only velocity differences enter
    np.testing.assert_array_equal(acc2, acc)
    # rotation: vectors rotate with the frame
    q, _ = np.linalg.qr(np.random.default_rng(1).normal(size=(3, 3)))
    acc3, jerk3, pot3 = oracle.force_jerk(x @ q.T, v @ q.T, x @ q.T, v @ q.T, m, 0.01)
    np.testing.assert_allclose(jerk3, jerk @ q.T, rtol=1e-10, atol=1e-11)
    np.testing.assert_allclose(pot3, pot, rtol=1e-12)
    # velocity scaling: jerk is linear in the velocities, a does not depend on them
    acc4, jerk4, _ = oracle.force_jerk(x, 2.5 * v, x, 2.5 * v, m, 0.01)
    np.testing.assert_allclose(jerk4, 2.5 * jerk, rtol=1e-12, atol=1e-13)
    np.testing.assert_array_equal(acc4, acc)


def test_h5_circular_binary_jerk_is_omega_cross_a():
    """On a circular orbit a rotates rigidly: jerk = omega x a, |jerk| = omega |a|."""
    d, m, eps2 = 1.0, 0.5, 0.01
    w2 = 2 * m / (d * d + eps2) ** 1.5
    x = np.array([[-d / 2, 0, 0], [d / 2, 0, 0]]); mm = np.array([m, m])
    vorb = np.sqrt(w2) * d / 2
    v = np.array([[0, -vorb, 0], [0, vorb, 0]])
    acc, jerk, _ = oracle.force_jerk(x, v, x, v, mm, eps2)
    omega = np.array([0, 0, np.sqrt(w2)])
    np.testing.assert_allclose(jerk, np.cross(omega, acc), rtol=1e-13, atol=1e-15)


def test_h6_edge_sizes_and_coincidence():
    z3 = np.zeros((0, 3)); z1 = np.zeros(0)
    x, v, m = _random_system(4, 9)
    a, j, p = oracle.force_jerk(x, v, z3, z3, z1, 0.1)
    assert not a.any() and not j.any() and not p.any()
    a, j, p = oracle.force_jerk(z3, z3, x, v, m, 0.1)
    assert a.shape == (0, 3) and j.shape == (0, 3)
    one = np.array([[1.0, 2.0, 3.0]])
    a, j, p = oracle.force_jerk(one, np.array([[1.0, 0, 0]]), one, np.array([[0, 5.0, 0]]), np.array([2.0]), 0.0)
    assert not a.any() and not j.any() and p[0] == 0.0               # coincident in position: nothing, even at eps2 = 0


# ----------------------------------------------------------------------------- h7: the Hermite integrator
def _three_body():
    x = np.array([[1.0, 0.0, 0.0], [-0.5, 0.8, 0.1], [-0.4, -0.9, -0.2]])
    v = np.array([[0.0, 0.4, 0.1], [-0.35, -0.2, 0.0], [0.3, -0.15, -0.1]])
    m = np.array([1.0, 0.8, 1.2])
    return x, v, m


def _energy3(x, v, m, eps2):
    t = 0.5 * (m * (v * v).sum(1)).sum()
    w = 0.0
    for a in range(len(m)):
        for b in range(a + 1, len(m)):
            w -= m[a] * m[b] / np.sqrt(((x[a] - x[b]) ** 2).sum() + eps2)
    return t + w


def test_h7_hermite_matches_an_adaptive_high_order_solver_and_is_fourth_order():
    from scipy.integrate import solve_ivp
    x0, v0, m = _three_body()
    eps2, T = 0.01, 1.0

    def rhs(t, y):
        x, v = y[:9].reshape(3, 3), y[9:].reshape(3, 3)
        a = np.zeros((3, 3))
        for p in range(3):
            for q in range(3):
                if p != q:
                    d = x[q] - x[p]
                    a[p] += m[q] * d / (d @ d + eps2) ** 1.5
        return np.concatenate([v.ravel(), a.ravel()])

    sol = solve_ivp(rhs, (0.0, T), np.concatenate([x0.ravel(), v0.ravel()]), method="DOP853", rtol=1e-13, atol=1e-14)
    x_ref, v_ref = sol.y[:9, -1].reshape(3, 3), sol.y[9:, -1].reshape(3, 3)
    errs = []
    for steps in (32, 64, 128):
        x, v, _, _, _ = oracle.hermite4(x0, v0, m, eps2, T / steps, steps)
        errs.append(max(np.abs(x - x_ref).max(), np.abs(v - v_ref).max()))
    assert errs[2] < 2e-7
    assert 11.0 < errs[0] / errs[1] < 22.0 and 11.0 < errs[1] / errs[2] < 22.0       # error ~ dt^4


def test_h7_hermite_energy_error_far_below_leapfrog_and_outputs_are_the_carried_values():
    x0, v0, m = _three_body()
    eps2, dt, steps = 0.01, 1.0 / 64, 64
    e0 = _energy3(x0, v0, m, eps2)
    xh, vh, ah, jh, ph = oracle.hermite4(x0, v0, m, eps2, dt, steps)
    xl, vl, _, _ = oracle.leapfrog_kdk(x0, v0, m, eps2, dt, steps)
    err_h, err_l = abs(_energy3(xh, vh, m, eps2) - e0), abs(_energy3(xl, vl, m, eps2) - e0)
    assert err_h < 1e-7 and err_h < 0.02 * err_l
    tot = (m[:, None] * vh).sum(0) - (m[:, None] * v0).sum(0)
    assert np.abs(tot).max() < 1e-14                                              # momentum
    # zero steps: just the evaluation
    x, v, a, j, p = oracle.hermite4(x0, v0, m, eps2, dt, 0)
    ra, rj, rp = oracle.force_jerk(x0, v0, x0, v0, m, eps2)
    assert np.array_equal(x, x0) and np.array_equal(a, ra) and np.array_equal(j, rj) and np.array_equal(p, rp)


# ----------------------------------------------------------------------------- h8: one block step (individual time steps)
def _block_run(x0, v0, m, eps2, T, base_steps, slow, ratio):
    """Two-level block schedule: particles in ``slow`` step with ratio * dt, the others with dt = T / base_steps."""
    n = len(m)
    x, v = x0.copy(), v0.copy()
    a, j, _ = oracle.force_jerk(x, v, x, v, m, eps2)
    t = np.zeros(n)
    fast = np.array([k for k in range(n) if k not in slow], dtype=np.int32)
    everybody = np.arange(n, dtype=np.int32)
    dt = T / base_steps
    for s in range(1, base_steps + 1):
        active = everybody if s % ratio == 0 else fast
        x, v, a, j, t = oracle.hermite4_block_step(x, v, m, a, j, t, active, s * dt, eps2)
    assert np.all(t == T)
    return x, v


def test_h8_all_active_at_equal_times_is_one_shared_step():
    x0, v0, m = _random_system(17, 5)
    eps2, dt = 0.02, 1.0 / 32
    a0, j0, _ = oracle.force_jerk(x0, v0, x0, v0, m, eps2)
    x, v, a, j, t = oracle.hermite4_block_step(x0, v0, m, a0, j0, np.full(17, 0.25), np.arange(17), 0.25 + dt, eps2)
    xr, vr, ar, jr, _ = oracle.hermite4(x0, v0, m, eps2, dt, 1)                    # pinned by h7
    for got, ref in ((x, xr), (v, vr), (a, ar), (j, jr)):
        np.testing.assert_allclose(got, ref, rtol=1e-14, atol=1e-15)
    assert np.all(t == 0.25 + dt)
    # the order in which the active particles are listed does not matter
    perm = np.random.default_rng(0).permutation(17)
    x2, v2, a2, j2, _ = oracle.hermite4_block_step(x0, v0, m, a0, j0, np.full(17, 0.25), perm, 0.25 + dt, eps2)
    assert np.array_equal(x2, x) and np.array_equal(v2, v) and np.array_equal(a2, a) and np.array_equal(j2, j)


def test_h8_inactive_particles_are_untouched_and_empty_active_set_is_a_no_op():
    x0, v0, m = _random_system(12, 6)
    eps2 = 0.01
    a0, j0, _ = oracle.force_jerk(x0, v0, x0, v0, m, eps2)
    t0 = np.linspace(0.0, 0.05, 12)
    active = np.array([7, 2, 9], dtype=np.int32)
    x, v, a, j, t = oracle.hermite4_block_step(x0, v0, m, a0, j0, t0, active, 0.0625, eps2)
    rest = np.setdiff1d(np.arange(12), active)
    for got, ref in ((x, x0), (v, v0), (a, a0), (j, j0), (t, t0)):
        assert np.array_equal(got[rest], ref[rest])
        assert not np.array_equal(got[active], ref[active])
    assert np.all(t[active] == 0.0625)
    out = oracle.hermite4_block_step(x0, v0, m, a0, j0, t0, np.zeros(0, dtype=np.int32), 0.0625, eps2)
    for got, ref in zip(out, (x0, v0, a0, j0, t0)):
        assert np.array_equal(got, ref)
    with pytest.raises(ValueError):
        oracle.hermite4_block_step(x0, v0, m, a0, j0, t0, np.array([3, 3]), 0.0625, eps2)
    with pytest.raises(ValueError):
        oracle.hermite4_block_step(x0, v0, m, a0, j0, t0, np.array([12]), 0.0625, eps2)


def test_h8_pure_python_restatement_of_one_block_step():
    """Independent evaluator: textbook formulas in Python floats with math.fsum, own pair loop, own indexing."""
    import math
    x0, v0, m = _random_system(6, 7)
    eps2, t_now = 0.03, 0.125
    a0, j0, _ = oracle.force_jerk(x0, v0, x0, v0, m, eps2)
    t0 = np.array([0.0, 0.0625, 0.09375, 0.0, 0.0625, 0.109375])
    active = [4, 0, 5]
    got = oracle.hermite4_block_step(x0, v0, m, a0, j0, t0, np.array(active), t_now, eps2)
    xp, vp = [], []
    for k in range(6):
        h = t_now - t0[k]
        xp.append([math.fsum([x0[k][c], v0[k][c] * h, a0[k][c] * h * h / 2, j0[k][c] * h ** 3 / 6]) for c in range(3)])
        vp.append([math.fsum([v0[k][c], a0[k][c] * h, j0[k][c] * h * h / 2]) for c in range(3)])
    for i in active:
        h = t_now - t0[i]
        a1, j1 = [[], [], []], [[], [], []]
        for q in range(6):
            if q == i:
                continue
            d = [xp[q][c] - xp[i][c] for c in range(3)]
            w = [vp[q][c] - vp[i][c] for c in range(3)]
            r2 = math.fsum([d[0] ** 2, d[1] ** 2, d[2] ** 2, eps2])
            rv = math.fsum([d[c] * w[c] for c in range(3)])
            for c in range(3):
                a1[c].append(m[q] * d[c] / r2 ** 1.5)
                j1[c].append(m[q] * (w[c] / r2 ** 1.5 - 3 * rv * d[c] / r2 ** 2.5))
        for c in range(3):
            an, jn = math.fsum(a1[c]), math.fsum(j1[c])
            vn = math.fsum([v0[i][c], (a0[i][c] + an) * h / 2, (j0[i][c] - jn) * h * h / 12])
            xn = math.fsum([x0[i][c], (v0[i][c] + vn) * h / 2, (a0[i][c] - an) * h * h / 12])
            assert got[0][i][c] == pytest.approx(xn, rel=1e-13, abs=1e-15)
            assert got[1][i][c] == pytest.approx(vn, rel=1e-13, abs=1e-15)
            assert got[2][i][c] == pytest.approx(an, rel=1e-13, abs=1e-15)
            assert got[3][i][c] == pytest.approx(jn, rel=1e-12, abs=1e-14)


def test_h8_two_level_schedule_matches_an_adaptive_solver_and_is_fourth_order():
    """Particle 0 steps with 2 dt, particles 1 and 2 with dt: at every odd sub-step particle 0 enters only through its
    prediction from a stale state.  A missing or mis-timed prediction leaves a first- or second-order error."""
    from scipy.integrate import solve_ivp
    x0, v0, m = _three_body()
    eps2, T = 0.01, 1.0

    def rhs(t, y):
        x, v = y[:9].reshape(3, 3), y[9:].reshape(3, 3)
        a = np.zeros((3, 3))
        for p in range(3):
            for q in range(3):
                if p != q:
                    d = x[q] - x[p]
                    a[p] += m[q] * d / (d @ d + eps2) ** 1.5
        return np.concatenate([v.ravel(), a.ravel()])

    sol = solve_ivp(rhs, (0.0, T), np.concatenate([x0.ravel(), v0.ravel()]), method="DOP853", rtol=1e-13, atol=1e-14)
    x_ref, v_ref = sol.y[:9, -1].reshape(3, 3), sol.y[9:, -1].reshape(3, 3)
    errs = []
    for steps in (64, 128, 256):
        x, v = _block_run(x0, v0, m, eps2, T, steps, slow={0}, ratio=2)
        errs.append(max(np.abs(x - x_ref).max(), np.abs(v - v_ref).max()))
    assert errs[2] < 1e-7
    assert 10.0 < errs[0] / errs[1] < 24.0 and 10.0 < errs[1] / errs[2] < 24.0       # error ~ dt^4
    # and the block scheme's result differs from the shared-step one (the schedule really is two-level)
    xs, _, _, _, _ = oracle.hermite4(x0, v0, m, eps2, T / 64, 64)
    xb, _ = _block_run(x0, v0, m, eps2, T, 64, slow={0}, ratio=2)
    assert np.abs(xs - xb).max() > 1e-9


# ----------------------------------------------------------------------------- h9: the block-step scheduler
def test_h9_block_schedule_hand_worked_cases():
    t = np.array([0.0, 0.5, 0.25, 0.0, 0.75])
    dt = np.array([1.0, 0.25, 0.5, 0.5, 0.125])
    # due times: 1.0, 0.75, 0.75, 0.5, 0.875  ->  particle 3 alone at 0.5
    t_next, active = oracle.block_schedule(t, dt)
    assert t_next == 0.5 and active.dtype == np.int32 and active.tolist() == [3]
    # after particle 3 has stepped to 0.5 with dt 0.25, three particles tie at 0.75, listed in ascending order
    t[3] = 0.5; dt[3] = 0.25
    t_next, active = oracle.block_schedule(t, dt)
    assert t_next == 0.75 and active.tolist() == [1, 2, 3]
    # negative times, a single particle, everybody due, nobody there
    assert oracle.block_schedule(np.array([-2.0, -1.5]), np.array([0.25, 0.5]))[1].tolist() == [0]
    assert oracle.block_schedule(np.array([3.0]), np.array([0.125])) == (3.125, np.array([0], dtype=np.int32))
    t_next, active = oracle.block_schedule(np.full(7, 1.0), np.full(7, 0.5))
    assert t_next == 1.5 and active.tolist() == list(range(7))
    t_next, active = oracle.block_schedule(np.zeros(0), np.zeros(0))
    assert t_next == float("inf") and active.size == 0


def test_h9_block_schedule_against_a_python_loop():
    rng = np.random.default_rng(9)
    for n in (1, 2, 33, 500):
        level = rng.integers(0, 5, n)
        dt = 2.0 ** -(3 + level)
        t = dt * rng.integers(0, 4, n)                                   # clocks on each particle's own dyadic grid
        t_next, active = oracle.block_schedule(t, dt)
        best, who = None, []
        for k in range(n):
            due = float(t[k]) + float(dt[k])
            if best is None or due < best:
                best, who = due, [k]
            elif due == best:
                who.append(k)
        assert t_next == best and active.tolist() == who


# ----------------------------------------------------------------------------- h10: the step-size criterion
def test_h10_cubic_acceleration_is_interpolated_exactly():
    """a(t) = c0 + c1 t + c2 t^2 + c3 t^3 with small integer coefficients and h = 2: every FP32 operation of the
    interpolation is exact, so dt must be the criterion evaluated on the true derivatives at t + h."""
    rng = np.random.default_rng(10)
    c = rng.integers(-4, 5, size=(4, 50, 3)).astype(np.float64)
    c[3][c[3] == 0] = 1.0
    t0, h = 1.0, 2.0
    def acc(t): return c[0] + c[1] * t + c[2] * t ** 2 + c[3] * t ** 3
    def jerk(t): return c[1] + 2 * c[2] * t + 3 * c[3] * t ** 2
    a0, j0, a1, j1 = acc(t0), jerk(t0), acc(t0 + h), jerk(t0 + h)
    a2 = 2 * c[2] + 6 * c[3] * (t0 + h)
    a3 = 6 * c[3]
    nrm = lambda z: np.sqrt((z * z).sum(1))
    eta = 0.02
    want = np.sqrt(eta * (nrm(a1) * nrm(a2) + nrm(j1) ** 2) / (nrm(j1) * nrm(a3) + nrm(a2) ** 2))
    got = oracle.block_step_size(a0, j0, a1, j1, np.full(50, h), eta)
    assert got.dtype == np.float32
    np.testing.assert_allclose(got, want, rtol=1e-6)


def test_h10_circular_orbit_gives_sqrt_eta_over_omega():
    """r(t) on a circle of radius R with angular speed w: |a| = R w^2, |j| = R w^3, |a2| = R w^4, |a3| = R w^5, so the
    criterion is sqrt(eta) / w whatever R; the interpolated derivatives carry an O((w h)^2) error."""
    eta = 0.01
    errs = []
    for h in (0.25, 0.125):
        w_, R = 1.5, 2.0
        def state(t):
            cs, sn = np.cos(w_ * t), np.sin(w_ * t)
            a = -R * w_ ** 2 * np.array([[cs, sn, 0.0]])
            j = -R * w_ ** 3 * np.array([[-sn, cs, 0.0]])
            return a, j
        a0, j0 = state(0.3)
        a1, j1 = state(0.3 + h)
        got = float(oracle.block_step_size(a0, j0, a1, j1, np.array([h]), eta)[0])
        errs.append(abs(got * w_ / np.sqrt(eta) - 1.0))
    assert errs[1] < 5e-3 and 3.0 < errs[0] / errs[1] < 5.0


def test_h10_scaling_laws():
    """dt scales with sqrt(eta); rescaling time by s (a -> a/s^2, j -> j/s^3, h -> s h) rescales dt by s."""
    rng = np.random.default_rng(11)
    a0, j0 = rng.normal(size=(30, 3)), rng.normal(size=(30, 3))
    a1, j1 = a0 + 0.1 * rng.normal(size=(30, 3)), j0 + 0.1 * rng.normal(size=(30, 3))
    h = np.full(30, 0.125)
    d1 = oracle.block_step_size(a0, j0, a1, j1, h, 0.01)
    d4 = oracle.block_step_size(a0, j0, a1, j1, h, 0.04)
    np.testing.assert_allclose(d4, 2 * d1, rtol=1e-6)
    ds = oracle.block_step_size(a0 / 4, j0 / 8, a1 / 4, j1 / 8, 2 * h, 0.01)        # s = 2: powers of two, exact
    np.testing.assert_array_equal(ds, 2 * d1)


# ----------------------------------------------------------------------------- h10 (FP64): the plain definition
def test_h10_f64_cubic_circular_scaling_and_agreement_with_the_fp32_definition():
    """oracle.block_step_size_f64 is the Aarseth formula in plain FP64.  Same pins as the FP32 definition, tighter:
    a cubic a(t) is interpolated exactly (1e-13), the circular orbit gives sqrt(eta)/omega with an O((omega h)^2)
    error that falls 4x per halving, dt scales with sqrt(eta) and with a rescaling of time -- and the two definitions
    agree to FP32 rounding on FP32 inputs (they are the same formula, so a dropped term in either shows here)."""
    rng = np.random.default_rng(10)
    c = rng.integers(-4, 5, size=(4, 50, 3)).astype(np.float64)
    c[3][c[3] == 0] = 1.0
    t0, h = 0.7, 0.3                                   # nothing dyadic: FP64 carries it anyway
    acc = lambda t: c[0] + c[1] * t + c[2] * t ** 2 + c[3] * t ** 3
    jerk = lambda t: c[1] + 2 * c[2] * t + 3 * c[3] * t ** 2
    a2 = 2 * c[2] + 6 * c[3] * (t0 + h)
    a3 = 6 * c[3]
    nrm = lambda z: np.sqrt((z * z).sum(1))
    eta = 0.02
    want = np.sqrt(eta * (nrm(acc(t0 + h)) * nrm(a2) + nrm(jerk(t0 + h)) ** 2) / (nrm(jerk(t0 + h)) * nrm(a3) + nrm(a2) ** 2))
    got = oracle.block_step_size_f64(acc(t0), jerk(t0), acc(t0 + h), jerk(t0 + h), np.full(50, h), eta)
    assert got.dtype == np.float64
    np.testing.assert_allclose(got, want, rtol=1e-11)
    # circular orbit
    errs = []
    for hh in (0.25, 0.125, 0.0625):
        w_, R = 1.5, 2.0
        def state(t):
            cs, sn = np.cos(w_ * t), np.sin(w_ * t)
            return -R * w_ ** 2 * np.array([[cs, sn, 0.0]]), -R * w_ ** 3 * np.array([[-sn, cs, 0.0]])
        a0, j0 = state(0.3)
        a1, j1 = state(0.3 + hh)
        errs.append(abs(float(oracle.block_step_size_f64(a0, j0, a1, j1, np.array([hh]), 0.01)[0]) * w_ / 0.1 - 1.0))
    assert errs[2] < 1.5e-3 and 3.5 < errs[0] / errs[1] < 4.5 and 3.5 < errs[1] / errs[2] < 4.5
    # scaling laws
    a0, j0 = rng.normal(size=(30, 3)), rng.normal(size=(30, 3))
    a1, j1 = a0 + 0.1 * rng.normal(size=(30, 3)), j0 + 0.1 * rng.normal(size=(30, 3))
    hs = np.full(30, 0.125)
    d1 = oracle.block_step_size_f64(a0, j0, a1, j1, hs, 0.01)
    np.testing.assert_allclose(oracle.block_step_size_f64(a0, j0, a1, j1, hs, 0.04), 2 * d1, rtol=1e-14)
    np.testing.assert_allclose(oracle.block_step_size_f64(a0 / 9, j0 / 27, a1 / 9, j1 / 27, 3 * hs, 0.01), 3 * d1, rtol=1e-12)
    # the FP32 definition on the same (FP32) inputs: same formula, FP32 rounding apart
    f = [z.astype(np.float32) for z in (a0, j0, a1, j1)]
    d32 = oracle.block_step_size(*f, hs.astype(np.float32), 0.01)
    d64 = oracle.block_step_size_f64(*f, hs.astype(np.float32), np.float32(0.01))
    np.testing.assert_allclose(d32, d64, rtol=2e-5)


def test_h9_non_finite_due_times_take_no_part():
    """Reading R20 / include/nbody_b200.h: a due time that is not finite is never the minimum and never due -- dt = +inf
    parks a particle, a NaN or -inf clock cannot stall or hijack the schedule.  Hand-worked cases."""
    inf, nan = float("inf"), float("nan")
    t_next, act = oracle.block_schedule([0.0, 0.0, 0.0, 0.0], [0.5, inf, 0.25, 0.25])
    assert t_next == 0.25 and act.tolist() == [2, 3]
    t_next, act = oracle.block_schedule([0.0, -inf, nan, 1.0], [0.5, 0.25, 0.25, -0.5])
    assert t_next == 0.5 and act.tolist() == [0, 3]
    t_next, act = oracle.block_schedule([0.0, 1.0], [inf, inf])
    assert t_next == inf and act.size == 0
    t_next, act = oracle.block_schedule([nan, -inf, inf], [1.0, 1.0, -inf])     # inf + (-inf) = NaN
    assert t_next == inf and act.size == 0
