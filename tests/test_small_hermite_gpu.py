"""The small-i-set force + jerk kernel (csrc/nb_small_hermite.cuh: packed over j, one i-particle per thread, ten sums through
lanes, warps, a thread-block cluster and ticketed FP64 partials) through nb_force_jerk and the block step against the CPU
oracle: every instantiated decomposition, ragged shapes, coincident pairs with different velocities, determinism.

Tolerances as in test_hermite_gpu.py (BASELINE.json north_star / DESIGN.md R16): acceleration and jerk RMS <= 1e-5,
max <= 1e-4; phi RMS <= 1e-5.
"""
import numpy as np
import pytest

import oracle
from paper_astro_ph_0703100_b200 import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def nb():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device (no CPU fallback exists)"
    import paper_astro_ph_0703100_b200 as nb_
    nb_.lib()
    return nb_


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def gpu_fj(nb, x_i, v_i, x_j, v_j, m_j, eps2, want_pot=True):
    import torch
    acc, jerk, pot = nb.force_jerk(dev(x_i), dev(v_i), dev(x_j), dev(v_j), dev(m_j), eps2, want_pot=want_pot)
    torch.cuda.synchronize()
    return acc.cpu().numpy(), jerk.cpu().numpy(), (None if pot is None else pot.cpu().numpy())


def check(acc, jerk, pot, ra, rj, rp, label=""):
    e = oracle.error_metrics(acc, ra, pot, rp)
    ej = oracle.error_metrics(jerk, rj)
    assert e["acc_rms"] <= 1e-5 and e["acc_max"] <= 1e-4, (label, e)
    assert ej["acc_rms"] <= 1e-5 and ej["acc_max"] <= 1e-4, (label, "jerk", ej)
    if pot is not None:
        assert e["pot_rms"] <= 1e-5, (label, e)
    return e, ej


def subset_case(n_j, n_i, eps, seed):
    """C2's recipe with velocities: the i-set is a seeded random subset of the j-set (every i coincides with one j)."""
    w = wl.plummer_workload(n_j, eps, seed=seed, with_velocities=True)
    idx = np.sort(np.random.default_rng(seed + 1000).choice(n_j, n_i, replace=False))
    return w.x_j[idx].copy(), w.v[idx].copy(), w.x_j, w.v, w.m_j, w.eps2


# (NW, LJ, WJ) shapes x (S, CS): every instantiation, with and without the cluster level and the global level
SHAPES = [(16, 1, 2), (16, 1, 4), (16, 1, 8), (16, 1, 16), (8, 2, 8), (8, 4, 8)]
PLANS = [(nw, lj, wj, s, cs) for (nw, lj, wj) in SHAPES for (s, cs) in ((1, 1), (3, 1), (8, 8), (24, 8), (4, 4), (6, 2))]


@pytest.mark.parametrize("plan", PLANS, ids=lambda p: "NW%d_LJ%d_WJ%d_S%d_CS%d" % p)
def test_every_decomposition_matches_oracle(nb, plan, nbdebug):
    nbdebug.setenv("NB_SMALL_JERK", "1")
    nbdebug.setenv("NB_SMALL_JERK_PLAN", "%d,%d,%d,%d,%d" % plan)
    xi, vi, xj, vj, mj, eps2 = subset_case(3001, 333, 1.0 / 128, 21)
    acc, jerk, pot = gpu_fj(nb, xi, vi, xj, vj, mj, eps2)
    assert nb.last_launch_count() == 1                                  # one kernel: it packs the j-records itself
    ra, rj, rp = oracle.force_jerk(xi, vi, xj, vj, mj, eps2)
    check(acc, jerk, pot, ra, rj, rp, str(plan))
    # without the potential: the same a and jerk bit for bit (phi's accumulator is not formed)
    acc2, jerk2, pot2 = gpu_fj(nb, xi, vi, xj, vj, mj, eps2, want_pot=False)
    assert pot2 is None and np.array_equal(acc, acc2) and np.array_equal(jerk, jerk2)
    # repeated calls find the ticket counters back at zero
    acc3, jerk3, pot3 = gpu_fj(nb, xi, vi, xj, vj, mj, eps2)
    assert np.array_equal(acc, acc3) and np.array_equal(jerk, jerk3) and np.array_equal(pot, pot3)


@pytest.mark.parametrize("n_i,n_j", [(1, 1), (1, 777), (3, 100000), (129, 8), (31, 1000), (2048, 3), (1500, 4999), (17, 4097),
                                     (2048, 9000), (64, 70001), (5, 2), (512, 65536)])
def test_ragged_shapes_default_plan(nb, n_i, n_j, nbdebug):
    nbdebug.setenv("NB_SMALL_JERK", "1")
    rng = np.random.default_rng(n_i * 7919 + n_j)
    x_i, v_i = rng.normal(size=(n_i, 3)).astype(np.float32), rng.normal(size=(n_i, 3)).astype(np.float32)
    x_j, v_j = rng.normal(size=(n_j, 3)).astype(np.float32), rng.normal(size=(n_j, 3)).astype(np.float32)
    m_j = (rng.uniform(0.5, 1.5, n_j) / n_j).astype(np.float32)
    acc, jerk, pot = gpu_fj(nb, x_i, v_i, x_j, v_j, m_j, 2.0 ** -10)
    ra, rj, rp = oracle.force_jerk(x_i, v_i, x_j, v_j, m_j, np.float32(2.0 ** -10))
    check(acc, jerk, pot, ra, rj, rp, f"{n_i}x{n_j}")


def test_default_choice_and_its_edges(nb):
    for n_i, n_j, small in [(2048, 2048, 1), (4096, 8192, 1), (4096, 8193, 0), (1024, 65536, 1), (1025, 65536, 0), (300, 300, 1),
                            (4097, 1023, 0), (256, 1048576, 1), (257, 1048576, 0)]:
        assert nb.plan_query_small_jerk(n_i, n_j)["default"] == small
        xi, vi, xj, vj, mj, eps2 = subset_case(max(n_j, n_i), n_i, 1.0 / 128, n_i + n_j)
        xj, vj, mj = xj[:n_j], vj[:n_j], mj[:n_j]
        acc, jerk, pot = gpu_fj(nb, xi, vi, xj, vj, mj, eps2)
        if small:
            assert nb.last_launch_count() == 1
        idx = np.unique(np.concatenate([np.arange(0, n_i, max(1, n_i // 64)), [n_i - 1]]))
        ra, rj, rp = oracle.force_jerk(xi[idx], vi[idx], xj, vj, mj, eps2)
        check(acc[idx], jerk[idx], pot[idx], ra, rj, rp, f"{n_i}x{n_j}")
        assert np.all(np.isfinite(acc)) and np.all(np.isfinite(jerk)) and np.all(np.isfinite(pot))


def test_coincident_pairs_with_other_velocities_and_eps0(nb, nbdebug):
    """Reading R1: a pair whose POSITIONS coincide adds nothing -- whatever the velocities, for every eps2 including 0."""
    nbdebug.setenv("NB_SMALL_JERK", "1")
    w = wl.plummer_workload(1800, 1.0 / 64, seed=12, with_velocities=True)
    x, v = w.x_j.copy(), w.v.copy()
    x[1799] = x[5]; x[900] = x[5]                      # duplicates far apart in j, each with its own velocity
    x[700] = (0.0, 0.5, -0.0); x[1300] = (-0.0, 0.5, 0.0)   # the same point, opposite zero signs
    x[300] = x[8] + np.float32(1e-7)                   # near, not coincident
    for eps2 in (w.eps2, 0.0, 1e-30):
        acc, jerk, pot = gpu_fj(nb, x, v, x, v, w.m_j, eps2)
        assert np.all(np.isfinite(acc)) and np.all(np.isfinite(jerk)) and np.all(np.isfinite(pot))
        ra, rj, rp = oracle.force_jerk(x, v, x, v, w.m_j, np.float32(eps2))
        ok = np.ones(len(x), bool)
        if eps2 < 1e-20:
            ok[[300, 8]] = False                       # a 1e-7 separation without softening: FP32 differences, not the oracle's bar
        check(acc[ok], jerk[ok], pot[ok], ra[ok], rj[ok], rp[ok], f"eps2={eps2}")
    one_x, one_v = np.array([[1.5, -2.0, 0.25]], np.float32), np.array([[0.1, 0.2, 0.3]], np.float32)
    acc, jerk, pot = gpu_fj(nb, one_x, one_v, one_x, -one_v, np.array([3.0], np.float32), 0.0)
    assert np.all(acc == 0.0) and np.all(jerk == 0.0) and pot[0] == 0.0


@pytest.mark.parametrize("plan", [(8, 2, 8, 1, 1), (16, 1, 2, 5, 1), (16, 1, 4, 8, 8), (16, 1, 16, 12, 4)],
                         ids=lambda p: "NW%d_LJ%d_WJ%d_S%d_CS%d" % p)
def test_bitwise_reproducible_and_i_permutation_invariant(nb, plan, nbdebug):
    nbdebug.setenv("NB_SMALL_JERK", "1")
    nbdebug.setenv("NB_SMALL_JERK_PLAN", "%d,%d,%d,%d,%d" % plan)
    xi, vi, xj, vj, mj, eps2 = subset_case(6000, 1000, 1.0 / 128, 8)
    a1, j1, p1 = gpu_fj(nb, xi, vi, xj, vj, mj, eps2)
    a2, j2, p2 = gpu_fj(nb, xi, vi, xj, vj, mj, eps2)
    assert np.array_equal(a1, a2) and np.array_equal(j1, j2) and np.array_equal(p1, p2)
    perm = np.random.default_rng(5).permutation(len(xi))
    a3, j3, p3 = gpu_fj(nb, xi[perm], vi[perm], xj, vj, mj, eps2)
    assert np.array_equal(a1[perm], a3) and np.array_equal(j1[perm], j3) and np.array_equal(p1[perm], p3)


def test_outputs_are_written_inside_their_bounds_only(nb, nbdebug):
    """Guard bands around a, jerk and phi (compute-sanitizer is closed on this pool)."""
    import torch
    nbdebug.setenv("NB_SMALL_JERK", "1")
    for n_i, n_j in [(1, 2), (33, 777), (513, 4097), (2048, 2048), (70, 9001)]:
        xi, vi, xj, vj, mj, eps2 = subset_case(max(n_j, n_i), n_i, 1.0 / 64, n_i)
        xj, vj, mj = xj[:n_j], vj[:n_j], mj[:n_j]
        g = 64
        big_a = torch.full((n_i + 2 * g, 3), 1234.5, device="cuda"); big_j = torch.full((n_i + 2 * g, 3), -77.25, device="cuda")
        big_p = torch.full((n_i + 2 * g,), 99.0, device="cuda")
        nb.force_jerk(dev(xi), dev(vi), dev(xj), dev(vj), dev(mj), eps2, acc_out=big_a[g:g + n_i], jerk_out=big_j[g:g + n_i],
                      pot_out=big_p[g:g + n_i])
        torch.cuda.synchronize()
        for big, val in ((big_a, 1234.5), (big_j, -77.25), (big_p, 99.0)):
            assert float(big[:g].min()) == val and float(big[:g].max()) == val
            assert float(big[g + n_i:].min()) == val and float(big[g + n_i:].max()) == val
        ra, rj, rp = oracle.force_jerk(xi, vi, xj, vj, mj, eps2)
        check(big_a[g:g + n_i].cpu().numpy(), big_j[g:g + n_i].cpu().numpy(), big_p[g:g + n_i].cpu().numpy(), ra, rj, rp, f"{n_i}x{n_j}")
