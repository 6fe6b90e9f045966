"""Parity of nb_force_eps_i (row f3: eps^2 per i-particle, Fig. A.1) against the oracle.
Tolerances as for nb_force: acc RMS <= 1e-5, max <= 1e-4; phi RMS <= 1e-5."""
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


def gpu(nb, x_i, e2, x_j, m_j, alias=False, want_pot=True):
    import torch
    d_xj = dev(x_j)
    d_xi = d_xj if alias else dev(x_i)
    acc, pot = nb.force_eps_i(d_xi, dev(e2), d_xj, dev(m_j), want_pot=want_pot)
    torch.cuda.synchronize()
    return acc.cpu().numpy(), (None if pot is None else pot.cpu().numpy())


def check(acc, pot, ra, rp, label):
    e = oracle.error_metrics(acc, ra, pot, rp)
    assert e["acc_rms"] <= 1e-5 and e["acc_max"] <= 1e-4 and e["pot_rms"] <= 1e-5, (label, e)


def eps2_mix(n, seed):
    """Softenings spread over four decades, some exactly zero (point masses)."""
    rng = np.random.default_rng(seed)
    e = (2.0 ** rng.integers(-20, -6, n)).astype(np.float32)
    e[rng.random(n) < 0.05] = 0.0
    return e


@pytest.mark.parametrize("mode", ["exact", "list"])
@pytest.mark.parametrize("plan", [(8, 8, 1, 3), (8, 4, 2, 1), (4, 2, 4, 5), (2, 1, 8, 2), (4, 8, 1, 1), (2, 4, 2, 7),
                                  (8, 1, 8, 2), (8, 2, 4, 1)], ids=lambda p: "K%d_WI%d_WJ%d_S%d" % p)
def test_every_decomposition_matches_oracle(nb, plan, mode, nbdebug):
    nbdebug.setenv("NB_PLAN", "%d,%d,%d,%d" % plan)
    nbdebug.setenv("NB_MASK", mode)
    w = wl.plummer_workload(3000, 1.0 / 64, seed=31)
    e2 = eps2_mix(3000, 1)
    acc, pot = gpu(nb, w.x_j, e2, w.x_j, w.m_j, alias=True)
    ra, rp = oracle.force_eps_i(w.x_j, e2, w.x_j, w.m_j)
    check(acc, pot, ra, rp, str(plan) + mode)


def test_constant_array_equals_nb_force_bitwise_in_masked_mode(nb, nbdebug):
    import torch
    nbdebug.setenv("NB_MASK", "exact")
    w = wl.subset_workload(5000, 700, 1.0 / 128, seed=9)
    acc, pot = gpu(nb, w.x_i, np.full(700, w.eps2, np.float32), w.x_j, w.m_j)
    a0, p0 = nb.force(dev(w.x_i), dev(w.x_j), dev(w.m_j), w.eps2)
    torch.cuda.synchronize()
    assert np.array_equal(acc, a0.cpu().numpy()) and np.array_equal(pot, p0.cpu().numpy())


def test_two_body_each_i_its_own_eps2(nb):
    xj = np.array([[10.0, -20.0, 5.0]], np.float32)
    d = np.array([[3, 0, 0], [2, 3, 6], [1, 2, 2], [3, 0, 0]], np.float32)
    e2 = np.array([16.0, 0.0, 0.0, 0.0], np.float32)
    s = np.array([5.0, 7.0, 3.0, 3.0])
    acc, pot = gpu(nb, xj - d, e2, xj, np.array([2.0], np.float32))
    np.testing.assert_allclose(acc, 2.0 * d / s[:, None] ** 3, rtol=2e-6)
    np.testing.assert_allclose(pot, -2.0 / s, rtol=1e-6)


def test_ragged_separate_sets_edge_sizes_and_errors(nb):
    import torch
    for n_i, n_j in [(1, 777), (31, 1000), (1025, 2051)]:
        rng = np.random.default_rng(n_i)
        xi = rng.normal(size=(n_i, 3)).astype(np.float32); xj = rng.normal(size=(n_j, 3)).astype(np.float32)
        mj = rng.uniform(0.5, 1.5, n_j).astype(np.float32); e2 = eps2_mix(n_i, 2)
        acc, pot = gpu(nb, xi, e2, xj, mj)
        ra, rp = oracle.force_eps_i(xi, e2, xj, mj)
        check(acc, pot, ra, rp, f"{n_i}x{n_j}")
    z3 = torch.zeros((0, 3), device="cuda"); z1 = torch.zeros((0,), device="cuda")
    a, p = nb.force_eps_i(dev(xi), dev(e2), z3, z1)
    torch.cuda.synchronize()
    assert not a.any() and not p.any()
    a, p = nb.force_eps_i(z3, z1, dev(xj), dev(mj))
    assert a.shape == (0, 3)
    assert nb.lib().nb_force_eps_i(5, None, None, 5, None, None, None, None, None) == 1


def test_full_size_list_mode_sampled(nb):
    """N = 131072 (C1's particles), softening per particle: the large-call path (coincidence lists), 2048 sampled i."""
    w = wl.config(1)
    e2 = eps2_mix(w.n_j, 3)
    acc, pot = gpu(nb, w.x_j, e2, w.x_j, w.m_j, alias=True)
    idx = np.sort(np.random.default_rng(5).choice(w.n_j, 2048, replace=False))
    ra, rp = oracle.force_eps_i(w.x_j[idx], e2[idx], w.x_j, w.m_j)
    check(acc[idx], pot[idx], ra, rp, "C1 eps_i sampled")
