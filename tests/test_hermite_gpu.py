"""Parity of nb_force_jerk (row f1: force + jerk + potential, Fig. A.4) against the CPU oracle.

Tolerances: acceleration and potential as for nb_force (BASELINE.json north_star: acc RMS <= 1e-5,
max <= 1e-4; phi RMS <= 1e-5).  Jerk: the same relative bars on |jerk_gpu - jerk_ref| / |jerk_ref|
(DESIGN.md derives them: the jerk is a sum of the same number of FP32 terms with the same rsqrt error,
formed as J1 - 3 J2 in FP64 from FP32 block partials).
"""
import os
from fractions import Fraction

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


@pytest.fixture(params=["default-kernel", "nb_hermite_kernel"])
def both_kernels(request, nbdebug):
    """Small shapes take the small-i-set force + jerk kernel (csrc/nb_small_hermite.cuh) by default: the tests that carry this
    fixture run a second time with NB_SMALL_JERK=0, on nb_hermite_kernel."""
    if request.param == "nb_hermite_kernel":
        nbdebug.setenv("NB_SMALL_JERK", "0")


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def gpu_fj(nb, x_i, v_i, x_j, v_j, m_j, eps2, want_pot=True, alias=False):
    import torch
    d_xj, d_vj = dev(x_j), dev(v_j)
    d_xi, d_vi = (d_xj, d_vj) if alias else (dev(x_i), dev(v_i))
    acc, jerk, pot = nb.force_jerk(d_xi, d_vi, d_xj, d_vj, dev(m_j), eps2, want_pot=want_pot)
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


def plummer_xv(n, eps, seed):
    w = wl.plummer_workload(n, eps, seed=seed, with_velocities=True)
    return w.x_j, w.v, w.m_j, w.eps2


@pytest.mark.usefixtures("both_kernels")
def test_c0_shape_full_parity(nb):
    x, v, m, eps2 = plummer_xv(2048, 1.0 / 64, 0)
    acc, jerk, pot = gpu_fj(nb, x, v, x, v, m, eps2, alias=True)
    ra, rj, rp = oracle.force_jerk(x, v, x, v, m, eps2)
    e, ej = check(acc, jerk, pot, ra, rj, rp, "C0 shape")
    assert ej["acc_max"] < 2e-5


@pytest.mark.usefixtures("both_kernels")
@pytest.mark.parametrize("n_i,n_j", [(1500, 4999), (31, 1000), (1, 777), (129, 8), (1025, 2051), (4096, 513)])
def test_ragged_shapes_separate_sets(nb, n_i, n_j):
    xj, vj, mj, eps2 = plummer_xv(n_j, 1.0 / 32, 11)
    xi, vi, _, _ = plummer_xv(n_i, 1.0 / 32, 12)
    mj = (mj * np.random.default_rng(1).uniform(0.5, 2.0, n_j)).astype(np.float32)
    acc, jerk, pot = gpu_fj(nb, xi, vi, xj, vj, mj, eps2)
    ra, rj, rp = oracle.force_jerk(xi, vi, xj, vj, mj, eps2)
    check(acc, jerk, pot, ra, rj, rp, f"{n_i}x{n_j}")


PLANS = [(k, 8 // wj, wj, s) for k in (2, 4) for wj in (1, 2, 4, 8) for s in (1, 3)]


@pytest.mark.parametrize("mode", ["exact", "list", "bloom"])
@pytest.mark.parametrize("plan", PLANS, ids=lambda p: "K%d_WI%d_WJ%d_S%d" % p)
def test_every_decomposition_matches_oracle(nb, plan, mode, nbdebug):
    nbdebug.setenv("NB_PLAN", "%d,%d,%d,%d" % plan)
    nbdebug.setenv("NB_MASK", mode)
    w = wl.subset_workload(3001, 777, 1.0 / 128, seed=21)
    rng = np.random.default_rng(5)
    vj = rng.normal(size=(3001, 3)).astype(np.float32)
    vi = rng.normal(size=(777, 3)).astype(np.float32)            # same positions as some j, other velocities
    acc, jerk, pot = gpu_fj(nb, w.x_i, vi, w.x_j, vj, w.m_j, w.eps2)
    ra, rj, rp = oracle.force_jerk(w.x_i, vi, w.x_j, vj, w.m_j, w.eps2)
    check(acc, jerk, pot, ra, rj, rp, str(plan) + mode)


def test_list_mode_agrees_bitwise_with_masked_kernel(nb, nbdebug):
    x, v, m, eps2 = plummer_xv(3000, 1.0 / 64, 12)
    x = x.copy(); v = v.copy()
    x[2999] = x[5]; x[1500] = x[5]                 # duplicates in other segments, with their own velocities
    x[700] = (0.0, 0.0, 0.0); x[2100] = (-0.0, 1e-41, 0.0)
    out = {}
    for mode in ("exact", "list", "bloom"):
        nbdebug.setenv("NB_MASK", mode)
        out[mode] = gpu_fj(nb, x, v, x, v, m, eps2, alias=True)
    for a, b, c in zip(out["exact"], out["list"], out["bloom"]):
        assert np.array_equal(a, b) and np.array_equal(a, c)
    nbdebug.setenv("NB_PLAN", "4,8,1,2")       # K = 4: without the potential the 26-instruction loop runs; same a and jerk
    nbdebug.setenv("NB_MASK", "exact")
    ref = gpu_fj(nb, x, v, x, v, m, eps2, alias=True)
    for mode in ("list", "bloom"):
        nbdebug.setenv("NB_MASK", mode)
        a, j, p = gpu_fj(nb, x, v, x, v, m, eps2, alias=True, want_pot=False)
        assert p is None and np.array_equal(a, ref[0]) and np.array_equal(j, ref[1])
    nbdebug.delenv("NB_PLAN")
    ra, rj, rp = oracle.force_jerk(x, v, x, v, m, eps2)
    keep = np.ones(3000, bool); keep[[700, 2100]] = False       # the oracle does not flush 1e-41
    check(out["list"][0][keep], out["list"][1][keep], out["list"][2][keep], ra[keep], rj[keep], rp[keep], "list")


@pytest.mark.usefixtures("both_kernels")
def test_coincident_positions_with_other_velocities_add_nothing(nb):
    one = np.array([[1.0, 2.0, 3.0]], dtype=np.float32)
    for eps2 in (0.0, 1e-4):
        acc, jerk, pot = gpu_fj(nb, one, np.array([[1, 0, 0]], np.float32), one, np.array([[0, 5, 0]], np.float32),
                                np.array([2.0], np.float32), eps2)
        assert not acc.any() and not jerk.any() and pot[0] == 0.0


@pytest.mark.usefixtures("both_kernels")
def test_two_body_exact_cases(nb):
    path = os.path.join(os.path.dirname(__file__), "golden", "hermite_two_body_exact.txt")
    for line in open(path):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        dx, dy, dz, ux, uy, uz, eps2, m, s = (Fraction(t) for t in line.split())
        d, dv = (dx, dy, dz), (ux, uy, uz)
        ddv = sum(a * b for a, b in zip(d, dv))
        a_exact = np.array([float(m * c / s ** 3) for c in d])
        j_exact = np.array([float(m * w / s ** 3 - 3 * m * ddv * c / s ** 5) for c, w in zip(d, dv)])
        xi = np.zeros((1, 3), np.float32); vi = np.zeros((1, 3), np.float32)
        xj = np.array([[float(c) for c in d]], np.float32); vj = np.array([[float(c) for c in dv]], np.float32)
        acc, jerk, pot = gpu_fj(nb, xi, vi, xj, vj, np.array([float(m)], np.float32), float(eps2))
        np.testing.assert_allclose(acc[0], a_exact, rtol=2e-6, atol=1e-9)
        np.testing.assert_allclose(jerk[0], j_exact, rtol=4e-6, atol=1e-6 * np.abs(j_exact).max())
        assert pot[0] == pytest.approx(float(-m / s), rel=1e-6)


@pytest.mark.usefixtures("both_kernels")
def test_empty_sets_null_pot_and_invalid_arguments(nb):
    import torch
    x, v, m, eps2 = plummer_xv(100, 1.0 / 16, 3)
    z3 = torch.zeros((0, 3), device="cuda"); z1 = torch.zeros((0,), device="cuda")
    acc, jerk, pot = nb.force_jerk(dev(x), dev(v), z3, z3, z1, eps2)
    torch.cuda.synchronize()
    assert not acc.any() and not jerk.any() and not pot.any()
    acc, jerk, pot = nb.force_jerk(z3, z3, dev(x), dev(v), dev(m), eps2)
    assert acc.shape == (0, 3) and jerk.shape == (0, 3)
    acc, jerk, pot = gpu_fj(nb, x, v, x, v, m, eps2, want_pot=False, alias=True)
    assert pot is None
    ra, rj, _ = oracle.force_jerk(x, v, x, v, m, eps2)
    check(acc, jerk, None, ra, rj, None, "no pot")
    with pytest.raises(nb.NBError):
        nb.force_jerk(dev(x), dev(v), dev(x), dev(v), dev(m), -1.0)
    L = nb.lib()
    assert L.nb_force_jerk(5, None, None, 5, None, None, None, 0.1, None, None, None, None) == 1


@pytest.mark.usefixtures("both_kernels")
def test_bitwise_reproducible_and_i_permutation_invariant(nb):
    x, v, m, eps2 = plummer_xv(5000, 1.0 / 64, 8)
    a1 = gpu_fj(nb, x, v, x, v, m, eps2, alias=True)
    a2 = gpu_fj(nb, x, v, x, v, m, eps2, alias=True)
    for p, q in zip(a1, a2):
        assert np.array_equal(p, q)
    perm = np.random.default_rng(0).permutation(5000)
    a3 = gpu_fj(nb, x[perm], v[perm], x, v, m, eps2)
    for p, q in zip(a1, a3):
        assert np.array_equal(p[perm], q)


@pytest.mark.usefixtures("both_kernels")
def test_jerk_momentum_antisymmetry_fp32(nb):
    x, v, m, eps2 = plummer_xv(4096, 1.0 / 64, 9)
    acc, jerk, _ = gpu_fj(nb, x, v, x, v, m, eps2, alias=True)
    for arr in (acc, jerk):
        tot = np.linalg.norm((m[:, None].astype(np.float64) * arr).sum(0))
        assert tot <= 1e-5 * (m[:, None] * np.linalg.norm(arr, axis=1)[:, None]).sum()


def test_h1_full_size_all_elements(nb):
    """N = 131072 Plummer sphere with velocities, in the launch configuration `bench.py --op jerk` times: ALL 131072
    accelerations, jerks and potentials against the oracle (Eq. (3): the maximum is over all particles;
    the FP64 direct sum is 1.7e10 pairs, ~11 s on the GPU box's host cores)."""
    x, v, m, eps2 = plummer_xv(131072, 1.0 / 256, 1)
    acc, jerk, pot = gpu_fj(nb, x, v, x, v, m, eps2, alias=True)
    ra, rj, rp = oracle.force_jerk(x, v, x, v, m, eps2)
    check(acc, jerk, pot, ra, rj, rp, "H1 all elements")
    tot = np.linalg.norm((m[:, None].astype(np.float64) * jerk).sum(0))
    assert tot <= 1e-5 * (m[:, None] * np.linalg.norm(jerk, axis=1)[:, None]).sum()


@pytest.mark.usefixtures("both_kernels")
def test_force_jerk_host_matches_device_path(nb):
    x, v, m, eps2 = plummer_xv(3000, 1.0 / 64, 15)
    a_d, j_d, p_d = gpu_fj(nb, x, v, x, v, m, eps2, alias=True)
    a_h, j_h, p_h = nb.force_jerk_host(x, v, x, v, m, eps2)
    assert np.array_equal(a_d, a_h) and np.array_equal(j_d, j_h) and np.array_equal(p_d, p_h)
    xi, vi = x[:100].copy(), v[:100].copy()
    a_h, j_h, p_h = nb.force_jerk_host(xi, vi, x, v, m, eps2, want_pot=False)
    ra, rj, _ = oracle.force_jerk(xi, vi, x, v, m, eps2)
    assert p_h is None
    check(a_h, j_h, None, ra, rj, None, "host subset")


@pytest.mark.parametrize("plan", [(4, 8, 1, 5), (4, 2, 4, 3), (2, 1, 8, 7), (2, 4, 2, 2)], ids=lambda p: "K%d_WI%d_WJ%d_S%d" % p)
def test_fused_second_pass_is_bitwise_the_separate_reduce(nb, plan, nbdebug):
    """nb_force_jerk: the last CTA of an i-tile sums the S chunk partials in the order nb_hermite_reduce_kernel does;
    same bits, one launch fewer, ticket counters back at zero after every call."""
    nbdebug.setenv("NB_PLAN", "%d,%d,%d,%d" % plan)
    x, v, m, eps2 = plummer_xv(4000, 1.0 / 64, 19)
    out = {}
    for fused in ("1", "0"):
        nbdebug.setenv("NB_FUSED_REDUCE", fused)
        runs = [gpu_fj(nb, x, v, x, v, m, eps2, alias=True) for _ in range(3)]
        for r in runs[1:]:
            assert all(np.array_equal(a, b) for a, b in zip(r, runs[0]))
        out[fused] = runs[0] + (nb.last_launch_count(),)
    assert all(np.array_equal(a, b) for a, b in zip(out["1"][:3], out["0"][:3]))
    assert out["0"][3] == out["1"][3] + 1
    ra, rj, rp = oracle.force_jerk(x, v, x, v, m, eps2)
    check(out["1"][0], out["1"][1], out["1"][2], ra, rj, rp, "fused " + str(plan))
