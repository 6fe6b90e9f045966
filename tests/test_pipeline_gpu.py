"""The generalised pair kernel (section 4.5; include/nb_pipeline.cuh) running the paper's two
pipeline descriptions through the paper's own call shape cunbody_api(p_xj, p_xi, p_fi, ni, nj),
against the CPU oracle.  Same tolerances as the specialised kernels."""
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
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()


def rows_a3(x_i, eps2_i, x_j, m_j):
    """Fig. A.1 packing loops: p_xi[i] = (x, y, z, eps2), p_xj[j] = (x, y, z, m)."""
    return np.concatenate([x_i, eps2_i[:, None]], 1), np.concatenate([x_j, m_j[:, None]], 1)


def rows_a4(x_i, v_i, x_j, v_j, m_j):
    """Fig. A.2 packing loop: p_xi[i] = (x, v), p_xj[j] = (x, v, m)."""
    return np.concatenate([x_i, v_i], 1), np.concatenate([x_j, v_j, m_j[:, None]], 1)


@pytest.mark.parametrize("n_i,n_j", [(3000, 3000), (1, 777), (31, 1000), (1025, 2051), (70000, 300), (513, 40000)])
def test_fig_a3_pipeline_matches_oracle(nb, n_i, n_j):
    import torch
    w = wl.plummer_workload(max(n_i, n_j), 1.0 / 64, seed=41)
    rng = np.random.default_rng(n_i)
    x_j, m_j = w.x_j[:n_j], (w.m_j[:n_j] * rng.uniform(0.5, 2.0, n_j)).astype(np.float32)
    x_i = w.x_j[:n_i] if n_i <= n_j else rng.normal(size=(n_i, 3)).astype(np.float32)   # subsets coincide with their j
    e2 = (2.0 ** rng.integers(-18, -6, n_i)).astype(np.float32)
    p_xi, p_xj = rows_a3(x_i, e2, x_j, m_j)
    p_fi = nb.cunbody_force(dev(p_xj), dev(p_xi))
    torch.cuda.synchronize()
    ra, _ = oracle.force_eps_i(x_i, e2, x_j, m_j)
    e = oracle.error_metrics(p_fi.cpu().numpy(), ra)
    assert e["acc_rms"] <= 1e-5 and e["acc_max"] <= 1e-4, e


@pytest.mark.parametrize("n_i,n_j", [(2048, 2048), (100, 5000), (4097, 777)])
def test_fig_a4_pipeline_matches_oracle(nb, n_i, n_j):
    import torch
    w = wl.plummer_workload(max(n_i, n_j), 1.0 / 256, seed=42, with_velocities=True)
    x_j, v_j, m_j = w.x_j[:n_j], w.v[:n_j], w.m_j[:n_j]
    x_i, v_i = w.x_j[:n_i], w.v[:n_i] * np.float32(1.5)
    p_xi, p_xj = rows_a4(x_i, v_i, x_j, v_j, m_j)
    p_fi = nb.cunbody_force_jerk_pot(dev(p_xj), dev(p_xi)).cpu().numpy()
    torch.cuda.synchronize()
    ra, rj, rp = oracle.force_jerk(x_i, v_i, x_j, v_j, m_j, np.float32(1.0 / 65536.0))     # the listing's eps2
    e = oracle.error_metrics(p_fi[:, 0:3], ra, p_fi[:, 6], rp)
    ej = oracle.error_metrics(p_fi[:, 3:6], rj)
    assert e["acc_rms"] <= 1e-5 and e["acc_max"] <= 1e-4 and e["pot_rms"] <= 1e-5, e
    assert ej["acc_rms"] <= 1e-5 and ej["acc_max"] <= 1e-4, ej


def test_agrees_with_the_specialised_kernels_and_edge_sizes(nb):
    import torch
    w = wl.plummer_workload(5000, 1.0 / 64, seed=43)
    e2 = np.full(5000, w.eps2, np.float32)
    p_xi, p_xj = rows_a3(w.x_j, e2, w.x_j, w.m_j)
    a_gen = nb.cunbody_force(dev(p_xj), dev(p_xi))
    a_gen2 = nb.cunbody_force(dev(p_xj), dev(p_xi))
    a_spec, _ = nb.force(dev(w.x_j), dev(w.x_j), dev(w.m_j), w.eps2)
    torch.cuda.synchronize()
    assert torch.equal(a_gen, a_gen2)                                           # reproducible
    assert torch.allclose(a_gen, a_spec, rtol=2e-5, atol=1e-6)
    z = torch.zeros((0, 4), device="cuda")
    out = nb.cunbody_force(z, dev(p_xi))                                        # nj = 0: zero-filled
    torch.cuda.synchronize()
    assert out.shape == (5000, 3) and not out.any()
    assert nb.cunbody_force(dev(p_xj), z).shape == (0, 3)                       # ni = 0
    assert nb.lib().nb_cunbody_force(None, None, None, 5, 5, None) == 1


# ------------------------------------------------------------------ a central force other than gravity (reading R19)
def _lj_scales(rows_i, rows_j):
    """sum_j |f_ij| |d| and sum_j |u_ij| per i, in double: what the FP32 rounding errors of the pairs are relative to."""
    xi, xj = rows_i.astype(np.float64), rows_j.astype(np.float64)
    fs, us = np.zeros(xi.shape[0]), np.zeros(xi.shape[0])
    for lo in range(0, xi.shape[0], 256):
        I = xi[lo:lo + 256]
        d = xj[None, :, :3] - I[:, None, :3]
        r2 = (d * d).sum(-1)
        ok = r2 > 0
        r2 = np.where(ok, r2, 1.0)
        s6 = ((I[:, None, 3] + xj[None, :, 3]) ** 2 / r2) ** 3
        e = I[:, None, 4] * xj[None, :, 4]
        fs[lo:lo + 256] = np.where(ok, 24 * e * (2 * s6 * s6 + s6) / np.sqrt(r2), 0.0).sum(1)
        us[lo:lo + 256] = np.where(ok, 4 * e * (s6 * s6 + s6), 0.0).sum(1)
    return fs, us


@pytest.mark.parametrize("n_i,n_j", [(1, 1), (700, 3001), (2500, 2500), (257, 20000)])
def test_lennard_jones_pipeline_matches_oracle(nb, n_i, n_j):
    """nb_cunbody_lennard_jones against the double-precision oracle on a dense fluid (jittered lattice, density 0.8,
    mixed sigma and eps).  Tolerance: every pair carries the rsqrt.approx error (2^-22) six times in s^12 plus ~10 FP32
    roundings, < 4e-6 of its own magnitude; block partials are FP32 over <= 256 j, totals FP64 -- so
    |F - F_ref| <= 1e-5 sum_j |f_ij| and |U - U_ref| <= 1e-5 sum_j |u_ij| (measured: 1e-6)."""
    import torch
    rows = wl.lj_fluid_rows(max(n_i, n_j), 0.8, 0.1, seed=41)
    rows_j = rows[:n_j]
    rows_i = rows[:n_i] if n_i <= n_j else rows
    if n_i == 257:
        rows_i = rows[::-1][:n_i].copy()                              # a subset from the other end of the list
    out = nb.cunbody_lennard_jones(dev(rows_j), dev(rows_i))
    torch.cuda.synchronize()
    out = out.cpu().numpy().astype(np.float64)
    ref = oracle.lennard_jones(rows_i, rows_j)
    if n_j == 1:
        assert not out.any() and not ref.any()                        # the only pair is the particle with itself
        return
    fs, us = _lj_scales(rows_i, rows_j)
    assert np.all(np.isfinite(out))
    assert (np.linalg.norm(out[:, :3] - ref[:, :3], axis=1) / fs).max() <= 1e-5
    assert (np.abs(out[:, 3] - ref[:, 3]) / us).max() <= 1e-5
    if n_i == n_j:                                                    # closed system: the forces sum to zero up to the
        # accumulated rounding of n_i independent results
        assert np.abs(out[:, :3].sum(0)).max() <= 1e-5 * fs.mean() * np.sqrt(n_i)


def test_lennard_jones_pipeline_edge_cases(nb):
    import torch
    rows = wl.lj_fluid_rows(100, 0.8, 0.1, seed=42)
    empty = torch.empty((0, 5), dtype=torch.float32, device="cuda")
    out = nb.cunbody_lennard_jones(empty, dev(rows))                  # no j-particles: zeros
    assert out.shape == (100, 4) and not out.cpu().numpy().any()
    out = nb.cunbody_lennard_jones(dev(rows), empty)                  # no i-particles: nothing to do
    assert out.shape == (0, 4)
    # two particles at the potential minimum: no force, U = -eps for both
    sigma, eps = 1.0, 2.0
    pair = np.array([[0, 0, 0, sigma / 2, np.sqrt(eps)], [2 ** (1 / 6) * sigma, 0, 0, sigma / 2, np.sqrt(eps)]], np.float32)
    out = nb.cunbody_lennard_jones(dev(pair), dev(pair)).cpu().numpy()
    assert np.abs(out[:, :3]).max() <= 2e-5 * 24 * eps / sigma and np.abs(out[:, 3] + eps).max() <= 1e-5 * eps


@pytest.mark.parametrize("which", ["a3", "a4", "lj"])
def test_bench_size_in_the_launch_configuration_bench_times(nb, which):
    """N = 131072, the calls `bench.py --op cunbody | cunbody4 | lj` time (packed path, S j-chunks in whole waves, second
    pass): 2048 seeded i-records of the full-size output against the oracle, plus finiteness of everything."""
    import torch
    n = 131072
    idx = np.sort(np.random.default_rng(3).choice(n, 2048, replace=False))
    if which == "lj":
        rows = wl.lj_fluid_rows(n, 0.8, 0.1, seed=1)
        out = nb.cunbody_lennard_jones(dev(rows), dev(rows))
        torch.cuda.synchronize()
        out = out.cpu().numpy().astype(np.float64)
        assert np.all(np.isfinite(out))
        ref = oracle.lennard_jones(np.ascontiguousarray(rows[idx]), rows)
        sub = idx[::16]                                               # the error scales need an [i][j][3] array: 128 records
        fs, us = np.concatenate([_lj_scales(np.ascontiguousarray(rows[sub[k:k + 32]]), rows) for k in range(0, sub.size, 32)], axis=1)
        assert (np.linalg.norm(out[sub, :3] - ref[::16, :3], axis=1) / fs).max() <= 1e-5
        assert (np.abs(out[sub, 3] - ref[::16, 3]) / us).max() <= 1e-5
        # all 2048: relative to the largest force / energy scale of the sample (the fluid is homogeneous)
        assert np.abs(out[idx, :3] - ref[:, :3]).max() <= 1e-5 * fs.max() and np.abs(out[idx, 3] - ref[:, 3]).max() <= 1e-5 * us.max()
        return
    w = wl.plummer_workload(n, 1.0 / 256, seed=1, with_velocities=True)
    if which == "a3":
        e2 = np.full(n, w.eps2, np.float32)
        p_xi, p_xj = rows_a3(w.x_j, e2, w.x_j, w.m_j)
        p_fi = nb.cunbody_force(dev(p_xj), dev(p_xi))
        torch.cuda.synchronize()
        p_fi = p_fi.cpu().numpy()
        assert np.all(np.isfinite(p_fi))
        ra, _ = oracle.force(np.ascontiguousarray(w.x_j[idx]), w.x_j, w.m_j, w.eps2)
        e = oracle.error_metrics(p_fi[idx], ra)
        assert e["acc_rms"] <= 1e-5 and e["acc_max"] <= 1e-4, e
    else:
        p_xi, p_xj = rows_a4(w.x_j, w.v, w.x_j, w.v, w.m_j)
        p_fi = nb.cunbody_force_jerk_pot(dev(p_xj), dev(p_xi))
        torch.cuda.synchronize()
        p_fi = p_fi.cpu().numpy()
        assert np.all(np.isfinite(p_fi))
        ra, rj, rp = oracle.force_jerk(np.ascontiguousarray(w.x_j[idx]), np.ascontiguousarray(w.v[idx]), w.x_j, w.v, w.m_j,
                                       np.float32(1.0 / 65536.0))
        e = oracle.error_metrics(p_fi[idx, 0:3], ra, p_fi[idx, 6], rp)
        ej = oracle.error_metrics(p_fi[idx, 3:6], rj)
        assert e["acc_rms"] <= 1e-5 and e["acc_max"] <= 1e-4 and e["pot_rms"] <= 1e-5, e
        assert ej["acc_rms"] <= 1e-5 and ej["acc_max"] <= 1e-4, ej


def test_generalised_kernel_writes_inside_its_bounds_only(nb):
    """Guard bands around p_fi for the three pipelines on the packed path, ragged sizes (compute-sanitizer is closed here)."""
    import torch
    n_i, n_j, pad, sentinel = 2500, 3001, 200, -999.0
    w = wl.plummer_workload(n_j, 1.0 / 256, seed=43, with_velocities=True)
    rows = wl.lj_fluid_rows(n_j, 0.8, 0.1, seed=43)
    e2 = np.full(n_i, w.eps2, np.float32)
    a3 = rows_a3(w.x_j[:n_i], e2, w.x_j, w.m_j)
    a4 = rows_a4(w.x_j[:n_i], w.v[:n_i], w.x_j, w.v, w.m_j)
    for fn, p_xi, p_xj, fdim in ((nb.cunbody_force, a3[0], a3[1], 3), (nb.cunbody_force_jerk_pot, a4[0], a4[1], 7),
                                 (nb.cunbody_lennard_jones, rows[:n_i], rows, 4)):
        big = torch.full((n_i + 2 * pad, fdim), sentinel, device="cuda")
        fn(dev(p_xj), dev(p_xi), big[pad:pad + n_i])
        torch.cuda.synchronize()
        assert torch.all(big[:pad] == sentinel) and torch.all(big[pad + n_i:] == sentinel)
        assert not torch.any(big[pad:pad + n_i] == sentinel) and torch.all(torch.isfinite(big[pad:pad + n_i]))
