"""Parity of the CUDA path (through the C ABI, via the ctypes binding) against the CPU oracle.

Tolerances are BASELINE.json north_star's: per-particle relative acceleration error
|a_gpu - a_ref| / |a_ref| (Eq. (3)): RMS <= 1e-5 and max <= 1e-4; relative potential
error <= 1e-5 RMS.  All inputs are seeded and synthetic (paper_astro_ph_0703100_b200/workloads.py).
"""
import os

import numpy as np
import pytest

import oracle
from paper_astro_ph_0703100_b200 import workloads as wl

pytestmark = pytest.mark.gpu

ACC_RMS_TOL = 1e-5
ACC_MAX_TOL = 1e-4
POT_RMS_TOL = 1e-5


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


def gpu_force(nb, x_i, x_j, m_j, eps2, want_pot=True, alias=False):
    import torch
    d_xj = dev(x_j)
    d_xi = d_xj if alias else dev(x_i)
    acc, pot = nb.force(d_xi, d_xj, dev(m_j), eps2, want_pot=want_pot)
    torch.cuda.synchronize()
    return acc.cpu().numpy(), (None if pot is None else pot.cpu().numpy())


def check_parity(acc, pot, ref_acc, ref_pot, label=""):
    e = oracle.error_metrics(acc, ref_acc, pot, ref_pot)
    assert e["acc_rms"] <= ACC_RMS_TOL, (label, e)
    assert e["acc_max"] <= ACC_MAX_TOL, (label, e)
    if pot is not None:
        assert e["pot_rms"] <= POT_RMS_TOL, (label, e)
    return e


# ------------------------------------------------------------------ element-by-element, small
def test_c0_full_parity(nb):
    w = wl.config(0)
    acc, pot = gpu_force(nb, w.xi, w.x_j, w.m_j, w.eps2, alias=True)
    ref_acc, ref_pot = oracle.force(w.xi, w.x_j, w.m_j, w.eps2)
    e = check_parity(acc, pot, ref_acc, ref_pot, "C0")
    # paper's Table 2: blocked FP32 sums give E_max ~ 3e-7 ... 1.5e-6; same order here
    assert e["acc_max"] < 2e-5


@pytest.mark.parametrize("n_i,n_j", [(1500, 4999), (31, 1000), (1, 777), (129, 8), (1025, 2051), (4096, 513)])
def test_ragged_shapes_separate_sets(nb, n_i, n_j):
    rng = np.random.default_rng(n_i * 7919 + n_j)
    pos_j, _ = wl.plummer_positions(n_j, rng)
    pos_i, _ = wl.plummer_positions(n_i, rng)
    m = rng.uniform(0.5, 1.5, n_j) / n_j
    x_i, x_j, m_j = pos_i.astype(np.float32), pos_j.astype(np.float32), m.astype(np.float32)
    eps2 = np.float32(2.0 ** -12)
    acc, pot = gpu_force(nb, x_i, x_j, m_j, eps2)
    ref_acc, ref_pot = oracle.force(x_i, x_j, m_j, eps2)
    check_parity(acc, pot, ref_acc, ref_pot, f"{n_i}x{n_j}")


PLANS = [(k, 8 // wj, wj, s) for k in (2, 4, 8) for wj in (1, 2, 4, 8) for s in (1, 3)]


@pytest.mark.parametrize("plan", PLANS, ids=lambda p: "K%d_WI%d_WJ%d_S%d" % p)
def test_every_decomposition_matches_oracle(nb, plan, nbdebug):
    """Each kernel instantiation (K x WJ) with and without the second-pass reduce (S)."""
    nbdebug.setenv("NB_PLAN", "%d,%d,%d,%d" % plan)
    w = wl.subset_workload(3001, 777, 1.0 / 128, seed=21)
    acc, pot = gpu_force(nb, w.x_i, w.x_j, w.m_j, w.eps2)
    ref_acc, ref_pot = oracle.force(w.x_i, w.x_j, w.m_j, w.eps2)
    check_parity(acc, pot, ref_acc, ref_pot, str(plan))


def test_masked_list_and_acceleration_only_paths_agree_bitwise(nb, nbdebug):
    """Masked kernel, list-mode kernel and the acceleration-only path (untested loop everywhere) store the same bits --
    with self pairs (aliased sets), duplicates, and a near-coincident pair whose r2 rounds to eps2."""
    nbdebug.setenv("NB_SMALL", "0")                # nb_force_kernel's paths (the small-i-set kernel: tests/test_small_gpu.py)
    w = wl.config(0)
    x = w.x_j.copy()
    x[100] = x[7]                                  # exact duplicates
    x[101] = x[7]
    x[300] = x[8] + np.float32(1e-7)               # closer than eps * 2.4e-4: r2 rounds to eps2 without coincidence
    ref_acc, ref_pot = oracle.force(x, x, w.m_j, w.eps2)
    nbdebug.setenv("NB_MASK", "exact")
    a_e, p_e = gpu_force(nb, x, x, w.m_j, w.eps2, alias=True)
    nbdebug.setenv("NB_MASK", "list")
    a_l, p_l = gpu_force(nb, x, x, w.m_j, w.eps2, alias=True)
    nbdebug.delenv("NB_MASK")
    a_d, p_d = gpu_force(nb, x, x, w.m_j, w.eps2, alias=True)                  # default (small call: masked)
    a_o, _ = gpu_force(nb, x, x, w.m_j, w.eps2, want_pot=False, alias=True)    # acceleration only: no mask at all
    assert np.array_equal(a_e, a_l) and np.array_equal(p_e, p_l)
    assert np.array_equal(a_e, a_d) and np.array_equal(p_e, p_d) and np.array_equal(a_e, a_o)
    # the self term would shift phi by m/eps = 64/2048 = 3e-2 absolute (~3 % relative): far outside tolerance
    check_parity(a_d, p_d, ref_acc, ref_pot, "C0 + duplicates")
    # separate i-set drawn from the j-set (C2 shape): each i coincides with exactly one j
    w2 = wl.subset_workload(5000, 700, 1.0 / 128, seed=9)
    nbdebug.setenv("NB_MASK", "exact")
    a_e, p_e = gpu_force(nb, w2.x_i, w2.x_j, w2.m_j, w2.eps2)
    nbdebug.setenv("NB_MASK", "list")
    a_l, p_l = gpu_force(nb, w2.x_i, w2.x_j, w2.m_j, w2.eps2)
    assert np.array_equal(a_e, a_l) and np.array_equal(p_e, p_l)


def _both_modes(nb, nbdebug, x_i, x_j, m_j, eps2, alias=False):
    out = {}
    for mode in ("exact", "list", "bloom"):
        nbdebug.setenv("NB_MASK", mode)
        out[mode] = gpu_force(nb, x_i, x_j, m_j, eps2, alias=alias)
    nbdebug.delenv("NB_MASK")
    # MODE_BLOOM (filter of the warp's i-positions in shared memory, every 256-j block tested in the kernel) must
    # store what the always-masked kernel stores, bit for bit, wherever the list mode must
    assert np.array_equal(out["exact"][0], out["bloom"][0]) and np.array_equal(out["exact"][1], out["bloom"][1])
    return out


@pytest.mark.parametrize("plan", [(8, 8, 1, 3), (8, 4, 2, 1), (4, 2, 4, 5), (2, 1, 8, 2), (4, 8, 1, 1), (2, 4, 2, 7)],
                         ids=lambda p: "K%d_WI%d_WJ%d_S%d" % p)
def test_list_mode_agrees_bitwise_with_masked_kernel(nb, plan, nbdebug):
    """MODE_LIST (hash-join pre-pass, untested hot loop, masked loop only on listed j-segments) stores what the
    always-masked kernel stores, bit for bit: self pairs, duplicates across segments, -0 vs +0, subnormals."""
    nbdebug.setenv("NB_PLAN", "%d,%d,%d,%d" % plan)
    w = wl.plummer_workload(3000, 1.0 / 64, seed=12)
    x = w.x_j.copy()
    x[2999] = x[5]                                 # duplicate far away in j (another segment)
    x[1500] = x[5]
    x[700] = (0.0, 0.0, 0.0)
    x[2100] = (-0.0, 1e-41, 0.0)                   # canonically equal to particle 700 (add.ftz flushes subnormals)
    x[300] = x[8] + np.float32(1e-7)               # near, not coincident
    out = _both_modes(nb, nbdebug, x, x, w.m_j, w.eps2, alias=True)
    assert np.array_equal(out["exact"][0], out["list"][0]) and np.array_equal(out["exact"][1], out["list"][1])
    ref_acc, ref_pot = oracle.force(x, x, w.m_j, w.eps2)
    keep = np.ones(3000, bool); keep[[700, 2100]] = False      # the oracle does not flush 1e-41: that pair differs by design
    check_parity(out["list"][0][keep], out["list"][1][keep], ref_acc[keep], ref_pot[keep], "list " + str(plan))
    # separate i-set drawn from the j-set (C2 shape)
    w2 = wl.subset_workload(5000, 700, 1.0 / 128, seed=9)
    out = _both_modes(nb, nbdebug, w2.x_i, w2.x_j, w2.m_j, w2.eps2)
    assert np.array_equal(out["exact"][0], out["list"][0]) and np.array_equal(out["exact"][1], out["list"][1])
    ref_acc, ref_pot = oracle.force(w2.x_i, w2.x_j, w2.m_j, w2.eps2)
    check_parity(out["list"][0], out["list"][1], ref_acc, ref_pot, "list subset " + str(plan))


def test_list_mode_degenerate_inputs(nb, nbdebug):
    """Overflowing lists (> 8 partner segments per i-group) and a degenerate table (thousands of identical
    positions) fall back to masking everywhere: still the always-masked result."""
    rng = np.random.default_rng(3)
    n = 6000
    x = rng.normal(size=(n, 3)).astype(np.float32)
    m = rng.uniform(0.5, 1.5, n).astype(np.float32) / n
    x[::300] = x[0]                                # 20 copies spread over 20 segments: list overflow for group 0
    out = _both_modes(nb, nbdebug, x, x, m, 1e-3, alias=True)
    assert np.array_equal(out["exact"][0], out["list"][0]) and np.array_equal(out["exact"][1], out["list"][1])
    ref_acc, ref_pot = oracle.force(x, x, m, 1e-3)
    check_parity(out["list"][0], out["list"][1], ref_acc, ref_pot, "overflow")
    x[:5000] = (1.0, 2.0, 3.0)                     # 5000 identical positions: probe chains exceed the cap
    out = _both_modes(nb, nbdebug, x, x, m, 1e-3, alias=True)
    assert np.array_equal(out["exact"][0], out["list"][0]) and np.array_equal(out["exact"][1], out["list"][1])
    ref_acc, ref_pot = oracle.force(x, x, m, 1e-3)
    sel = slice(5000, n)                           # the 5000 coincident ones have a ~ 0: compare the others relatively
    check_parity(out["list"][0][sel], out["list"][1][sel], ref_acc[sel], ref_pot[sel], "degenerate")
    assert np.abs(out["list"][1][:5000] - ref_pot[:5000]).max() <= 1e-5 * np.abs(ref_pot[:5000]).max()


def test_tiny_eps2_uses_masked_kernel(nb):
    # eps2 below the threshold of the unmasked loops (and denormal-small): still finite and within tolerance
    w = wl.plummer_workload(700, 1.0 / 64, seed=6)
    for eps2 in (1e-13, 1e-30):
        acc, pot = gpu_force(nb, w.xi, w.x_j, w.m_j, eps2, alias=True)
        ref_acc, ref_pot = oracle.force(w.xi, w.x_j, w.m_j, np.float32(eps2))
        assert np.all(np.isfinite(acc)) and np.all(np.isfinite(pot))
        check_parity(acc, pot, ref_acc, ref_pot, f"eps2={eps2}")


# ------------------------------------------------------------------ edge cases
def test_coincident_and_eps0(nb):
    # same point: a = 0, phi = 0, for eps2 = 0 too (no NaN)
    x = np.array([[1.5, -2.0, 0.25]], dtype=np.float32)
    m = np.array([3.0], dtype=np.float32)
    for eps2 in (0.0, 1e-4):
        acc, pot = gpu_force(nb, x, x, m, eps2)
        assert np.all(acc == 0.0) and pot[0] == 0.0
    # duplicates in the j-set, eps2 = 0, distinct third particle
    xj = np.array([[1, 1, 1], [1, 1, 1], [4, 1, 1]], dtype=np.float32)
    mj = np.array([5.0, 7.0, 2.0], dtype=np.float32)
    xi = np.array([[1, 1, 1]], dtype=np.float32)
    acc, pot = gpu_force(nb, xi, xj, mj, 0.0)
    np.testing.assert_allclose(acc[0], [2.0 / 9.0, 0, 0], rtol=1e-6, atol=1e-12)
    assert pot[0] == pytest.approx(-2.0 / 3.0, rel=1e-6)
    # eps2 = 0 with distinct particles against the oracle
    rng = np.random.default_rng(5)
    x = rng.normal(size=(300, 3)).astype(np.float32)
    mm = rng.uniform(0.5, 1.5, 300).astype(np.float32)
    acc, pot = gpu_force(nb, x, x, mm, 0.0, alias=True)
    ref_acc, ref_pot = oracle.force(x, x, mm, 0.0)
    assert np.all(np.isfinite(acc)) and np.all(np.isfinite(pot))
    check_parity(acc, pot, ref_acc, ref_pot, "eps0")


def test_two_body_exact_cases(nb):
    # d = (3,0,0), eps2 = 16 -> a = 3/125, phi = -1/5  (tests/golden/two_body_exact.txt row 1)
    acc, pot = gpu_force(nb, np.zeros((1, 3), np.float32), np.array([[3, 0, 0]], np.float32),
                         np.array([1.0], np.float32), 16.0)
    np.testing.assert_allclose(acc[0], [3.0 / 125.0, 0, 0], rtol=1e-6, atol=0)
    assert pot[0] == pytest.approx(-0.2, rel=1e-6)


def test_empty_sets(nb):
    import torch
    x = dev(np.ones((5, 3), np.float32))
    m = dev(np.ones(5, np.float32))
    empty_x = torch.empty((0, 3), dtype=torch.float32, device="cuda")
    empty_m = torch.empty((0,), dtype=torch.float32, device="cuda")
    # n_j = 0: outputs zero-filled
    acc = torch.full((5, 3), 7.0, device="cuda")
    pot = torch.full((5,), 7.0, device="cuda")
    nb.force(x, empty_x, empty_m, 0.1, acc_out=acc, pot_out=pot)
    torch.cuda.synchronize()
    assert torch.all(acc == 0) and torch.all(pot == 0)
    # n_i = 0: nothing written, OK
    acc0, pot0 = nb.force(empty_x, x, m, 0.1)
    assert acc0.shape == (0, 3)


def test_pot_null_and_invalid_arguments(nb):
    import torch
    w = wl.plummer_workload(300, 1.0 / 64, seed=3)
    acc, pot = gpu_force(nb, w.xi, w.x_j, w.m_j, w.eps2, want_pot=False)
    assert pot is None
    ref_acc, _ = oracle.force(w.xi, w.x_j, w.m_j, w.eps2)
    check_parity(acc, None, ref_acc, None)
    x, m = dev(w.x_j), dev(w.m_j)
    for bad in (-1.0, float("nan"), float("inf")):
        with pytest.raises(nb.NBError) as ei:
            nb.force(x, x, m, bad)
        assert ei.value.status == 1
    l = nb.lib()
    out = torch.empty((300, 3), device="cuda")
    assert l.nb_force(-1, x.data_ptr(), 300, x.data_ptr(), m.data_ptr(), 0.1, out.data_ptr(), None, None) == 1
    assert l.nb_force(300, None, 300, x.data_ptr(), m.data_ptr(), 0.1, out.data_ptr(), None, None) == 1
    assert l.nb_force(300, x.data_ptr(), 300, x.data_ptr(), m.data_ptr(), 0.1, None, None, None) == 1
    assert l.nb_force(2 ** 31, x.data_ptr(), 300, x.data_ptr(), m.data_ptr(), 0.1, out.data_ptr(), None, None) == 1


# ------------------------------------------------------------------ determinism (P11)
def test_bitwise_reproducible_and_i_permutation_invariant(nb):
    w = wl.subset_workload(6000, 1000, 1.0 / 128, seed=8)
    a1, p1 = gpu_force(nb, w.x_i, w.x_j, w.m_j, w.eps2)
    a2, p2 = gpu_force(nb, w.x_i, w.x_j, w.m_j, w.eps2)
    assert np.array_equal(a1, a2) and np.array_equal(p1, p2)
    perm = np.random.default_rng(0).permutation(1000)
    a3, p3 = gpu_force(nb, w.x_i[perm], w.x_j, w.m_j, w.eps2)
    assert np.array_equal(a3, a1[perm]) and np.array_equal(p3, p1[perm])


def test_momentum_antisymmetry_fp32(nb):
    w = wl.config(0)
    acc, _ = gpu_force(nb, w.xi, w.x_j, w.m_j, w.eps2, alias=True)
    m = w.m_j.astype(np.float64)
    net = np.linalg.norm((m[:, None] * acc.astype(np.float64)).sum(axis=0))
    scale = (m * np.linalg.norm(acc, axis=1)).sum()
    assert net <= 1e-5 * scale


# ------------------------------------------------------------------ host-buffer entry (paper's force())
def test_force_host_matches_device_path(nb):
    w = wl.subset_workload(5000, 600, 1.0 / 128, seed=12)
    acc_h, pot_h = nb.force_host(w.x_i, w.x_j, w.m_j, w.eps2)
    acc_d, pot_d = gpu_force(nb, w.x_i, w.x_j, w.m_j, w.eps2)
    assert np.array_equal(acc_h, acc_d) and np.array_equal(pot_h, pot_d)
    # aliased i == j
    w0 = wl.config(0)
    acc_h, pot_h = nb.force_host(w0.x_j, w0.x_j, w0.m_j, w0.eps2)
    ref_acc, ref_pot = oracle.force(w0.xi, w0.x_j, w0.m_j, w0.eps2)
    check_parity(acc_h, pot_h, ref_acc, ref_pot, "host C0")


# ------------------------------------------------------------------ full-size configs, bench launch configuration
def _sampled_parity(nb, w, n_sample, seed, label):
    import torch
    d_xj, d_mj = dev(w.x_j), dev(w.m_j)
    d_xi = d_xj if w.x_i is None else dev(w.x_i)
    acc, pot = nb.force(d_xi, d_xj, d_mj, w.eps2)
    torch.cuda.synchronize()
    acc, pot = acc.cpu().numpy(), pot.cpu().numpy()
    assert np.all(np.isfinite(acc)) and np.all(np.isfinite(pot))
    idx = np.sort(np.random.default_rng(seed).choice(w.n_i, min(n_sample, w.n_i), replace=False))
    ref_acc, ref_pot = oracle.force(np.ascontiguousarray(w.xi[idx]), w.x_j, w.m_j, w.eps2)
    e = check_parity(acc[idx], pot[idx], ref_acc, ref_pot, label)
    return acc, pot, e


def test_c1_full_size_all_elements(nb):
    """BASELINE.json configs[1] in the launch configuration bench.py times: ALL 131072 outputs against the oracle
    (Eq. (3), and Table 2: the maximum is over all particles).  The full FP64 direct
    sum is 1.7e10 pairs, a few seconds on the GPU box's host cores."""
    w = wl.config(1)
    acc, pot, e = _sampled_parity(nb, w, w.n_i, 1, "C1")
    assert e["acc_max"] < 2e-5                      # paper's blocked FP32 sums: 1.5e-6 at this N; same order
    m = w.m_j.astype(np.float64)
    net = np.linalg.norm((m[:, None] * acc.astype(np.float64)).sum(axis=0))
    assert net <= 1e-5 * (m * np.linalg.norm(acc, axis=1)).sum()
    # P5: Plummer potential energy of the truncated model, W = -0.302443 (1 - 1/N) within 3 sigma
    W = 0.5 * float(np.sum(m * pot.astype(np.float64)))
    n = w.n_j
    assert abs(W / (-0.302443 * (1 - 1.0 / n)) - 1.0) <= 3 * 0.5 / np.sqrt(n)


def test_c2_full_size_all_elements(nb):
    w = wl.config(2)
    acc, pot = gpu_force(nb, w.x_i, w.x_j, w.m_j, w.eps2)
    ref_acc, ref_pot = oracle.force(w.x_i, w.x_j, w.m_j, w.eps2)
    check_parity(acc, pot, ref_acc, ref_pot, "C2")


def test_c3_full_size_sampled(nb):
    w = wl.config(3)
    acc, pot, e = _sampled_parity(nb, w, 4096, 3, "C3")       # 4096 seeded i x all 2^20 j
    m = w.m_j.astype(np.float64)
    net = np.linalg.norm((m[:, None] * acc.astype(np.float64)).sum(axis=0))
    assert net <= 1e-5 * (m * np.linalg.norm(acc, axis=1)).sum()
    # P7: uniform sphere, E[W] = -(3/5)(1 - sum m^2)/R
    W = 0.5 * float(np.sum(m * pot.astype(np.float64)))
    assert abs(W / (-0.6 * (1.0 - float(np.sum(m * m)))) - 1.0) < 0.01


def test_no_potential_variant_gives_the_same_acceleration_bitwise(nb, nbdebug):
    """pot_out = NULL on a large call runs the 12-instruction loop (no phi): a_i is the same, bit for bit."""
    nbdebug.setenv("NB_MASK", "list")
    for plan in ("8,8,1,3", "8,4,2,1", "8,2,4,2", "8,1,8,5"):
        nbdebug.setenv("NB_PLAN", plan)
        w = wl.plummer_workload(3000, 1.0 / 64, seed=17)
        a1, p1 = gpu_force(nb, w.x_j, w.x_j, w.m_j, w.eps2, alias=True)
        a2, p2 = gpu_force(nb, w.x_j, w.x_j, w.m_j, w.eps2, want_pot=False, alias=True)
        assert p2 is None and np.array_equal(a1, a2), plan


@pytest.mark.parametrize("n,mode", [(2048, ""), (3000, "list"), (3000, "exact"), (3000, "bloom"), (9000, "")])
def test_cuda_graph_capture_and_replay(nb, n, mode, nbdebug):
    """include/nbody_b200.h: "once warm the call is CUDA-graph capturable" -- capture nb_force (small-call path with the
    fused second pass; large-call path with the coincidence pre-pass and its memset), replay on new inputs."""
    import torch
    if mode:
        nbdebug.setenv("NB_MASK", mode)
    w = wl.plummer_workload(n, 1.0 / 64, seed=23)
    x, m = dev(w.x_j), dev(w.m_j)
    acc = torch.empty((n, 3), device="cuda"); pot = torch.empty((n,), device="cuda")
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        for _ in range(2):                                             # warm: workspace allocated on this stream
            nb.force(x, x, m, w.eps2, acc_out=acc, pot_out=pot)
        s.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            nb.force(x, x, m, w.eps2, acc_out=acc, pot_out=pot)
    ref = (acc.clone(), pot.clone())
    # new positions in the same buffers, replay twice
    w2 = wl.plummer_workload(n, 1.0 / 64, seed=24)
    x.copy_(dev(w2.x_j))
    acc.zero_(); pot.zero_()
    g.replay(); g.replay()
    torch.cuda.synchronize()
    ra, rp = oracle.force(w2.x_j, w2.x_j, w2.m_j, w2.eps2)
    check_parity(acc.cpu().numpy(), pot.cpu().numpy(), ra, rp, f"graph replay {n} {mode}")
    assert not torch.equal(ref[0], acc)


@pytest.mark.parametrize("n", [700, 3000, 40000])
def test_acceleration_only_calls_need_no_mask(nb, n, nbdebug):
    """pot_out = NULL, eps2 >= 2^-40: the untested loop runs everywhere (no pre-pass); an unmasked coincident pair adds
    +-0 to a, so the result is the masked kernel's bit for bit -- self pairs, duplicates, -0 / subnormal coordinates."""
    nbdebug.setenv("NB_SMALL", "0")
    w = wl.plummer_workload(n, 1.0 / 64, seed=27)
    x = w.x_j.copy()
    x[5] = x[n - 1]; x[n // 2] = x[5]
    x[7] = (0.0, 0.0, 0.0); x[9] = (-0.0, 1e-41, 0.0)
    a_free, p_free = gpu_force(nb, x, x, w.m_j, w.eps2, want_pot=False, alias=True)
    nbdebug.setenv("NB_MASK", "exact")
    a_mask, _ = gpu_force(nb, x, x, w.m_j, w.eps2, alias=True)
    assert p_free is None and np.array_equal(a_free, a_mask)


@pytest.mark.parametrize("n_i,n_j", [(2048, 2048), (512, 8192), (1, 5), (700, 3001), (4096, 4096)])
def test_small_call_direct_pack_path_agrees_bitwise(nb, n_i, n_j, nbdebug):
    """Small calls pack their j sub-ranges inside the force kernel (no nb_pack_j_kernel launch, no TMA): same bits as
    the pack + TMA path (NB_DIRECT=0), one launch fewer."""
    nbdebug.setenv("NB_SMALL", "0")
    w = wl.plummer_workload(max(n_i, n_j), 1.0 / 64, seed=33)
    x_j, m_j, x_i = w.x_j[:n_j], w.m_j[:n_j], w.x_j[:n_i]
    a1, p1 = gpu_force(nb, x_i, x_j, m_j, w.eps2)
    launches_direct = nb.last_launch_count()
    nbdebug.setenv("NB_DIRECT", "0")
    a0, p0 = gpu_force(nb, x_i, x_j, m_j, w.eps2)
    assert nb.last_launch_count() == launches_direct + 1
    assert np.array_equal(a0, a1) and np.array_equal(p0, p1)
    ref_acc, ref_pot = oracle.force(x_i, x_j, m_j, w.eps2)
    if n_i > 1:
        check_parity(a1, p1, ref_acc, ref_pot, f"direct {n_i}x{n_j}")


# ------------------------------------------------------------------ stress cases for the FP32 arithmetic
def test_far_from_the_origin_large_mass_contrast_and_tight_cluster(nb):
    rng = np.random.default_rng(40)
    w = wl.plummer_workload(4000, 1.0 / 64, seed=41)
    # (i) the whole system shifted by ~1000 length units: d = r_j - r_i is still formed exactly from the FP32 inputs
    xs = (w.x_j.astype(np.float64) + np.array([1000.0, -2000.0, 512.0])).astype(np.float32)
    acc, pot = gpu_force(nb, xs, xs, w.m_j, w.eps2, alias=True)
    ra, rp = oracle.force(xs, xs, w.m_j, w.eps2)
    check_parity(acc, pot, ra, rp, "shifted")
    # (ii) masses spread over six decades (a few particles dominate every sum)
    m = (10.0 ** rng.uniform(-6, 0, 4000)).astype(np.float32)
    acc, pot = gpu_force(nb, w.x_j, w.x_j, m, w.eps2, alias=True)
    ra, rp = oracle.force(w.x_j, w.x_j, m, w.eps2)
    check_parity(acc, pot, ra, rp, "mass contrast")
    # (iii) everything inside 1e-3 of a point far from the origin, softening of the same order
    xt = (np.array([3.0, 4.0, 5.0]) + 1e-3 * rng.normal(size=(3000, 3))).astype(np.float32)
    mt = np.full(3000, 1.0 / 3000, np.float32)
    acc, pot = gpu_force(nb, xt, xt, mt, np.float32(1e-6), alias=True)
    ra, rp = oracle.force(xt, xt, mt, np.float32(1e-6))
    check_parity(acc, pot, ra, rp, "tight cluster")


@pytest.mark.parametrize("n_i,n_j", [(200000, 1), (200000, 7), (3, 200000), (1, 1)])
def test_extreme_aspect_ratios(nb, n_i, n_j):
    rng = np.random.default_rng(n_i + n_j)
    xi = rng.normal(size=(n_i, 3)).astype(np.float32)
    xj = rng.normal(size=(n_j, 3)).astype(np.float32)
    mj = rng.uniform(0.5, 1.5, n_j).astype(np.float32)
    acc, pot = gpu_force(nb, xi, xj, mj, 0.01)
    ra, rp = oracle.force(xi, xj, mj, 0.01)
    check_parity(acc, pot, ra, rp, f"{n_i}x{n_j}")


def test_newton_shell_theorem_on_the_gpu(nb):
    """P13 on the CUDA path: a quasi-uniform shell exerts no force inside and M / r^2 outside (eps = 0: masked kernel)."""
    n = 20000
    k = np.arange(n) + 0.5
    z = 1 - 2 * k / n; ph = np.pi * (1 + 5 ** 0.5) * k
    shell = np.stack([np.sqrt(1 - z * z) * np.cos(ph), np.sqrt(1 - z * z) * np.sin(ph), z], 1).astype(np.float32)
    m = np.full(n, 1.0 / n, np.float32)
    probes = np.array([[0, 0, 0], [0.3, -0.2, 0.1], [2, 0, 0], [0, -3, 4]], np.float32)
    acc, pot = gpu_force(nb, probes, shell, m, 0.0)
    assert np.abs(acc[:2]).max() < 1e-4 and np.abs(pot[:2] + 1.0).max() < 1e-5
    r = np.linalg.norm(probes[2:], axis=1)
    np.testing.assert_allclose(acc[2:], -probes[2:] / r[:, None] ** 3, rtol=1e-4, atol=1e-6)
    np.testing.assert_allclose(pot[2:], -1.0 / r, rtol=1e-5)


def test_randomised_shapes_plans_and_modes(nb, nbdebug):
    """40 seeded random cases: ragged sizes, every decomposition the planner could pick, both coincidence modes, with
    and without aliasing, duplicates and phi -- each against the oracle."""
    rng = np.random.default_rng(2024)
    for case in range(40):
        n_j = int(rng.integers(1, 6000))
        alias = bool(rng.integers(0, 2))
        n_i = n_j if alias else int(rng.integers(1, 3000))
        k = int(rng.choice([2, 4, 8])); wj = int(rng.choice([1, 2, 4, 8])); s = int(rng.integers(1, 7))
        mode = str(rng.choice(["exact", "list", "bloom", ""]))
        want_pot = bool(rng.integers(0, 4))
        eps2 = float(np.float32(2.0 ** rng.integers(-16, -2)))
        x_j = rng.normal(size=(n_j, 3)).astype(np.float32)
        m_j = rng.uniform(0.1, 2.0, n_j).astype(np.float32)
        if n_j > 10:
            x_j[rng.integers(0, n_j, 3)] = x_j[0]                      # a few duplicates
        x_i = x_j if alias else np.concatenate([x_j[: min(n_i, n_j) // 2],
                                                rng.normal(size=(n_i - min(n_i, n_j) // 2, 3)).astype(np.float32)])
        nbdebug.setenv("NB_PLAN", f"{k},{8 // wj},{wj},{s}")
        if mode:
            nbdebug.setenv("NB_MASK", mode)
        else:
            nbdebug.delenv("NB_MASK", raising=False)
        acc, pot = gpu_force(nb, x_i, x_j, m_j, eps2, want_pot=want_pot, alias=alias)
        ra, rp = oracle.force(x_i, x_j, m_j, eps2)
        label = f"case {case}: {n_i}x{n_j} plan {k},{8 // wj},{wj},{s} mode '{mode}' alias {alias} pot {want_pot}"
        scale = np.linalg.norm(ra, axis=1)
        ok = scale > 1e-3 * np.median(scale)                           # a particle whose field cancels has no relative error
        e = oracle.error_metrics(acc[ok], ra[ok], None if pot is None else pot[ok], None if pot is None else rp[ok])
        assert e["acc_rms"] <= 1e-5 and e["acc_max"] <= 1e-4, (label, e)
        if pot is not None:
            assert e["pot_rms"] <= 1e-5, (label, e)


@pytest.mark.parametrize("eps2", [0.0, 1.0 / 4096])
def test_signed_zero_coordinates_coincide(nb, eps2):
    """Reading R1 asks for differences that are exactly zero, whatever the signs of the zeros: x_i = +0 against
    x_j = -0 (and the reverse) is a coincident pair.  The kernels hold -x_i with zeros canonicalised to +0, so the
    difference is +0 in all four sign combinations and the bitwise test catches it."""
    rng = np.random.default_rng(21)
    n = 1500
    x = rng.normal(size=(n, 3)).astype(np.float32)
    m = (rng.uniform(0.5, 1.5, n) / n).astype(np.float32)
    x[10] = (0.0, 0.5, -0.0); x[900] = (-0.0, 0.5, 0.0)          # the same point, opposite zero signs
    x[11] = (-0.0, -0.0, -0.0); x[901] = (0.0, 0.0, 0.0); x[1400] = (-0.0, 0.0, -0.0)
    acc, pot = gpu_force(nb, x, x, m, eps2)
    assert np.all(np.isfinite(acc)) and np.all(np.isfinite(pot))
    ref_acc, ref_pot = oracle.force(x, x, m, eps2)
    check_parity(acc, pot, ref_acc, ref_pot, "signed zeros")
    # separate i-set (not aliased), zeros of the other sign
    xi = x[[10, 11, 900, 901, 1400]].copy() * np.float32(-1.0)
    xi[:, 1] = x[[10, 11, 900, 901, 1400], 1]
    acc, pot = gpu_force(nb, xi, x, m, eps2)
    assert np.all(np.isfinite(acc)) and np.all(np.isfinite(pot))
    ref_acc, ref_pot = oracle.force(xi, x, m, eps2)
    check_parity(acc, pot, ref_acc, ref_pot, "signed zeros, separate i")


@pytest.mark.parametrize("n", [4096, 9000])
def test_bloom_mode_lattice_duplicates_and_eps_threshold(nb, n, nbdebug):
    """MODE_BLOOM on inputs that stress the filter: a cubic lattice (few mantissa bits set: weak keys would collide),
    every particle present twice, planar z = +-0, one sub-call direct (one launch) and one through the packed ring;
    the result is the always-masked one bit for bit and within tolerance of the oracle."""
    side = int(round((n / 2) ** (1.0 / 3.0))) + 1
    g = np.stack(np.meshgrid(*[np.arange(side, dtype=np.float32)] * 3, indexing="ij"), -1).reshape(-1, 3)[: n // 2]
    g = g / np.float32(side) - np.float32(0.5)
    g[:, 2] = np.where(np.arange(g.shape[0]) % 2 == 0, np.float32(0.0), np.float32(-0.0)) if n == 4096 else g[:, 2]
    x = np.concatenate([g, g[::-1]]).astype(np.float32)               # every position twice, far apart in j
    rng = np.random.default_rng(5)
    m = (rng.uniform(0.5, 1.5, x.shape[0]) / x.shape[0]).astype(np.float32)
    eps2 = 1.0 / 1024
    for direct in ("1", "0"):
        nbdebug.setenv("NB_DIRECT", direct)
        out = {}
        for mode in ("exact", "bloom"):
            nbdebug.setenv("NB_MASK", mode)
            out[mode] = gpu_force(nb, x, x, m, eps2, alias=True)
        nbdebug.delenv("NB_MASK")
        assert np.array_equal(out["exact"][0], out["bloom"][0]) and np.array_equal(out["exact"][1], out["bloom"][1])
    ref_acc, ref_pot = oracle.force(x, x, m, eps2)
    e = oracle.error_metrics(out["bloom"][0], ref_acc, out["bloom"][1], ref_pot)
    assert e["pot_rms"] <= 1e-5, e                                     # a missed duplicate would shift phi by m / eps
    # lattice forces cancel by symmetry in the interior: compare a absolutely against the typical magnitude
    scale = np.sqrt((ref_acc.astype(np.float64) ** 2).sum(1)).max()
    assert np.abs(out["bloom"][0] - ref_acc).max() <= 1e-5 * scale


@pytest.mark.parametrize("plan", [(8, 8, 1, 5), (4, 2, 4, 3), (2, 1, 8, 7), (8, 4, 2, 2)], ids=lambda p: "K%d_WI%d_WJ%d_S%d" % p)
def test_fused_second_pass_is_bitwise_the_separate_reduce(nb, plan, nbdebug):
    """The sum over the S chunk partials is made in the order s = 0 .. S-1 whoever makes it: the last CTA of an
    i-tile inside the force kernel (ticket counter) or nb_reduce_kernel.  Same bits; repeated calls find the ticket
    counters back at zero."""
    nbdebug.setenv("NB_PLAN", "%d,%d,%d,%d" % plan)
    w = wl.plummer_workload(5000, 1.0 / 64, seed=17)
    out = {}
    for fused in ("1", "0"):
        nbdebug.setenv("NB_FUSED_REDUCE", fused)
        runs = [gpu_force(nb, w.x_j, w.x_j, w.m_j, w.eps2, alias=True) for _ in range(3)]
        for r in runs[1:]:
            assert np.array_equal(r[0], runs[0][0]) and np.array_equal(r[1], runs[0][1])
        out[fused] = runs[0] + (nb.last_launch_count(),)
    assert np.array_equal(out["1"][0], out["0"][0]) and np.array_equal(out["1"][1], out["0"][1])
    assert out["0"][2] == out["1"][2] + 1                              # one launch fewer
    ref_acc, ref_pot = oracle.force(w.x_j, w.x_j, w.m_j, w.eps2)
    check_parity(out["1"][0], out["1"][1], ref_acc, ref_pot, "fused " + str(plan))


@pytest.mark.parametrize("mode", ["exact", "bloom", "list", ""])
def test_ftz_deviation_is_confined_to_subnormal_differences(nb, mode, nbdebug):
    """DESIGN.md reading R1 / include/nbody_b200.h "coordinate range": the kernels run flush-to-zero, so a pair whose
    coordinate differences are all SUBNORMAL (|dx| < 2^-126) may be taken as coincident, which the FP64 oracle does
    not do.  This bounds the deviation from the other side: a difference >= 2^-126 (the smallest normal number) in
    any one coordinate is NEVER treated as coincident, in any mode -- the pair adds -m / eps to phi exactly as the
    oracle says (d^2 underflows against eps2, so r2 = eps2 on both sides).  With coordinates that are 0 or >= 2^-102 in
    magnitude (the supported range) every non-zero difference is >= 2^-125, so there the rule is the oracle's."""
    if mode:
        nbdebug.setenv("NB_MASK", mode)
    tiny = np.float32(2.0 ** -126)
    w = wl.plummer_workload(3000, 1.0 / 64, seed=31)
    x = w.x_j.copy()
    x[10] = (0.0, 0.0, 0.0)
    x[2000] = (tiny, 0.0, 0.0)                      # 2^-126 from particle 10 in x only
    x[11] = (0.0, 1.0, 0.0)
    x[2001] = (0.0, 1.0, -tiny)                     # 2^-126 from particle 11 in z only, negative
    x[12] = (np.float32(2.0 ** -102), 0.5, 0.25)
    x[2002] = (np.float32(2.0 ** -102 * (1 + 2.0 ** -23)), 0.5, 0.25)   # neighbouring floats at the bottom of the range
    acc, pot = gpu_force(nb, x, x, w.m_j, w.eps2, alias=True)
    ref_acc, ref_pot = oracle.force(x, x, w.m_j, w.eps2)
    check_parity(acc, pot, ref_acc, ref_pot, "ftz bound " + mode)
    # the six particles themselves: phi holds the partner's -m / eps (3 % of phi; a masked partner would miss it)
    who = [10, 2000, 11, 2001, 12, 2002]
    assert np.abs(pot[who] / ref_pot[who] - 1.0).max() < 1e-5
    # separate i-set, so that the masked loop sees the difference with both signs
    xi = np.ascontiguousarray(x[who])
    acc, pot = gpu_force(nb, xi, x, w.m_j, w.eps2)
    ref_acc, ref_pot = oracle.force(xi, x, w.m_j, w.eps2)
    assert np.abs(pot / ref_pot - 1.0).max() < 1e-5


def test_concurrent_host_threads_share_the_default_stream_safely(nb):
    """include/nbody_b200.h "threads": the workspace of a (device, stream) is locked while a call grows it and enqueues
    the work that uses it.  Two host threads hammer nb_force_host (both on the default stream, different sizes, so the
    shared staging buffer is re-grown and re-filled all the time) and a third one nb_force on its own stream; every result
    must be the one the same call gives alone, bit for bit."""
    import threading
    import torch
    ws = [wl.subset_workload(3000 + 517 * k, 300 + 91 * k, 1.0 / 128, seed=60 + k) for k in range(4)]
    alone = [nb.force_host(w.x_i, w.x_j, w.m_j, w.eps2) for w in ws]
    errors = []

    def host_worker(offset):
        try:
            for r in range(12):
                k = (r + offset) % 4
                a, p = nb.force_host(ws[k].x_i, ws[k].x_j, ws[k].m_j, ws[k].eps2)
                if not (np.array_equal(a, alone[k][0]) and np.array_equal(p, alone[k][1])):
                    errors.append(("host", offset, r, k))
        except Exception as exc:                                       # pragma: no cover
            errors.append(repr(exc))

    def device_worker():
        try:
            torch.cuda.set_device(0)
            s = torch.cuda.Stream()
            with torch.cuda.stream(s):
                for r in range(12):
                    k = r % 4
                    a, p = nb.force(dev(ws[k].x_i), dev(ws[k].x_j), dev(ws[k].m_j), ws[k].eps2)
                    s.synchronize()
                    if not (np.array_equal(a.cpu().numpy(), alone[k][0]) and np.array_equal(p.cpu().numpy(), alone[k][1])):
                        errors.append(("device", r, k))
            nb.release_stream(s)                                       # the stream's workspace goes with it
        except Exception as exc:                                       # pragma: no cover
            errors.append(repr(exc))

    threads = [threading.Thread(target=host_worker, args=(0,)), threading.Thread(target=host_worker, args=(2,)),
               threading.Thread(target=device_worker)]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    assert not errors, errors[:5]
