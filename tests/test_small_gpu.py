"""The small-i-set kernel (csrc/nb_small.cuh: packed over j, lanes LI x LJ, cluster + ticket reduction of the j-split)
through nb_force against the CPU oracle: every decomposition, ragged shapes, coincident pairs, determinism.

Tolerances are BASELINE.json north_star's (Eq. (3)): acceleration RMS <= 1e-5, max <= 1e-4; phi RMS <= 1e-5.
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


def gpu_force(nb, x_i, x_j, m_j, eps2, want_pot=True, alias=False):
    import torch
    d_xj = dev(x_j)
    d_xi = d_xj if alias else dev(x_i)
    acc, pot = nb.force(d_xi, d_xj, dev(m_j), eps2, want_pot=want_pot)
    torch.cuda.synchronize()
    return acc.cpu().numpy(), (None if pot is None else pot.cpu().numpy())


def check_parity(acc, pot, ref_acc, ref_pot, label=""):
    e = oracle.error_metrics(acc, ref_acc, pot, ref_pot)
    assert e["acc_rms"] <= 1e-5 and e["acc_max"] <= 1e-4, (label, e)
    if pot is not None:
        assert e["pot_rms"] <= 1e-5, (label, e)
    return e


# (NW, KI, LJ) shapes x WJ x (S, CS): every instantiation, with and without the cluster level and the global level
SHAPES = [(16, 2, 1), (8, 2, 1), (16, 1, 1), (8, 1, 1), (8, 1, 2), (8, 1, 4)]
SMALL_PLANS = [(nw, ki, lj, wj, s, cs) for (nw, ki, lj) in SHAPES for wj in (((1, 2, 4, 8, 16) if nw == 16 else (1, 2, 4, 8)) if lj == 1 else (8,))
               for (s, cs) in ((1, 1), (3, 1), (8, 8), (24, 8), (4, 4), (6, 2))
               if ((nw // wj) * ki * (32 // lj)) % cs == 0]
PLAN_FMT = "%d,%d,%d,%d,%d,%d"


@pytest.mark.parametrize("plan", SMALL_PLANS, ids=lambda p: "NW%d_KI%d_LJ%d_WJ%d_S%d_CS%d" % p)
def test_every_small_decomposition_matches_oracle(nb, plan, nbdebug):
    nbdebug.setenv("NB_SMALL", "1")
    nbdebug.setenv("NB_SMALL_PLAN", PLAN_FMT % plan)
    w = wl.subset_workload(3001, 333, 1.0 / 128, seed=21)          # every i coincides with exactly one j
    acc, pot = gpu_force(nb, w.x_i, w.x_j, w.m_j, w.eps2)
    assert nb.last_launch_count() == 1
    ref_acc, ref_pot = oracle.force(w.x_i, w.x_j, w.m_j, w.eps2)
    check_parity(acc, pot, ref_acc, ref_pot, str(plan))
    # masking only the j-pairs marked while staged (Bloom filter of the tile's i-positions; LJ = 1 shapes, the default for
    # large j-chunks) and masking every pair store the same bits
    nbdebug.setenv("NB_SMALL_MASK", "flag")
    acc, pot = gpu_force(nb, w.x_i, w.x_j, w.m_j, w.eps2)
    nbdebug.setenv("NB_SMALL_MASK", "exact")
    acc_e, pot_e = gpu_force(nb, w.x_i, w.x_j, w.m_j, w.eps2)
    nbdebug.delenv("NB_SMALL_MASK")
    assert np.array_equal(acc, acc_e) and np.array_equal(pot, pot_e)
    # acceleration only: the unmasked 12-instruction loop (a coincident pair adds m u^3 (+-0) = +-0); the same sum as the
    # masked loop's bit for bit
    acc2, pot2 = gpu_force(nb, w.x_i, w.x_j, w.m_j, w.eps2, want_pot=False)
    assert pot2 is None and np.array_equal(acc, acc2)
    # repeated calls find the ticket counters back at zero
    acc3, pot3 = gpu_force(nb, w.x_i, w.x_j, w.m_j, w.eps2)
    assert np.array_equal(acc, acc3) and np.array_equal(pot, pot3)


def test_c0_and_c2_take_the_small_kernel_by_default(nb):
    for cfg in (0, 2):
        w = wl.config(cfg)
        assert nb.plan_query_small(w.n_i, w.n_j)["default"] == 1
        acc, pot = gpu_force(nb, w.xi, w.x_j, w.m_j, w.eps2, alias=(w.x_i is None))
        assert nb.last_launch_count() == 1
        ref_acc, ref_pot = oracle.force(w.xi, w.x_j, w.m_j, w.eps2)
        e = check_parity(acc, pot, ref_acc, ref_pot, f"C{cfg}")
        assert e["acc_max"] < 2e-5                                   # paper's blocked sums: ~1e-6 (Table 2)


@pytest.mark.parametrize("n_i,n_j,small", [(4096, 8192, 1), (4097, 8191, 0), (4096, 8193, 0), (512, 131072, 1), (513, 131072, 0),
                                           (3000, 3000, 1), (4096, 2048, 1), (40, 1600000, 1), (32, 4194304, 1), (33, 4194304, 0)])
def test_the_edges_of_the_default_choice(nb, n_i, n_j, small):
    """`small_by_default` (nb_plan.h): n_i <= 512 up to 2^26 pairs, n_i <= 4096 up to 2^25 pairs, n_i <= 32 up to 2^29 pairs.  On both sides of every
    edge nb_force -- no switch set -- matches the oracle on a sample of the i-particles, all of which coincide with a j."""
    assert nb.plan_query_small(n_i, n_j)["default"] == small
    if n_i <= n_j:
        w = wl.subset_workload(n_j, n_i, 1.0 / 256, seed=n_i + n_j)
        x_i = w.x_i
    else:                                                    # more i than j: every j is an i, the rest lie elsewhere
        w = wl.plummer_workload(n_j, 1.0 / 256, seed=n_i + n_j)
        extra = np.random.default_rng(n_i).normal(size=(n_i - n_j, 3)).astype(np.float32)
        x_i = np.ascontiguousarray(np.concatenate([w.x_j, extra]))
    acc, pot = gpu_force(nb, x_i, w.x_j, w.m_j, w.eps2)
    if small:
        assert nb.last_launch_count() == 1
    idx = np.unique(np.concatenate([np.arange(0, n_i, max(1, n_i // 64)), [n_i - 1]]))
    ref_acc, ref_pot = oracle.force(x_i[idx], w.x_j, w.m_j, w.eps2)
    check_parity(acc[idx], pot[idx], ref_acc, ref_pot, f"{n_i}x{n_j}")
    assert np.all(np.isfinite(acc)) and np.all(np.isfinite(pot))


@pytest.mark.parametrize("n_i,n_j", [(1, 1), (1, 777), (3, 200000), (129, 8), (31, 1000), (2048, 3), (1500, 4999),
                                     (17, 4097), (2048, 9000), (64, 70001), (5, 2)])
def test_ragged_shapes_default_plan(nb, n_i, n_j, nbdebug):
    nbdebug.setenv("NB_SMALL", "1")
    rng = np.random.default_rng(n_i * 7919 + n_j)
    x_i = rng.normal(size=(n_i, 3)).astype(np.float32)
    x_j = rng.normal(size=(n_j, 3)).astype(np.float32)
    m_j = (rng.uniform(0.5, 1.5, n_j) / n_j).astype(np.float32)
    acc, pot = gpu_force(nb, x_i, x_j, m_j, 2.0 ** -10)
    ref_acc, ref_pot = oracle.force(x_i, x_j, m_j, np.float32(2.0 ** -10))
    check_parity(acc, pot, ref_acc, ref_pot, f"{n_i}x{n_j}")


def test_coincident_pairs_duplicates_signed_zeros_and_eps0(nb, nbdebug):
    nbdebug.setenv("NB_SMALL", "1")
    w = wl.plummer_workload(1800, 1.0 / 64, seed=12)
    x = w.x_j.copy()
    x[1799] = x[5]; x[900] = x[5]                      # duplicates far apart in j
    x[700] = (0.0, 0.5, -0.0); x[1300] = (-0.0, 0.5, 0.0)   # the same point, opposite zero signs
    x[300] = x[8] + np.float32(1e-7)                   # near, not coincident
    for eps2 in (w.eps2, 0.0, 1e-30):                  
        acc, pot = gpu_force(nb, x, x, w.m_j, eps2, alias=True)
        assert np.all(np.isfinite(acc)) and np.all(np.isfinite(pot))
        ref_acc, ref_pot = oracle.force(x, x, w.m_j, np.float32(eps2))
        check_parity(acc, pot, ref_acc, ref_pot, f"eps2={eps2}")
    # one particle against itself; duplicates in the j-set with eps2 = 0
    one = np.array([[1.5, -2.0, 0.25]], np.float32)
    for eps2 in (0.0, 1e-4):
        acc, pot = gpu_force(nb, one, one, np.array([3.0], np.float32), eps2)
        assert np.all(acc == 0.0) and pot[0] == 0.0
    xj = np.array([[1, 1, 1], [1, 1, 1], [4, 1, 1]], np.float32)
    acc, pot = gpu_force(nb, np.array([[1, 1, 1]], np.float32), xj, np.array([5.0, 7.0, 2.0], np.float32), 0.0)
    np.testing.assert_allclose(acc[0], [2.0 / 9.0, 0, 0], rtol=1e-6, atol=1e-12)
    assert pot[0] == pytest.approx(-2.0 / 3.0, rel=1e-6)


@pytest.mark.parametrize("plan", [(8, 2, 1, 1, 16, 8), (8, 1, 2, 8, 1, 1), (16, 1, 1, 2, 5, 1), (16, 2, 1, 4, 8, 8)],
                         ids=lambda p: "NW%d_KI%d_LJ%d_WJ%d_S%d_CS%d" % p)
def test_bitwise_reproducible_and_i_permutation_invariant(nb, plan, nbdebug):
    """No floating-point atomics, fixed orders at every level (lanes, warps, cluster, tickets): same bits run to run,
    and a particle's result does not depend on where it sits in the i-set."""
    nbdebug.setenv("NB_SMALL", "1")
    nbdebug.setenv("NB_SMALL_PLAN", PLAN_FMT % plan)
    w = wl.subset_workload(6000, 1000, 1.0 / 128, seed=8)
    a1, p1 = gpu_force(nb, w.x_i, w.x_j, w.m_j, w.eps2)
    a2, p2 = gpu_force(nb, w.x_i, w.x_j, w.m_j, w.eps2)
    assert np.array_equal(a1, a2) and np.array_equal(p1, p2)
    perm = np.random.default_rng(0).permutation(1000)
    a3, p3 = gpu_force(nb, w.x_i[perm], w.x_j, w.m_j, w.eps2)
    assert np.array_equal(a3, a1[perm]) and np.array_equal(p3, p1[perm])


def test_packed_entry_and_graph_capture(nb, nbdebug):
    """nb_force_packed on the same records gives the same bits; the one-launch call is CUDA-graph capturable."""
    import torch
    nbdebug.setenv("NB_SMALL", "1")
    w = wl.config(2)
    x_i, x_j, m_j = dev(w.x_i), dev(w.x_j), dev(w.m_j)
    xm = torch.cat([x_j, m_j[:, None]], dim=1).contiguous()
    a0, p0 = nb.force(x_i, x_j, m_j, w.eps2)
    a1, p1 = nb.force_packed(x_i, xm, w.eps2)
    torch.cuda.synchronize()
    assert torch.equal(a0, a1) and torch.equal(p0, p1)
    acc = torch.empty_like(a0); pot = torch.empty_like(p0)
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        for _ in range(2):
            nb.force(x_i, x_j, m_j, w.eps2, acc_out=acc, pot_out=pot)
        s.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            nb.force(x_i, x_j, m_j, w.eps2, acc_out=acc, pot_out=pot)
    acc.zero_(); pot.zero_()
    g.replay(); g.replay()
    torch.cuda.synchronize()
    assert torch.equal(acc, a0) and torch.equal(pot, p0)


def test_randomised_small_cases(nb, nbdebug):
    """30 seeded random cases over shapes, plans, eps2, aliasing, duplicates, with and without phi."""
    nbdebug.setenv("NB_SMALL", "1")
    rng = np.random.default_rng(2025)
    for case in range(30):
        n_j = int(rng.integers(1, 9000))
        alias = bool(rng.integers(0, 2)) and n_j <= 2500
        n_i = n_j if alias else int(rng.integers(1, 2049))
        nw, ki, lj = SHAPES[int(rng.integers(0, 6))]
        wj = int(rng.choice([1, 2, 4, 8] + ([16] if nw == 16 else []))) if lj == 1 else 8
        cs = int(rng.choice([2, 4, 8])) if ((nw // wj) * ki * (32 // lj)) % 8 == 0 and rng.integers(0, 2) else 1
        s = cs * int(rng.integers(1, 5))
        want_pot = bool(rng.integers(0, 4))
        eps2 = float(np.float32(2.0 ** rng.integers(-16, -2)))
        x_j = rng.normal(size=(n_j, 3)).astype(np.float32)
        m_j = rng.uniform(0.1, 2.0, n_j).astype(np.float32)
        if n_j > 10:
            x_j[rng.integers(0, n_j, 3)] = x_j[0]
        x_i = x_j if alias else np.concatenate([x_j[: min(n_i, n_j) // 2],
                                                rng.normal(size=(n_i - min(n_i, n_j) // 2, 3)).astype(np.float32)])
        if rng.integers(0, 2):
            nbdebug.setenv("NB_SMALL_PLAN", f"{nw},{ki},{lj},{wj},{s},{cs}")
        else:
            nbdebug.delenv("NB_SMALL_PLAN")
        acc, pot = gpu_force(nb, x_i, x_j, m_j, eps2, want_pot=want_pot, alias=alias)
        ra, rp = oracle.force(x_i, x_j, m_j, eps2)
        label = f"case {case}: {n_i}x{n_j} plan {nw},{ki},{lj},{wj},{s},{cs} alias {alias} pot {want_pot}"
        scale = np.linalg.norm(ra, axis=1)
        ok = scale > 1e-3 * np.median(scale)                           # a particle whose field cancels has no relative error
        e = oracle.error_metrics(acc[ok], ra[ok], None if pot is None else pot[ok], None if pot is None else rp[ok])
        assert e["acc_rms"] <= 1e-5 and e["acc_max"] <= 1e-4, (label, e)
        if pot is not None:
            assert e["pot_rms"] <= 1e-5, (label, e)


def test_degenerate_positions(nb, nbdebug):
    """Hundreds of identical positions, aliased sets, tiles that are a large part of their own j-chunk."""
    nbdebug.setenv("NB_SMALL", "1")
    rng = np.random.default_rng(4)
    n = 1500
    x = rng.normal(size=(n, 3)).astype(np.float32)
    m = (rng.uniform(0.5, 1.5, n) / n).astype(np.float32)
    x[:900] = (1.0, 2.0, 3.0)
    for plan in ("16,2,1,2,1,1", "8,1,1,8,3,1", None):
        nbdebug.setenv("NB_SMALL_PLAN", plan) if plan else nbdebug.delenv("NB_SMALL_PLAN")
        nbdebug.setenv("NB_SMALL_MASK", "flag")
        acc, pot = gpu_force(nb, x, x, m, 1e-3, alias=True)
        nbdebug.setenv("NB_SMALL_MASK", "exact")
        acc_e, pot_e = gpu_force(nb, x, x, m, 1e-3, alias=True)
        nbdebug.delenv("NB_SMALL_MASK")
        assert np.array_equal(acc, acc_e) and np.array_equal(pot, pot_e)       # every pair marked: same bits as masked everywhere
        ref_acc, ref_pot = oracle.force(x, x, m, 1e-3)
        sel = slice(900, n)                                       # the coincident ones have a ~ 0: compare the others relatively
        check_parity(acc[sel], pot[sel], ref_acc[sel], ref_pot[sel], f"degenerate {plan}")
        assert np.abs(pot[:900] - ref_pot[:900]).max() <= 1e-5 * np.abs(ref_pot[:900]).max()


@pytest.mark.parametrize("n_i,n_j", [(1, 1), (33, 777), (513, 4097), (2048, 2048), (512, 65536), (70, 9001)])
def test_outputs_are_written_inside_their_bounds_only(nb, n_i, n_j, nbdebug):
    """Guard bands (compute-sanitizer is closed on this pool): acc_out / pot_out are slices of larger buffers filled with a
    sentinel; the kernel (default plan and mode, with and without phi) must write every element of the slices and nothing
    around them; the workspace is re-grown from scratch for each shape."""
    import torch
    nbdebug.setenv("NB_SMALL", "1")
    nb.release_workspace()
    w = wl.plummer_workload(max(n_i, n_j), 1.0 / 64, seed=77)
    x_j, m_j, x_i = dev(w.x_j[:n_j]), dev(w.m_j[:n_j]), dev(w.x_j[:n_i] if n_i <= n_j else w.x_j[:n_i])
    pad, sentinel = 257, -12345.0
    for want_pot in (True, False):
        big_a = torch.full((n_i + 2 * pad, 3), sentinel, device="cuda")
        big_p = torch.full((n_i + 2 * pad,), sentinel, device="cuda")
        acc, pot = big_a[pad:pad + n_i], (big_p[pad:pad + n_i] if want_pot else None)
        nb.force(x_i, x_j, m_j, w.eps2, acc_out=acc, pot_out=pot, want_pot=want_pot)
        torch.cuda.synchronize()
        assert torch.all(big_a[:pad] == sentinel) and torch.all(big_a[pad + n_i:] == sentinel)
        assert torch.all(big_p[:pad] == sentinel) and torch.all(big_p[pad + n_i:] == sentinel)
        assert not torch.any(acc == sentinel)
        assert torch.all(big_p[pad:pad + n_i] != sentinel) if want_pot else torch.all(big_p == sentinel)
