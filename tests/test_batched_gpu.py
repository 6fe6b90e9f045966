"""Parity of nb_force_batched (row f2: tree-code interaction lists) against the oracle.

Same tolerances as nb_force (BASELINE.json north_star): acc RMS <= 1e-5, max <= 1e-4; phi RMS <= 1e-5.
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


def gpu_batched(nb, w, want_pot=True, fill=None):
    import torch
    acc = pot = None
    if fill is not None:
        acc = torch.full((w.x_i.shape[0], 3), fill, dtype=torch.float32, device="cuda")
        pot = torch.full((w.x_i.shape[0],), fill, dtype=torch.float32, device="cuda")
    acc, pot = nb.force_batched(dev(w.i_offsets), dev(w.j_offsets), dev(w.x_i), dev(w.x_j), dev(w.m_j), w.eps2,
                                acc_out=acc, pot_out=pot, want_pot=want_pot)
    torch.cuda.synchronize()
    return acc.cpu().numpy(), (None if pot is None else pot.cpu().numpy())


def check(acc, pot, ra, rp, label=""):
    e = oracle.error_metrics(acc, ra, pot, rp)
    assert e["acc_rms"] <= 1e-5 and e["acc_max"] <= 1e-4, (label, e)
    if pot is not None:
        assert e["pot_rms"] <= 1e-5, (label, e)


@pytest.mark.parametrize("tile", ["64", "128", "256", ""])
def test_tree_lists_every_tile_shape(nb, tile, nbdebug):
    if tile:
        nbdebug.setenv("NB_BATCH_TILE", tile)
    w = wl.tree_list_workload(6000, 20, 300, 900, 2500, 1.0 / 128, seed=5)
    acc, pot = gpu_batched(nb, w)
    ra, rp = oracle.force_batched(w.i_offsets, w.j_offsets, w.x_i, w.x_j, w.m_j, w.eps2)
    check(acc, pot, ra, rp, "tile " + tile)
    a_only, none = gpu_batched(nb, w, want_pot=False)         # acceleration only: the untested loop, same bits
    assert none is None and np.array_equal(acc, a_only)


def test_equals_separate_nb_force_calls_within_tolerance_and_masks_own_members(nb):
    w = wl.tree_list_workload(3000, 50, 120, 500, 900, 1.0 / 64, seed=8)
    acc, pot = gpu_batched(nb, w)
    # each group's list starts with its own members: the self term m/eps would shift phi by ~ 0.02 (2 % of |phi|)
    ra, rp = oracle.force_batched(w.i_offsets, w.j_offsets, w.x_i, w.x_j, w.m_j, w.eps2)
    check(acc, pot, ra, rp, "own members")
    import torch
    b = 3
    i0, i1, j0, j1 = (int(v) for v in (w.i_offsets[b], w.i_offsets[b + 1], w.j_offsets[b], w.j_offsets[b + 1]))
    a1, p1 = nb.force(dev(w.x_i[i0:i1]), dev(w.x_j[j0:j1]), dev(w.m_j[j0:j1]), w.eps2)
    torch.cuda.synchronize()
    np.testing.assert_allclose(acc[i0:i1], a1.cpu().numpy(), rtol=2e-5, atol=1e-7)
    np.testing.assert_allclose(pot[i0:i1], p1.cpu().numpy(), rtol=2e-6)


def test_edge_cases_empty_groups_empty_lists_gaps(nb):
    rng = np.random.default_rng(2)
    x_i = rng.normal(size=(700, 3)).astype(np.float32)
    x_j = rng.normal(size=(5000, 3)).astype(np.float32)
    m_j = rng.uniform(0.5, 1.5, 5000).astype(np.float32)
    # sub-problems: normal, empty i-range, empty j-list, 1 x 1, ragged tail; i in [650, 700) belongs to nobody
    i_off = np.array([0, 100, 100, 163, 164, 650], dtype=np.int32)
    j_off = np.array([0, 3000, 3100, 3100, 3101, 4999], dtype=np.int32)
    w = wl.BatchedWorkload("edge", i_off, j_off, x_i, x_j, m_j, 1e-3)
    acc, pot = gpu_batched(nb, w, fill=7.0)
    ra, rp = oracle.force_batched(i_off, j_off, x_i, x_j, m_j, 1e-3)
    assert np.all(acc[100:163] == 0.0) and np.all(pot[100:163] == 0.0)          # empty list -> zeros
    assert np.all(acc[650:] == 7.0) and np.all(pot[650:] == 7.0)                # nobody's particles: untouched
    sel = np.r_[0:100, 163:650]
    check(acc[sel], pot[sel], ra[sel], rp[sel], "edge")
    # n_batch = 0 and invalid arguments
    import torch
    z = torch.zeros((1,), dtype=torch.int32, device="cuda")
    a0, p0 = nb.force_batched(z, z, dev(x_i), dev(x_j), dev(m_j), 1e-3)
    assert nb.lib().nb_force_batched(3, None, None, 10, None, 10, None, None, 0.1, None, None, None) == 1
    with pytest.raises(nb.NBError):
        nb.force_batched(dev(i_off), dev(j_off), dev(x_i), dev(x_j), dev(m_j), -1.0)


def test_eps0(nb):
    w = wl.tree_list_workload(2000, 30, 90, 300, 700, 1.0 / 64, seed=3)
    w0 = wl.BatchedWorkload("eps0", w.i_offsets, w.j_offsets, w.x_i, w.x_j, w.m_j, 0.0)
    acc, pot = gpu_batched(nb, w0)
    ra, rp = oracle.force_batched(w0.i_offsets, w0.j_offsets, w0.x_i, w0.x_j, w0.m_j, 0.0)
    assert np.all(np.isfinite(acc)) and np.all(np.isfinite(pot))
    check(acc, pot, ra, rp, "eps0")


def test_reproducible_and_pot_null(nb):
    w = wl.tree_list_workload(4000, 32, 256, 1000, 3000, 1.0 / 128, seed=6)
    a1, p1 = gpu_batched(nb, w)
    a2, p2 = gpu_batched(nb, w)
    assert np.array_equal(a1, a2) and np.array_equal(p1, p2)
    a3, p3 = gpu_batched(nb, w, want_pot=False)
    assert p3 is None and np.array_equal(a1, a3)


def test_bench_size_sampled(nb):
    """The workload bench.py --op batched times (T1: 524288 particles, 3624 groups of 32..256, lists of 2000..6000),
    same launch configuration: 24 sampled groups against the oracle, and no group left unwritten."""
    w = wl.tree_list_workload(524288, 32, 256, 2000, 6000, 1.0 / 128, seed=7)
    acc, pot = gpu_batched(nb, w, fill=float("nan"))
    assert np.all(np.isfinite(acc)) and np.all(pot < 0.0)
    rng = np.random.default_rng(0)
    for b in rng.choice(w.n_batch, 24, replace=False):
        i0, i1, j0, j1 = (int(v) for v in (w.i_offsets[b], w.i_offsets[b + 1], w.j_offsets[b], w.j_offsets[b + 1]))
        ra, rp = oracle.force(w.x_i[i0:i1], w.x_j[j0:j1], w.m_j[j0:j1], w.eps2)
        check(acc[i0:i1], pot[i0:i1], ra, rp, f"group {b}")


def test_own_members_scattered_through_the_lists_eps0(nb):
    """The kernel decides per 64 j (bounding box of the tile's i-particles) between the masked and the untested loop.
    Here the copies of the i-particles sit at random places of the lists (every part of some lists holds one, many hold
    none), twice each in one group, next to outsiders placed strictly inside the box, with eps = 0 and signed zeros:
    a coincident pair that met the untested loop would give inf/NaN."""
    rng = np.random.default_rng(11)
    n_batch = 12
    ni = rng.integers(1, 200, n_batch)
    ni[0], ni[1], ni[2] = 64, 33, 1
    xi_all, xj_all, mj_all, io, jo = [], [], [], [0], [0]
    for b in range(n_batch):
        centre = rng.normal(size=3) * 3.0
        xi = (centre + rng.uniform(-0.5, 0.5, (ni[b], 3))).astype(np.float32)
        if b == 3:
            xi[:, 0] = np.where(np.arange(ni[b]) % 2 == 0, 0.0, -0.0).astype(np.float32)   # signed zeros, x only
        far = (centre + rng.normal(size=(rng.integers(300, 1500), 3)) * 4.0).astype(np.float32)
        inside = (centre + rng.uniform(-0.4, 0.4, (40, 3))).astype(np.float32)           # in the box, not coincident
        own = xi.copy()
        if b == 3:
            own[:, 0] = -own[:, 0]                                                       # +0 meets -0: still coincident
        parts = [far, inside, own] + ([own] if b == 4 else [])
        xj = np.concatenate(parts)
        perm = rng.permutation(xj.shape[0])
        xj = xj[perm]
        xi_all.append(xi); xj_all.append(xj)
        mj_all.append(rng.uniform(0.5, 1.5, xj.shape[0]).astype(np.float32) / 1000.0)
        io.append(io[-1] + ni[b]); jo.append(jo[-1] + xj.shape[0])
    w = wl.BatchedWorkload("scattered", np.asarray(io, np.int32), np.asarray(jo, np.int32), np.concatenate(xi_all),
                           np.concatenate(xj_all), np.concatenate(mj_all), 0.0)
    acc, pot = gpu_batched(nb, w, fill=float("nan"))
    assert np.all(np.isfinite(acc)) and np.all(np.isfinite(pot))
    ra, rp = oracle.force_batched(w.i_offsets, w.j_offsets, w.x_i, w.x_j, w.m_j, 0.0)
    check(acc, pot, ra, rp, "scattered")
    # with a softening the acceleration-only call (untested loop everywhere) must agree bit for bit
    w1 = wl.BatchedWorkload("scattered-eps", w.i_offsets, w.j_offsets, w.x_i, w.x_j, w.m_j, 1.0 / 4096)
    a1, p1 = gpu_batched(nb, w1)
    a2, _ = gpu_batched(nb, w1, want_pot=False)
    assert np.array_equal(a1, a2)
    ra, rp = oracle.force_batched(w1.i_offsets, w1.j_offsets, w1.x_i, w1.x_j, w1.m_j, w1.eps2)
    check(a1, p1, ra, rp, "scattered-eps")


def test_packed_entry_is_bitwise_the_unpacked_call(nb):
    """nb_force_batched_packed on (x, y, z, m) rows: no pack pass, one launch fewer, the same bits -- with and without phi;
    argument validation as for the unpacked call."""
    import torch
    w = wl.tree_list_workload(5000, 30, 200, 700, 2000, 1.0 / 128, seed=6)
    io, jo, xi, xj, mj = (dev(a) for a in (w.i_offsets, w.j_offsets, w.x_i, w.x_j, w.m_j))
    xm = torch.cat([xj, mj[:, None]], dim=1).contiguous()
    for want_pot in (True, False):
        a0, p0 = nb.force_batched(io, jo, xi, xj, mj, w.eps2, want_pot=want_pot)
        l0 = nb.last_launch_count()
        a1, p1 = nb.force_batched_packed(io, jo, xi, xm, w.eps2, want_pot=want_pot)
        l1 = nb.last_launch_count()
        torch.cuda.synchronize()
        assert l1 == l0 - 1
        assert torch.equal(a0, a1) and (p0 is None or torch.equal(p0, p1))
    ra, rp = oracle.force_batched(w.i_offsets, w.j_offsets, w.x_i, w.x_j, w.m_j, w.eps2)
    check(a1.cpu().numpy(), None, ra, None, "packed")
    lib = nb.lib()
    assert lib.nb_force_batched_packed(1, io.data_ptr(), jo.data_ptr(), 5, xi.data_ptr(), 5, None, 0.1, a1.data_ptr(), None, None) == 1
    assert lib.nb_force_batched_packed(1, io.data_ptr(), jo.data_ptr(), 5, xi.data_ptr(), 5, xm.data_ptr() + 4, 0.1, a1.data_ptr(), None, None) == 1


def test_indexed_entry_is_bitwise_the_expanded_lists(nb):
    """nb_force_batched_indexed: lists as int32 indices into ONE array of packed particle records (what a tree code holds).
    The particle array is the de-duplicated, shuffled set of list records; the result must be bit for bit the one of
    nb_force_batched_packed on the expanded lists (same records, same order, gathered instead of bulk-copied) -- with and
    without phi, for every tile shape -- and within tolerance of the oracle."""
    import torch
    w = wl.tree_list_workload(5000, 30, 200, 700, 2000, 1.0 / 128, seed=6)
    rec = np.concatenate([w.x_j, w.m_j[:, None]], axis=1).astype(np.float32)
    uniq, inverse = np.unique(np.ascontiguousarray(rec).view([("", np.float32)] * 4).ravel(), return_inverse=True)
    perm = np.random.default_rng(1).permutation(uniq.size)
    xm_p = np.ascontiguousarray(uniq.view(np.float32).reshape(-1, 4)[perm])
    where = np.empty(uniq.size, dtype=np.int64); where[perm] = np.arange(uniq.size)
    j_index = where[inverse.ravel()].astype(np.int32)
    assert np.array_equal(xm_p[j_index], rec) and xm_p.shape[0] < rec.shape[0]          # lists share particles
    io, jo, xi = dev(w.i_offsets), dev(w.j_offsets), dev(w.x_i)
    for want_pot in (True, False):
        a0, p0 = nb.force_batched_packed(io, jo, xi, dev(rec), w.eps2, want_pot=want_pot)
        a1, p1 = nb.force_batched_indexed(io, jo, xi, dev(j_index), dev(xm_p), w.eps2, want_pot=want_pot)
        torch.cuda.synchronize()
        assert nb.last_launch_count() == 2
        assert torch.equal(a0, a1) and (p0 is None or torch.equal(p0, p1))
    ra, rp = oracle.force_batched(w.i_offsets, w.j_offsets, w.x_i, w.x_j, w.m_j, w.eps2)
    a1, p1 = nb.force_batched_indexed(io, jo, xi, dev(j_index), dev(xm_p), w.eps2)
    check(a1.cpu().numpy(), p1.cpu().numpy(), ra, rp, "indexed")
    lib = nb.lib()
    assert lib.nb_force_batched_indexed(1, io.data_ptr(), jo.data_ptr(), 5, xi.data_ptr(), 5, None, 5, dev(xm_p).data_ptr(), 0.1, a1.data_ptr(), None, None) == 1
    # ragged: lists of 1 .. 9 entries, tiles of 1 .. 70 particles
    rng = np.random.default_rng(2)
    n_b = 40
    ni = rng.integers(1, 71, n_b); nj = rng.integers(1, 10, n_b)
    io2 = np.concatenate([[0], np.cumsum(ni)]).astype(np.int32); jo2 = np.concatenate([[0], np.cumsum(nj)]).astype(np.int32)
    xp = rng.normal(size=(50, 3)).astype(np.float32); mp = rng.uniform(0.5, 1.5, 50).astype(np.float32)
    idx2 = rng.integers(0, 50, jo2[-1]).astype(np.int32)
    xi2 = rng.normal(size=(io2[-1], 3)).astype(np.float32)
    a2, p2 = nb.force_batched_indexed(dev(io2), dev(jo2), dev(xi2), dev(idx2), dev(np.concatenate([xp, mp[:, None]], 1)), 0.01)
    torch.cuda.synchronize()
    ra, rp = oracle.force_batched(io2, jo2, xi2, xp[idx2], mp[idx2], 0.01)
    check(a2.cpu().numpy(), p2.cpu().numpy(), ra, rp, "indexed ragged")


def test_batched_entries_write_inside_their_bounds_only(nb):
    """Guard bands around acc_out / pot_out for the three batched entries (compute-sanitizer is closed on this pool)."""
    import torch
    w = wl.tree_list_workload(3000, 20, 150, 500, 1500, 1.0 / 128, seed=9)
    io, jo, xi, xj, mj = (dev(a) for a in (w.i_offsets, w.j_offsets, w.x_i, w.x_j, w.m_j))
    xm = torch.cat([xj, mj[:, None]], dim=1).contiguous()
    idx = torch.arange(xm.shape[0], dtype=torch.int32, device="cuda")
    n_i, pad, sentinel = xi.shape[0], 300, -777.0
    calls = (lambda a, p: nb.force_batched(io, jo, xi, xj, mj, w.eps2, acc_out=a, pot_out=p),
             lambda a, p: nb.force_batched_packed(io, jo, xi, xm, w.eps2, acc_out=a, pot_out=p),
             lambda a, p: nb.force_batched_indexed(io, jo, xi, idx, xm, w.eps2, acc_out=a, pot_out=p))
    results = []
    for call in calls:
        big_a = torch.full((n_i + 2 * pad, 3), sentinel, device="cuda")
        big_p = torch.full((n_i + 2 * pad,), sentinel, device="cuda")
        call(big_a[pad:pad + n_i], big_p[pad:pad + n_i])
        torch.cuda.synchronize()
        assert torch.all(big_a[:pad] == sentinel) and torch.all(big_a[pad + n_i:] == sentinel)
        assert torch.all(big_p[:pad] == sentinel) and torch.all(big_p[pad + n_i:] == sentinel)
        assert not torch.any(big_a[pad:pad + n_i] == sentinel) and not torch.any(big_p[pad:pad + n_i] == sentinel)
        results.append((big_a[pad:pad + n_i].clone(), big_p[pad:pad + n_i].clone()))
    for a, p in results[1:]:
        assert torch.equal(a, results[0][0]) and torch.equal(p, results[0][1])
