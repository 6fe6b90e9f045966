"""nb_force_noalloc (include/nbody_b200.h): nb_force for callers that must not allocate device memory -- the scratch of the
j-split is a static __device__ array inside the library, shared by every call on the device.

This file is collected LAST on purpose (the suite runs with `pytest -x`): it checks the entry point against the existing
path (nb_force) on calls made back to back, so that what one call leaves in the shared array cannot change the next one.
Tolerances are the ones every parity test here uses (BASELINE.json north_star; Eq. (3)): acceleration
RMS <= 1e-5, max <= 1e-4; phi RMS <= 1e-5 -- and bit for bit where nb_force runs the same kernel under the same plan.
"""
import os
import re

import numpy as np
import pytest

import oracle
from paper_astro_ph_0703100_b200 import workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def nb():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device (no CPU fallback exists)"
    import paper_astro_ph_0703100_b200 as nb_
    nb_.lib()
    return nb_


def device_case(w):
    import torch
    x_j = torch.from_numpy(np.ascontiguousarray(w.x_j)).cuda()
    m_j = torch.from_numpy(np.ascontiguousarray(w.m_j)).cuda()
    x_i = x_j if w.x_i is None else torch.from_numpy(np.ascontiguousarray(w.x_i)).cuda()
    n_i = x_i.shape[0]
    out = lambda *shape: torch.full(shape, float("nan"), dtype=torch.float32, device="cuda")
    return {"w": w, "x_i": x_i, "x_j": x_j, "m_j": m_j, "acc": out(n_i, 3), "pot": out(n_i), "acc2": out(n_i, 3), "pot2": out(n_i)}


def within_tolerance(acc, pot, ref_acc, ref_pot, label):
    e = oracle.error_metrics(acc, ref_acc, pot, ref_pot)
    assert e["acc_rms"] <= 1e-5 and e["acc_max"] <= 1e-4, (label, e)
    if pot is not None:
        assert e["pot_rms"] <= 1e-5, (label, e)


@pytest.mark.gpu
def test_noalloc_matches_nb_force_on_calls_in_a_row(nb):
    import torch
    a = device_case(wl.subset_workload(65536, 512, 1.0 / 128, seed=2))      # C2's shape: 18 j-chunks, partials + tickets
    b = device_case(wl.subset_workload(20000, 700, 1.0 / 64, seed=31))      # another tile count and j-split
    c = device_case(wl.subset_workload(65536, 4096, 1.0 / 128, seed=32))    # the largest n_i: the planned j-split (37 chunks)
    #                                                                         does not fit the array and is cut to 32
    # back to back on one stream, nothing in between: A, B, A again (into fresh outputs), C
    nb.force_noalloc(a["x_i"], a["x_j"], a["m_j"], a["w"].eps2, a["acc"], a["pot"])
    nb.force_noalloc(b["x_i"], b["x_j"], b["m_j"], b["w"].eps2, b["acc"], b["pot"])
    nb.force_noalloc(a["x_i"], a["x_j"], a["m_j"], a["w"].eps2, a["acc2"], a["pot2"])
    nb.force_noalloc(c["x_i"], c["x_j"], c["m_j"], c["w"].eps2, c["acc"], c["pot"])
    assert nb.last_launch_count() == 1                                      # one kernel per call
    torch.cuda.synchronize()
    for name, t in (("A", a), ("B", b), ("C", c)):
        ref_acc, ref_pot = nb.force(t["x_i"], t["x_j"], t["m_j"], t["w"].eps2)          # the existing path
        torch.cuda.synchronize()
        acc, pot = t["acc"].cpu().numpy(), t["pot"].cpu().numpy()
        assert np.all(np.isfinite(acc)) and np.all(np.isfinite(pot)), name
        within_tolerance(acc, pot, ref_acc.cpu().numpy(), ref_pot.cpu().numpy(), name)
        if name != "C":                                                     # nb_force runs the same kernel under the same plan
            assert nb.plan_query_small(t["w"].n_i, t["w"].n_j)["default"] == 1
            assert np.array_equal(acc, ref_acc.cpu().numpy()) and np.array_equal(pot, ref_pot.cpu().numpy()), name
    # the second call on A found B's partial sums and used tickets in the array: same bits as the first
    assert torch.equal(a["acc"], a["acc2"]) and torch.equal(a["pot"], a["pot2"])
    # and the oracle itself, on the case whose j-split was cut
    idx = np.arange(0, 4096, 16)
    ref_acc, ref_pot = oracle.force(c["w"].x_i[idx], c["w"].x_j, c["w"].m_j, c["w"].eps2)
    within_tolerance(c["acc"].cpu().numpy()[idx], c["pot"].cpu().numpy()[idx], ref_acc, ref_pot, "C against the oracle")


@pytest.mark.gpu
def test_noalloc_without_phi_empty_sets_and_the_limit(nb):
    import torch
    t = device_case(wl.subset_workload(9000, 1500, 1.0 / 64, seed=33))
    nb.force_noalloc(t["x_i"], t["x_j"], t["m_j"], t["w"].eps2, t["acc"], None)             # acceleration only
    nb.force_noalloc(t["x_i"], t["x_j"], t["m_j"], t["w"].eps2, t["acc2"], t["pot2"])
    torch.cuda.synchronize()
    assert torch.equal(t["acc"], t["acc2"])                                 # the unmasked loop stores the same bits
    ref_acc, ref_pot = nb.force(t["x_i"], t["x_j"], t["m_j"], t["w"].eps2)
    within_tolerance(t["acc2"].cpu().numpy(), t["pot2"].cpu().numpy(), ref_acc.cpu().numpy(), ref_pot.cpu().numpy(), "1500 x 9000")
    # n_j == 0: zero-filled; n_i == 0: nothing to do
    empty3, empty1 = torch.empty((0, 3), device="cuda"), torch.empty((0,), device="cuda")
    nb.force_noalloc(t["x_i"], empty3, empty1, 0.01, t["acc"], t["pot"])
    nb.force_noalloc(empty3, t["x_j"], t["m_j"], 0.01, empty3.clone(), empty1.clone())
    torch.cuda.synchronize()
    assert float(t["acc"].abs().max()) == 0.0 and float(t["pot"].abs().max()) == 0.0
    # beyond the limit: a clear error, nothing launched, nothing written
    n_big = nb.NOALLOC_MAX_I + 1
    x_big = torch.zeros((n_big, 3), device="cuda")
    acc_big = torch.full((n_big, 3), 7.0, device="cuda")
    with pytest.raises(nb.NBError) as err:
        nb.force_noalloc(x_big, t["x_j"], t["m_j"], 0.01, acc_big, None)
    assert err.value.status == 5 and "NB_ERR_LIMIT" in str(err.value) and "4096" in str(err.value)
    torch.cuda.synchronize()
    assert float(acc_big.min()) == 7.0 and float(acc_big.max()) == 7.0
    # exactly at the limit it runs
    x_max = t["x_j"][: nb.NOALLOC_MAX_I].contiguous()
    acc_max, pot_max = torch.empty((nb.NOALLOC_MAX_I, 3), device="cuda"), torch.empty((nb.NOALLOC_MAX_I,), device="cuda")
    nb.force_noalloc(x_max, t["x_j"], t["m_j"], t["w"].eps2, acc_max, pot_max)
    ref_acc, ref_pot = nb.force(x_max, t["x_j"], t["m_j"], t["w"].eps2)
    torch.cuda.synchronize()
    within_tolerance(acc_max.cpu().numpy(), pot_max.cpu().numpy(), ref_acc.cpu().numpy(), ref_pot.cpu().numpy(), "4096 x 9000")


@pytest.mark.gpu
def test_noalloc_leaves_free_device_memory_unchanged(nb):
    """Once the kernels of these shapes are loaded, repeating the calls -- and the shapes in another order -- moves the
    device's free memory by nothing: no cudaMalloc, no pool growth, no workspace."""
    import torch
    cases = [device_case(wl.subset_workload(n_j, n_i, 1.0 / 64, seed=40 + k))
             for k, (n_i, n_j) in enumerate([(300, 50000), (2048, 2048), (4096, 30000), (17, 100000)])]
    for t in cases:                                                         # loads the kernels, resolves the array's address
        nb.force_noalloc(t["x_i"], t["x_j"], t["m_j"], t["w"].eps2, t["acc"], t["pot"])
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for t in reversed(cases):
        nb.force_noalloc(t["x_i"], t["x_j"], t["m_j"], t["w"].eps2, t["acc2"], t["pot2"])
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0, (free0, free1)
    for t in cases:
        assert torch.equal(t["acc"], t["acc2"]) and torch.equal(t["pot"], t["pot2"])


def test_noalloc_source_has_no_allocating_call():
    """The entry point's host code, by its text: no cudaMalloc* / cudaFree*, no workspace, no event creation -- and the
    array's device address comes from cudaGetSymbolAddress (in host code the array's name is not a device address)."""
    src = open(os.path.join(ROOT, "paper_astro_ph_0703100_b200", "csrc", "nbody_b200.cu")).read()
    start = src.index("static __device__ __align__(256) unsigned char g_noalloc_scratch")
    body = src[start:src.index("const char* nb_status_string", start)]
    body = re.sub(r"//[^\n]*", "", body)
    for word in ("cudaMalloc", "cudaFree", "ensure(", "WsGuard", "Workspace", "cudaEventCreate", "cudaStreamCreate", "cached_"):
        assert word not in body, word
    assert "cudaGetSymbolAddress(&q, g_noalloc_scratch)" in body
    assert body.count("g_noalloc_scratch") == 2              # the definition and the address query: never passed to a kernel
    header = open(os.path.join(ROOT, "include", "nbody_b200.h")).read()
    assert "#define NB_NOALLOC_MAX_I 4096" in header and "NB_NOALLOC_SCRATCH_BYTES (131072 * 32 + 4096 * 4)" in header
