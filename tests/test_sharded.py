"""Row f4: i-sharded force evaluation and leapfrog.  CPU: slice arithmetic and the world-size-2/3 gloo paths (gather order,
ragged padding with zero-mass records, step sequence) with CPU stand-ins injected for the kernels; GPU: world size 2 on one
device (records exchanged through host memory) and world size 1 through nb_force_packed."""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import pytest

import oracle
from paper_astro_ph_0703100_b200 import sharded, workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_shard_ranges_cover_every_particle_once():
    for n in (0, 1, 7, 1000, 1001, 131072):
        for world in (1, 2, 3, 8):
            r = [sharded.shard_range(n, k, world) for k in range(world)]
            assert r[0][0] == 0 and r[-1][1] == n
            assert all(a[1] == b[0] for a, b in zip(r, r[1:]))
            assert all(hi - lo <= -(-n // world) for lo, hi in r) or n == 0


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _run_worker(nproc, *args, timeout=300):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={nproc}",
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port()),
           os.path.join(ROOT, "tests", "_gloo_shard_worker.py"), *[str(a) for a in args]]
    r = subprocess.run(cmd, cwd=ROOT, env=dict(os.environ, OMP_NUM_THREADS="2"), capture_output=True, text=True, timeout=timeout)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, r.stdout
    return json.loads(lines[0])


@pytest.mark.parametrize("n,nproc", [(1001, 2), (600, 3)])
def test_sharded_force_world_gloo_matches_unsharded_oracle(n, nproc):
    """Host logic at world size 2 and 3 on CPU ranks: the pack, the force (= the oracle) and nothing else injected."""
    d = _run_worker(nproc, "force", "cpu", n)
    assert d["world"] == nproc and d["slices"][-1][1] == n
    # same double-precision sums, only the zero-mass padding records differ: exact agreement
    assert d["acc_max_abs_diff"] == 0.0 and d["pot_max_abs_diff"] == 0.0


@pytest.mark.parametrize("n,nproc,steps", [(601, 2, 5), (300, 3, 4)])
def test_sharded_leapfrog_world_gloo_matches_oracle_integrator(n, nproc, steps):
    """every rank owns its slice of (x, v), one all-gather of the packed records per step.  CPU ranks
    with float64 stand-ins for the kernels: the step sequence (fused double kick, phi only at the end, ragged slices) must
    reproduce the oracle's textbook KDK on the whole system."""
    d = _run_worker(nproc, "leapfrog", "cpu", n, steps)
    assert d["world"] == nproc and d["slices"][-1][1] == n
    # float64 stand-ins, float64 records: the same arithmetic as the oracle's integrator up to the order of a few additions
    assert d["x_max_abs_diff"] <= 1e-12 and d["v_max_abs_diff"] <= 1e-12 and d["acc_rel"] <= 1e-12 and d["pot_rel"] <= 1e-12


@pytest.mark.gpu
@pytest.mark.parametrize("mode,n,steps", [("force", 5001, 0), ("leapfrog", 3001, 6)])
def test_sharded_world2_on_the_device(mode, n, steps):
    """Two ranks, both on cuda:0 (one GPU on the box; NCCL refuses two ranks on one device, so the records travel through
    host memory over gloo): nb_pack_j -> gather -> nb_force_packed (-> nb_kick_drift / nb_kick) on ragged slices with
    zero-mass padding, against the oracle on the whole system."""
    d = _run_worker(2, mode, "cuda", n, steps, timeout=600)
    assert d["world"] == 2 and d["slices"] == [[0, (n + 1) // 2], [(n + 1) // 2, n]]
    if mode == "force":
        assert d["acc_rms"] <= 1e-5 and d["acc_max"] <= 1e-4 and d["pot_rms"] <= 1e-5, d
    else:
        assert d["x_max_abs_diff"] <= 1e-5 and d["v_max_abs_diff"] <= 1e-5 and d["acc_rel"] <= 1e-4 and d["pot_rel"] <= 1e-5, d


@pytest.mark.gpu
def test_packed_entry_and_world1_sharded_force_on_gpu():
    import torch
    import paper_astro_ph_0703100_b200 as nb
    w = wl.plummer_workload(5000, 1.0 / 64, seed=14)
    x, m = torch.from_numpy(w.x_j).cuda(), torch.from_numpy(w.m_j).cuda()
    xm = torch.cat([x, m[:, None]], dim=1).contiguous()
    a0, p0 = nb.force(x, x, m, w.eps2)
    a1, p1 = nb.force_packed(x, xm, w.eps2)
    a2, p2 = sharded.sharded_force(x, m, 5000, w.eps2)
    torch.cuda.synchronize()
    ra, rp = oracle.force(w.x_j, w.x_j, w.m_j, w.eps2)
    for a, p in ((a1, p1), (a2, p2)):
        e = oracle.error_metrics(a.cpu().numpy(), ra, p.cpu().numpy(), rp)
        assert e["acc_rms"] <= 1e-5 and e["acc_max"] <= 1e-4 and e["pot_rms"] <= 1e-5, e
    # packed entry = same kernels on the same records: bitwise equal to nb_force when both mask every pair
    nb.debug_set("NB_MASK", "exact")
    try:
        b0, q0 = nb.force(x, x, m, w.eps2)
        b1, q1 = nb.force_packed(x, xm, w.eps2)
        torch.cuda.synchronize()
    finally:
        nb.debug_set("NB_MASK", None)
    assert torch.equal(b0, b1) and torch.equal(q0, q1)
    # zero-mass padding records add only zeros (the j-chunks move, so the FP32 summation order may differ)
    pad = torch.zeros((37, 4), device="cuda")
    b2, q2 = nb.force_packed(x, torch.cat([xm, pad]).contiguous(), w.eps2)
    torch.cuda.synchronize()
    e = oracle.error_metrics(b2.cpu().numpy(), ra, q2.cpu().numpy(), rp)
    assert e["acc_rms"] <= 1e-5 and e["acc_max"] <= 1e-4 and e["pot_rms"] <= 1e-5, e
    assert torch.allclose(b1, b2, rtol=1e-5, atol=1e-7) and torch.allclose(q1, q2, rtol=1e-6)
    assert nb.lib().nb_force_packed(4, None, 4, None, 0.1, None, None, None) == 1
