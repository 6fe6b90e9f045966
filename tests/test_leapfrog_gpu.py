"""nb_leapfrog_kdk (BASELINE.json configs[4]) against the double-precision oracle integrator and
against invariants of the kick-drift-kick scheme.  The KDK scheme is not in the paper (reading R8)."""
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
    return torch.from_numpy(np.ascontiguousarray(a).copy()).cuda()


def run_gpu(nb, w, dt, n_steps):
    import torch
    x, v, m = dev(w.x_j), dev(w.v), dev(w.m_j)
    acc, pot = nb.leapfrog_kdk(x, v, m, w.eps2, dt, n_steps)
    torch.cuda.synchronize()
    return x.cpu().numpy(), v.cpu().numpy(), acc.cpu().numpy(), pot.cpu().numpy()


@pytest.mark.parametrize("n,steps", [(300, 20), (1024, 8), (2049, 3)])
def test_matches_oracle_integrator(nb, n, steps):
    w = wl.plummer_workload(n, 1.0 / 32, seed=40 + n, with_velocities=True)
    dt = 1.0 / 128
    x, v, acc, pot = run_gpu(nb, w, dt, steps)
    xr, vr, ar, pr = oracle.leapfrog_kdk(w.x_j, w.v, w.m_j, w.eps2, dt, steps)
    # FP32 state with |x| <= 10, |v| <~ 1.4: absolute tolerances of a few ulp(10) accumulated over the steps
    assert np.abs(x - xr).max() < 2e-5 and np.abs(v - vr).max() < 2e-5
    e = oracle.error_metrics(acc, ar, pot, pr)
    assert e["acc_rms"] < 1e-4 and e["pot_rms"] < 1e-5


def test_zero_steps_is_a_force_evaluation(nb):
    w = wl.plummer_workload(500, 1.0 / 64, seed=7, with_velocities=True)
    x, v, acc, pot = run_gpu(nb, w, 1.0 / 64, 0)
    assert np.array_equal(x, w.x_j) and np.array_equal(v, w.v)
    ar, pr = oracle.force(w.x_j, w.x_j, w.m_j, w.eps2)
    e = oracle.error_metrics(acc, ar, pot, pr)
    assert e["acc_rms"] <= 1e-5 and e["acc_max"] <= 1e-4 and e["pot_rms"] <= 1e-5


def test_time_reversal_and_momentum(nb):
    import torch
    w = wl.plummer_workload(700, 1.0 / 32, seed=11, with_velocities=True)
    x, v, m = dev(w.x_j), dev(w.v), dev(w.m_j)
    dt, n = 1.0 / 256, 25
    nb.leapfrog_kdk(x, v, m, w.eps2, dt, n)
    v.neg_()
    nb.leapfrog_kdk(x, v, m, w.eps2, dt, n)
    v.neg_()
    torch.cuda.synchronize()
    # KDK is time reversible: back at the start up to FP32 round-off of the state
    assert np.abs(x.cpu().numpy() - w.x_j).max() < 2e-5
    assert np.abs(v.cpu().numpy() - w.v).max() < 2e-5
    # total momentum is conserved to round-off (pairwise antisymmetry of the force)
    x2, v2, _, _ = run_gpu(nb, w, dt, 40)
    mm = w.m_j.astype(np.float64)[:, None]
    p0 = (mm * w.v).sum(axis=0)
    p1 = (mm * v2).sum(axis=0)
    assert np.abs(p1 - p0).max() < 1e-6


def test_softened_circular_binary(nb):
    # masses m at +-d/2, v^2 = m d^2 / (2 (d^2+eps^2)^(3/2)): a circular orbit of the softened two-body problem (pin P12)
    import torch
    m, d, eps2 = 0.5, 1.0, 0.01
    vv = np.sqrt(m * d * d / (2.0 * (d * d + eps2) ** 1.5))
    x0 = np.array([[d / 2, 0, 0], [-d / 2, 0, 0]], dtype=np.float32)
    v0 = np.array([[0, vv, 0], [0, -vv, 0]], dtype=np.float32)
    x, v, mj = dev(x0), dev(v0), dev(np.array([m, m], np.float32))
    omega = np.sqrt(2.0 * m / (d * d + eps2) ** 1.5)
    period = 2.0 * np.pi / omega
    n = 2048
    nb.leapfrog_kdk(x, v, mj, eps2, period / n, n)
    torch.cuda.synchronize()
    xf = x.cpu().numpy()
    r = np.linalg.norm(xf, axis=1)
    assert np.allclose(r, d / 2, atol=1e-4)                        # radius stays put
    assert np.abs(xf - x0).max() < 5e-4                            # back after one period (phase error ~ dt^2)


def test_c4_energy_drift_full_size(nb):
    """BASELINE.json configs[4]: N = 65536, eps = 1/128, dt = 1/512, 1000 steps; relative total-energy drift
    against oracle-force energies evaluated on the GPU's own FP32 state at steps 0 and 1000."""
    import torch
    w = wl.config(4)
    x, v, m = dev(w.x_j), dev(w.v), dev(w.m_j)
    _, _, e0 = oracle.energy(w.x_j, w.v, w.m_j, w.eps2)
    acc, pot = nb.leapfrog_kdk(x, v, m, w.eps2, w.dt, w.n_steps)
    torch.cuda.synchronize()
    xf, vf = x.cpu().numpy(), v.cpu().numpy()
    assert np.all(np.isfinite(xf)) and np.all(np.isfinite(vf))
    t1, w1, e1 = oracle.energy(xf, vf, w.m_j, w.eps2)
    drift = abs(e1 - e0) / abs(e0)
    print(f"C4: E0={e0:.8f} E1000={e1:.8f} drift={drift:.3e} virial 2T/|W|={2 * t1 / abs(w1):.4f}")
    assert drift < 1e-4            # dt^2-scale truncation error of KDK at dt = 1/512; the value itself is unpinned
    # the GPU's own final potential agrees with the oracle's on the final state
    ref_acc, ref_pot = oracle.force(xf[:2048], xf, w.m_j, w.eps2)
    e = oracle.error_metrics(acc.cpu().numpy()[:2048], ref_acc, pot.cpu().numpy()[:2048], ref_pot)
    assert e["acc_rms"] <= 1e-5 and e["acc_max"] <= 1e-4 and e["pot_rms"] <= 1e-5


def test_step_graph_replay_is_bitwise_the_eager_sequence(nb, nbdebug):
    """Small systems replay their identical middle steps from a CUDA graph: same launches, same bits as eager."""
    import torch
    w = wl.plummer_workload(1500, 1.0 / 64, seed=8, with_velocities=True)
    out = {}
    side = torch.cuda.Stream()                     # the default stream cannot be captured: graphs need a real stream
    for mode in ("1", "0"):
        nbdebug.setenv("NB_STEP_GRAPH", mode)
        x, v, m = dev(w.x_j.copy()), dev(w.v.copy()), dev(w.m_j)
        torch.cuda.synchronize()
        with torch.cuda.stream(side):
            acc, pot = nb.leapfrog_kdk(x, v, m, w.eps2, 1.0 / 256, 85)      # >= 64 steps: the graph is used; 85 leaves left-over steps
        torch.cuda.synchronize()
        out[mode] = (x.cpu().numpy(), v.cpu().numpy(), acc.cpu().numpy(), pot.cpu().numpy(), nb.last_launch_count())
    for a, b in zip(out["1"][:4], out["0"][:4]):
        assert np.array_equal(a, b)
    assert out["1"][4] == out["0"][4]


def test_default_stream_runs_take_the_step_graph_too(nb):
    """The default streams cannot be captured: a long run on one is moved to a private stream of the device for the call, with
    the caller's stream order kept (it waits for what was enqueued before, the caller's later work waits for it).  Same bits
    and the same launches as on a side stream; work enqueued on the default stream right after the call sees the result."""
    import torch
    w = wl.plummer_workload(1500, 1.0 / 64, seed=8, with_velocities=True)
    out = {}
    side = torch.cuda.Stream()
    for where in ("default", "side"):
        x, v, m = dev(w.x_j.copy()), dev(w.v.copy()), dev(w.m_j)
        x.mul_(1.0)                                         # work on the default stream just before the call: the run must wait for it
        if where == "side":
            torch.cuda.synchronize()
            with torch.cuda.stream(side):
                acc, pot = nb.leapfrog_kdk(x, v, m, w.eps2, 1.0 / 256, 85)
            torch.cuda.synchronize()
            x_after = x.clone()
        else:
            acc, pot = nb.leapfrog_kdk(x, v, m, w.eps2, 1.0 / 256, 85)
            x_after = x.clone()                             # enqueued on the default stream, no synchronize in between
            torch.cuda.synchronize()
        out[where] = (x.cpu().numpy(), v.cpu().numpy(), acc.cpu().numpy(), pot.cpu().numpy(), x_after.cpu().numpy(), nb.last_launch_count())
    for a, b in zip(out["default"][:5], out["side"][:5]):
        assert np.array_equal(a, b)
    assert np.array_equal(out["default"][0], out["default"][4])
    assert out["default"][5] == out["side"][5]
