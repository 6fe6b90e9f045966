"""nb_hermite4 (shared-time-step 4th-order Hermite on the device, the consumer of nb_force_jerk) against the FP64 oracle
integrator, plus the properties of the scheme at FP32."""
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


def run_gpu(nb, w, dt, steps):
    import torch
    x, v, m = dev(w.x_j.copy()), dev(w.v.copy()), dev(w.m_j)
    acc, jerk, pot = nb.hermite4(x, v, m, w.eps2, dt, steps)
    torch.cuda.synchronize()
    return x.cpu().numpy(), v.cpu().numpy(), acc.cpu().numpy(), jerk.cpu().numpy(), pot.cpu().numpy()


@pytest.mark.usefixtures("both_kernels")
@pytest.mark.parametrize("n,steps", [(300, 20), (1024, 8), (2049, 3)])
def test_matches_oracle_integrator(nb, n, steps):
    w = wl.plummer_workload(n, 1.0 / 64, seed=4, with_velocities=True)
    dt = 1.0 / 256
    x, v, acc, jerk, pot = run_gpu(nb, w, dt, steps)
    xr, vr, ar, jr, pr = oracle.hermite4(w.x_j, w.v, w.m_j, w.eps2, dt, steps)
    assert np.abs(x - xr).max() < 1e-5 and np.abs(v - vr).max() < 1e-5
    e = oracle.error_metrics(acc, ar, pot, pr)
    ej = oracle.error_metrics(jerk, jr)
    assert e["acc_rms"] <= 1e-4 and e["pot_rms"] <= 1e-5 and ej["acc_rms"] <= 1e-3      # values at the FP32 trajectory's state


@pytest.mark.usefixtures("both_kernels")
def test_zero_steps_is_a_force_jerk_evaluation(nb):
    w = wl.plummer_workload(700, 1.0 / 64, seed=5, with_velocities=True)
    x, v, acc, jerk, pot = run_gpu(nb, w, 1.0 / 128, 0)
    assert np.array_equal(x, w.x_j) and np.array_equal(v, w.v)
    ra, rj, rp = oracle.force_jerk(w.x_j, w.v, w.x_j, w.v, w.m_j, w.eps2)
    e = oracle.error_metrics(acc, ra, pot, rp)
    ej = oracle.error_metrics(jerk, rj)
    assert e["acc_rms"] <= 1e-5 and e["acc_max"] <= 1e-4 and e["pot_rms"] <= 1e-5 and ej["acc_rms"] <= 1e-5


@pytest.mark.usefixtures("both_kernels")
def test_energy_error_below_leapfrog_and_momentum(nb):
    import torch
    w = wl.plummer_workload(4096, 1.0 / 32, seed=6, with_velocities=True)
    dt, steps = 1.0 / 64, 64
    _, _, e0 = oracle.energy(w.x_j, w.v, w.m_j, w.eps2)
    xh, vh, _, _, _ = run_gpu(nb, w, dt, steps)
    x, v, m = dev(w.x_j.copy()), dev(w.v.copy()), dev(w.m_j)
    nb.leapfrog_kdk(x, v, m, w.eps2, dt, steps)
    torch.cuda.synchronize()
    _, _, eh = oracle.energy(xh, vh, w.m_j, w.eps2)
    _, _, el = oracle.energy(x.cpu().numpy(), v.cpu().numpy(), w.m_j, w.eps2)
    err_h, err_l = abs(eh - e0) / abs(e0), abs(el - e0) / abs(e0)
    print(f"relative energy error after {steps} steps of dt = 1/64: hermite {err_h:.2e}, leapfrog {err_l:.2e}")
    assert err_h < 2e-6 and err_h < err_l
    p0 = (w.m_j[:, None].astype(np.float64) * w.v).sum(0)
    p1 = (w.m_j[:, None].astype(np.float64) * vh).sum(0)
    assert np.abs(p1 - p0).max() < 1e-6


def test_invalid_arguments(nb):
    L = nb.lib()
    assert L.nb_hermite4(5, None, None, None, 0.1, 0.1, 1, None, None, None, None) == 1
    assert L.nb_hermite4(0, None, None, None, 0.1, 0.1, -1, None, None, None, None) == 1


@pytest.mark.parametrize("n", [1500, 9000])
def test_step_graph_replay_is_bitwise_the_eager_sequence(nb, n, nbdebug):
    """Small systems replay their identical middle steps (predict, force + jerk without phi, correct) from a CUDA
    graph: same launches, same bits as the eager sequence (n = 9000: the Bloom-filter kernel inside the graph)."""
    import torch
    w = wl.plummer_workload(n, 1.0 / 64, seed=8, with_velocities=True)
    out = {}
    side = torch.cuda.Stream()                     # the default stream cannot be captured: graphs need a real stream
    for mode in ("1", "0"):
        nbdebug.setenv("NB_STEP_GRAPH", mode)
        x, v, m = dev(w.x_j.copy()), dev(w.v.copy()), dev(w.m_j)
        torch.cuda.synchronize()
        with torch.cuda.stream(side):
            acc, jerk, pot = nb.hermite4(x, v, m, w.eps2, 1.0 / 256, 85)      # >= 64 steps: the graph is used; 85 leaves left-over steps
        torch.cuda.synchronize()
        out[mode] = (x.cpu().numpy(), v.cpu().numpy(), acc.cpu().numpy(), jerk.cpu().numpy(), pot.cpu().numpy(),
                     nb.last_launch_count())
    for a, b in zip(out["1"][:5], out["0"][:5]):
        assert np.array_equal(a, b)
    assert out["1"][5] == out["0"][5]


@pytest.mark.parametrize("n", [700, 1500, 9000])
def test_fused_correct_predict_is_bitwise_the_two_launches(nb, n, nbdebug):
    """A step closes with ONE kernel that corrects it and predicts + packs the next (two launches per step); with
    NB_HERMITE_FUSE=0 the correction and the prediction are separate launches: the same bits, one launch more per step."""
    import torch
    w = wl.plummer_workload(n, 1.0 / 64, seed=9, with_velocities=True)
    out = {}
    for mode in ("1", "0"):
        nbdebug.setenv("NB_HERMITE_FUSE", mode)
        x, v, m = dev(w.x_j.copy()), dev(w.v.copy()), dev(w.m_j)
        acc, jerk, pot = nb.hermite4(x, v, m, w.eps2, 1.0 / 256, 7)
        torch.cuda.synchronize()
        out[mode] = (x.cpu().numpy(), v.cpu().numpy(), acc.cpu().numpy(), jerk.cpu().numpy(), pot.cpu().numpy(),
                     nb.last_launch_count())
    for a, b in zip(out["1"][:5], out["0"][:5]):
        assert np.array_equal(a, b)
    assert out["0"][5] == out["1"][5] + 6          # steps 0 .. 5 close with two launches instead of one


def test_default_stream_runs_take_the_step_graph_too(nb):
    """As for nb_leapfrog_kdk (test_leapfrog_gpu.py): a long nb_hermite4 run on a default stream is moved to a private stream of
    the device for the call; same bits and launches as on a side stream, and later default-stream work sees the result."""
    import torch
    w = wl.plummer_workload(1500, 1.0 / 64, seed=8, with_velocities=True)
    out = {}
    side = torch.cuda.Stream()
    for where in ("default", "side"):
        x, v, m = dev(w.x_j.copy()), dev(w.v.copy()), dev(w.m_j)
        x.mul_(1.0)
        if where == "side":
            torch.cuda.synchronize()
            with torch.cuda.stream(side):
                acc, jerk, pot = nb.hermite4(x, v, m, w.eps2, 1.0 / 256, 85)
            torch.cuda.synchronize()
            x_after = x.clone()
        else:
            acc, jerk, pot = nb.hermite4(x, v, m, w.eps2, 1.0 / 256, 85)
            x_after = x.clone()
            torch.cuda.synchronize()
        out[where] = (x.cpu().numpy(), v.cpu().numpy(), acc.cpu().numpy(), jerk.cpu().numpy(), pot.cpu().numpy(), x_after.cpu().numpy(),
                      nb.last_launch_count())
    for a, b in zip(out["default"][:6], out["side"][:6]):
        assert np.array_equal(a, b)
    assert np.array_equal(out["default"][0], out["default"][5])
    assert out["default"][6] == out["side"][6]
