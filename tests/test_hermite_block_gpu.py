"""nb_hermite4_block_step (row f4: active-subset integration with block time steps, on top of C2-style force + jerk
calls) against the FP64 oracle's block step on the same seeded state and the same schedule."""
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


def start(nb, w):
    """Device state with a, j of the initial state from nb_force_jerk, oracle state with its own evaluation."""
    x, v, m = dev(w.x_j.copy()), dev(w.v.copy()), dev(w.m_j)
    acc, jerk, _ = nb.force_jerk(x, v, x, v, m, w.eps2)
    ra, rj, _ = oracle.force_jerk(w.x_j, w.v, w.x_j, w.v, w.m_j, w.eps2)
    return (x, v, m, acc, jerk), (w.x_j.astype(np.float64), w.v.astype(np.float64), ra, rj)


def start_shared(w):
    """One FP32 start state for both sides: a, j come from the oracle, rounded to FP32 and uploaded -- no value computed
    by the CUDA path enters the oracle."""
    ra, rj, _ = oracle.force_jerk(w.x_j, w.v, w.x_j, w.v, w.m_j, w.eps2)
    a32, j32 = ra.astype(np.float32), rj.astype(np.float32)
    device = (dev(w.x_j.copy()), dev(w.v.copy()), dev(w.m_j), dev(a32), dev(j32))
    return device, (w.x_j.astype(np.float64), w.v.astype(np.float64), a32.astype(np.float64), j32.astype(np.float64))


def host(*ts):
    import torch
    torch.cuda.synchronize()
    return [t.cpu().numpy() for t in ts]


@pytest.mark.usefixtures("both_kernels")
@pytest.mark.parametrize("n,n_act,seed", [(1500, 1, 0), (1500, 37, 1), (2049, 513, 2), (700, 700, 3), (5000, 2500, 4)])
def test_one_block_step_matches_oracle(nb, n, n_act, seed):
    """Particles sit at different own times (three levels); a ragged, shuffled active set is advanced to t_now."""
    import torch
    w = wl.plummer_workload(n, 1.0 / 64, seed=10 + seed, with_velocities=True)
    (x, v, m, acc, jerk), (xr, vr, ar, jr) = start_shared(w)
    dt = 1.0 / 256
    t0 = -dt * wl.block_levels(n, seed).astype(np.float64)             # own times 0, -dt, -2 dt; t_now = dt
    active = np.random.default_rng(seed).permutation(n)[:n_act].astype(np.int32)
    t = dev(t0.copy())
    before = host(x, v, acc, jerk)
    nb.hermite4_block_step(x, v, m, acc, jerk, t, dev(active), dt, w.eps2)
    gx, gv, ga, gj, gt = host(x, v, acc, jerk, t)
    ox, ov, oa, oj, ot = oracle.hermite4_block_step(xr, vr, w.m_j, ar, jr, t0, active, dt, w.eps2)
    assert np.array_equal(gt, ot)                                                   # clocks: exact
    rest = np.setdiff1d(np.arange(n), active)
    for g, b in zip((gx, gv, ga, gj), before):
        assert np.array_equal(g[rest], b[rest])                                     # inactive rows: bitwise untouched
    assert np.abs(gx - ox).max() < 2e-6 and np.abs(gv - ov).max() < 2e-6
    e = oracle.error_metrics(ga[active], oa[active])
    ej = oracle.error_metrics(gj[active], oj[active])
    assert e["acc_rms"] <= 1e-5 and e["acc_max"] <= 1e-4
    assert ej["acc_rms"] <= 1e-5 and ej["acc_max"] <= 1e-4               # DESIGN.md R16 (measured: 2.6e-6 / 3e-5 at worst)


def test_empty_active_set_is_a_no_op(nb):
    import torch
    w = wl.plummer_workload(300, 1.0 / 64, seed=20, with_velocities=True)
    (x, v, m, acc, jerk), _ = start(nb, w)
    t = dev(np.zeros(300))
    before = host(x, v, acc, jerk, t)
    nb.hermite4_block_step(x, v, m, acc, jerk, t, torch.zeros(0, dtype=torch.int32, device="cuda"), 0.125, w.eps2)
    for g, b in zip(host(x, v, acc, jerk, t), before):
        assert np.array_equal(g, b)
    assert nb.last_launch_count() == 0


@pytest.mark.usefixtures("both_kernels")
def test_all_active_equals_one_shared_step_bitwise(nb):
    """Everybody due at the same time: the block step is one step of nb_hermite4 (same arithmetic, same kernels)."""
    import torch
    n = 1024
    w = wl.plummer_workload(n, 1.0 / 64, seed=21, with_velocities=True)
    dt = 1.0 / 128
    (x, v, m, acc, jerk), _ = start(nb, w)
    t = dev(np.full(n, 0.5))
    nb.hermite4_block_step(x, v, m, acc, jerk, t, torch.arange(n, dtype=torch.int32, device="cuda"), 0.5 + dt, w.eps2)
    x2, v2 = dev(w.x_j.copy()), dev(w.v.copy())
    a2, j2, _ = nb.hermite4(x2, v2, m, w.eps2, dt, 1)
    gx, gv, ga, gj, sx, sv, sa, sj = host(x, v, acc, jerk, x2, v2, a2, j2)
    assert np.array_equal(gx, sx) and np.array_equal(gv, sv) and np.array_equal(ga, sa) and np.array_equal(gj, sj)


@pytest.mark.usefixtures("both_kernels")
@pytest.mark.parametrize("n,sub_steps", [(1200, 8), (4096, 4)])
def test_three_level_schedule_matches_oracle_and_conserves_energy(nb, n, sub_steps):
    """A block-step run: level-L particles are due every 2^L sub-steps; device and oracle follow the same schedule."""
    w = wl.plummer_workload(n, 1.0 / 32, seed=22, with_velocities=True)
    (x, v, m, acc, jerk), (xr, vr, ar, jr) = start(nb, w)
    level = wl.block_levels(n, 5)
    dt = 1.0 / 512
    t, tr = dev(np.zeros(n)), np.zeros(n)
    n_due = []
    for s in range(1, sub_steps + 1):
        active = np.nonzero(s % (1 << level) == 0)[0].astype(np.int32)
        n_due.append(active.size)
        nb.hermite4_block_step(x, v, m, acc, jerk, t, dev(active), s * dt, w.eps2)
        xr, vr, ar, jr, tr = oracle.hermite4_block_step(xr, vr, w.m_j, ar, jr, tr, active, s * dt, w.eps2)
    assert len(set(n_due)) >= 3                                                     # the schedule really has three levels
    gx, gv, ga, gj, gt = host(x, v, acc, jerk, t)
    assert np.array_equal(gt, tr) and np.all(gt == sub_steps * dt)
    assert np.abs(gx - xr).max() < 1e-5 and np.abs(gv - vr).max() < 1e-5
    e = oracle.error_metrics(ga, ar)
    ej = oracle.error_metrics(gj, jr)
    # a, j sit at the FP32 trajectory's own state after up to 8 sub-steps; still inside DESIGN.md R16 (measured 2.5e-6 / 1.5e-5)
    assert e["acc_rms"] <= 1e-5 and e["acc_max"] <= 1e-4 and ej["acc_rms"] <= 1e-5 and ej["acc_max"] <= 1e-4
    _, _, e0 = oracle.energy(w.x_j, w.v, w.m_j, w.eps2)
    _, _, e1 = oracle.energy(gx, gv, w.m_j, w.eps2)
    assert abs(e1 - e0) / abs(e0) < 1e-5


def test_bench_size_block_steps_sampled_against_oracle(nb):
    """bench.py --op block's own configuration (C4's particles, N = 65536, workloads.block_levels(seed=4), list-mode
    force + jerk on n_act x n >= 2^31 pairs): each of the cycle's four due sets is advanced by one block step from the
    same oracle-made FP32 start state with staggered clocks, and checked on 384 sampled due particles -- the oracle
    advances only the sample (a due particle's update does not depend on who else is due)."""
    import torch
    w = wl.config(4)
    n = w.n_j
    level = wl.block_levels(n, seed=4)
    sub_dt = w.dt / 4
    t0 = -sub_dt * ((1 << level) - 1).astype(np.float64)                 # own times 0, -dt/4, -3 dt/4; t_now = dt/4
    (x0, v0, m, a0, j0), (xr, vr, ar, jr) = start_shared(w)
    rng = np.random.default_rng(0)
    for s in range(1, 5):
        active = np.nonzero(s % (1 << level) == 0)[0].astype(np.int32)
        assert active.size * n >= 2 ** 30
        x, v, acc, jerk, t = x0.clone(), v0.clone(), a0.clone(), j0.clone(), dev(t0.copy())
        bx, bv, ba, bj = host(x, v, acc, jerk)
        nb.hermite4_block_step(x, v, m, acc, jerk, t, dev(active), sub_dt, w.eps2)
        gx, gv, ga, gj, gt = host(x, v, acc, jerk, t)
        sample = np.sort(rng.choice(active, 384, replace=False)).astype(np.int32)
        ox, ov, oa, oj, ot = oracle.hermite4_block_step(xr, vr, w.m_j, ar, jr, t0, sample, sub_dt, w.eps2)
        assert np.all(gt[active] == sub_dt) and np.array_equal(gt[sample], ot[sample])
        rest = np.setdiff1d(np.arange(n), active)
        assert np.array_equal(gx[rest], bx[rest]) and np.array_equal(gj[rest], bj[rest]) and np.array_equal(gt[rest], t0[rest])
        assert np.abs(gx[sample] - ox[sample]).max() < 2e-6 and np.abs(gv[sample] - ov[sample]).max() < 2e-6
        e = oracle.error_metrics(ga[sample], oa[sample])
        ej = oracle.error_metrics(gj[sample], oj[sample])
        assert e["acc_rms"] <= 1e-5 and e["acc_max"] <= 1e-4 and ej["acc_rms"] <= 1e-5 and ej["acc_max"] <= 1e-4, (s, e, ej)


@pytest.mark.usefixtures("both_kernels")
def test_order_of_the_active_list_does_not_matter_bitwise(nb):
    """A due particle's sum over j runs in a fixed order wherever the particle sits in the i-set (P11 of SURVEY 8.1.3)."""
    n = 3000
    w = wl.plummer_workload(n, 1.0 / 64, seed=40, with_velocities=True)
    rng = np.random.default_rng(1)
    active = np.sort(rng.permutation(n)[:1111]).astype(np.int32)
    shuffled = rng.permutation(active).astype(np.int32)
    t0 = -(1.0 / 256) * wl.block_levels(n, 8).astype(np.float64)
    outs = []
    for lst in (active, shuffled):
        (x, v, m, acc, jerk), _ = start_shared(w)
        t = dev(t0.copy())
        nb.hermite4_block_step(x, v, m, acc, jerk, t, dev(lst), 1.0 / 256, w.eps2)
        outs.append(host(x, v, acc, jerk, t))
    for a, b in zip(*outs):
        assert np.array_equal(a, b)


@pytest.mark.usefixtures("both_kernels")
def test_coincident_particles_and_zero_softening(nb):
    """eps2 = 0 with exact duplicates among the particles (reading R1: a pair at zero distance adds nothing): finite
    results that match the oracle, for a due particle whose twin is due too and for one whose twin is only predicted."""
    n = 900
    w = wl.plummer_workload(n, 1.0 / 64, seed=41, with_velocities=True)
    x0, v0 = w.x_j.copy(), w.v.copy()
    x0[500:520], v0[500:520] = x0[0:20], v0[0:20]                       # twins: same position and velocity
    ra, rj, _ = oracle.force_jerk(x0, v0, x0, v0, w.m_j, 0.0)
    a32, j32 = ra.astype(np.float32), rj.astype(np.float32)
    assert np.array_equal(a32[500:520], a32[0:20])                       # so the twins stay together when predicted
    x, v, m, acc, jerk = dev(x0), dev(v0), dev(w.m_j), dev(a32), dev(j32)
    t = dev(np.zeros(n))
    active = np.concatenate([np.arange(0, 20), np.arange(500, 510), np.arange(600, 700)]).astype(np.int32)
    nb.hermite4_block_step(x, v, m, acc, jerk, t, dev(active), 1.0 / 512, 0.0)
    gx, gv, ga, gj = host(x, v, acc, jerk)
    ox, ov, oa, oj, _ = oracle.hermite4_block_step(x0, v0, w.m_j, a32, j32, np.zeros(n), active, 1.0 / 512, 0.0)
    assert np.isfinite(ga).all() and np.isfinite(gj).all()
    assert np.abs(gx - ox).max() < 2e-6 and np.abs(gv - ov).max() < 2e-6
    e = oracle.error_metrics(ga[active], oa[active])
    ej = oracle.error_metrics(gj[active], oj[active])
    assert e["acc_rms"] <= 1e-5 and e["acc_max"] <= 1e-4
    assert ej["acc_rms"] <= 1e-5 and ej["acc_max"] <= 1e-4               # DESIGN.md R16 (measured: 2.6e-6 / 3e-5 at worst)


def test_runs_on_a_side_stream_and_in_a_cuda_graph(nb):
    """Asynchronous on the caller's stream; capturable (no synchronisation, no allocation once the workspace is warm)."""
    import torch
    n = 2048
    w = wl.plummer_workload(n, 1.0 / 64, seed=42, with_velocities=True)
    active = dev(np.arange(0, n, 3, dtype=np.int32))
    (x, v, m, acc, jerk), _ = start_shared(w)
    t = dev(np.zeros(n))
    nb.hermite4_block_step(x, v, m, acc, jerk, t, active, 1.0 / 256, w.eps2)
    ref = host(x, v, acc, jerk, t)
    side = torch.cuda.Stream()
    (x, v, m, acc, jerk), _ = start_shared(w)
    t = dev(np.zeros(n))
    keep = [a.clone() for a in (x, v, acc, jerk, t)]
    torch.cuda.synchronize()
    with torch.cuda.stream(side):
        nb.hermite4_block_step(x, v, m, acc, jerk, t, active, 1.0 / 256, w.eps2, stream=side)      # warms this stream's workspace
        side.synchronize()
        for a, b in zip(host(x, v, acc, jerk, t), ref):
            assert np.array_equal(a, b)
        for a, k in zip((x, v, acc, jerk, t), keep):
            a.copy_(k)
        side.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=side):
            nb.hermite4_block_step(x, v, m, acc, jerk, t, active, 1.0 / 256, w.eps2, stream=side)
        for a, k in zip((x, v, acc, jerk, t), keep):                   # capture does not execute: restore and replay once
            a.copy_(k)
        g.replay()
        side.synchronize()
    for a, b in zip(host(x, v, acc, jerk, t), ref):
        assert np.array_equal(a, b)


@pytest.mark.usefixtures("both_kernels")
@pytest.mark.parametrize("case", range(16))
def test_randomised_block_steps(nb, case):
    """Seeded sweep over sizes, due-set sizes, softening (incl. 0), clock staggering and the block time."""
    rng = np.random.default_rng(1000 + case)
    n = int(rng.integers(2, 6000))
    n_act = int(rng.integers(1, n + 1)) if case % 4 else max(1, n // int(rng.integers(20, 200)))
    eps = [0.0, 1.0 / 1024, 1.0 / 64, 0.5][case % 4]
    w = wl.plummer_workload(n, 1.0 / 64, seed=2000 + case, with_velocities=True)
    eps2 = np.float32(eps * eps)
    ra, rj, _ = oracle.force_jerk(w.x_j, w.v, w.x_j, w.v, w.m_j, float(eps2))
    a32, j32 = ra.astype(np.float32), rj.astype(np.float32)
    dt = 2.0 ** -float(rng.integers(7, 11))
    t_now = dt * float(rng.integers(1, 9))
    t0 = t_now - dt * (1 << wl.block_levels(n, 3000 + case, n_levels=int(rng.integers(1, 5)))).astype(np.float64)
    active = rng.permutation(n)[:n_act].astype(np.int32)
    x, v, m, acc, jerk, t = dev(w.x_j.copy()), dev(w.v.copy()), dev(w.m_j), dev(a32), dev(j32), dev(t0.copy())
    nb.hermite4_block_step(x, v, m, acc, jerk, t, dev(active), t_now, float(eps2))
    gx, gv, ga, gj, gt = host(x, v, acc, jerk, t)
    ox, ov, oa, oj, ot = oracle.hermite4_block_step(w.x_j, w.v, w.m_j, a32, j32, t0, active, t_now, float(eps2))
    assert np.array_equal(gt, ot)
    rest = np.setdiff1d(np.arange(n), active)
    assert np.array_equal(gx[rest], w.x_j[rest]) and np.array_equal(ga[rest], a32[rest]) and np.array_equal(gj[rest], j32[rest])
    assert np.abs(gx - ox).max() < 4e-6 and np.abs(gv - ov).max() < 4e-6
    e = oracle.error_metrics(ga[active], oa[active])
    ej = oracle.error_metrics(gj[active], oj[active])
    assert e["acc_rms"] <= 1e-5 and e["acc_max"] <= 1e-4 and ej["acc_rms"] <= 1e-5 and ej["acc_max"] <= 1e-4, (n, n_act, eps, e, ej)
