"""nb_block_schedule (who is due next: index work, bit-exact against the oracle's definition) and a block-step run
driven by it on the device against the same run driven by the oracle's scheduler."""
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


def gpu_schedule(nb, t, dt):
    import torch
    t_next, active, n_act = nb.block_schedule(dev(t), dev(dt))
    torch.cuda.synchronize()
    k = int(n_act.item())
    return float(t_next.item()), active.cpu().numpy()[:k]


def clocks(n, seed, n_levels=5):
    """Clocks on each particle's own dyadic grid (exact in FP64), steps 2^-(3+level)."""
    rng = np.random.default_rng(seed)
    level = rng.integers(0, n_levels, n)
    dt = 2.0 ** -(3.0 + level)
    return dt * rng.integers(0, 6, n), dt


@pytest.mark.parametrize("n", [1, 2, 31, 1023, 1024, 1025, 4097, 100000, 1048576 + 3, 3 * 1048576 + 17])
def test_schedule_is_bit_exact(nb, n):
    t, dt = clocks(n, seed=n)
    t_next, active = gpu_schedule(nb, t, dt)
    rt, ra = oracle.block_schedule(t, dt)
    assert t_next == rt and active.dtype == np.int32 and np.array_equal(active, ra)
    assert nb.last_launch_count() == 5


def test_schedule_degenerate_cases(nb):
    import torch
    # everybody due; one particle due at the very end of the array; nobody there
    n = 5000
    t_next, active = gpu_schedule(nb, np.full(n, 0.25), np.full(n, 0.125))
    assert t_next == 0.375 and np.array_equal(active, np.arange(n, dtype=np.int32))
    t, dt = np.zeros(n), np.full(n, 0.5)
    dt[-1] = 0.25
    t_next, active = gpu_schedule(nb, t, dt)
    assert t_next == 0.25 and active.tolist() == [n - 1]
    t_next, active = gpu_schedule(nb, np.zeros(0), np.zeros(0))
    assert t_next == float("inf") and active.size == 0
    # negative times and steps that are not dyadic: the same FP64 sum on both sides
    rng = np.random.default_rng(3)
    t, dt = rng.normal(size=3000), rng.uniform(0.01, 0.02, 3000)
    t[100] = t[2000] = -7.0
    dt[100] = dt[2000] = 0.3
    t_next, active = gpu_schedule(nb, t, dt)
    rt, ra = oracle.block_schedule(t, dt)
    assert t_next == rt == -7.0 + 0.3 and active.tolist() == ra.tolist() == [100, 2000]
    # repeated calls are deterministic
    again = gpu_schedule(nb, t, dt)
    assert again[0] == t_next and np.array_equal(again[1], active)


def test_block_step_run_driven_by_the_device_scheduler(nb):
    """Three fixed levels; the device loop (schedule -> 4-byte read-back -> block step) and the oracle loop (its own
    scheduler and block step) must pick identical due sets at identical times, and end in the same state."""
    import torch
    n = 1500
    w = wl.plummer_workload(n, 1.0 / 32, seed=30, with_velocities=True)
    x, v, m = dev(w.x_j.copy()), dev(w.v.copy()), dev(w.m_j)
    acc, jerk, _ = nb.force_jerk(x, v, x, v, m, w.eps2)
    xr, vr = w.x_j.astype(np.float64), w.v.astype(np.float64)
    ar, jr, _ = oracle.force_jerk(w.x_j, w.v, w.x_j, w.v, w.m_j, w.eps2)
    dt_host = (1.0 / 512) * 2.0 ** wl.block_levels(n, 6).astype(np.float64)
    t, dt = dev(np.zeros(n)), dev(dt_host)
    tr = np.zeros(n)
    sizes = []
    for _ in range(8):
        t_next, active, n_act = nb.block_schedule(t, dt)
        k = int(n_act.item())                                                 # the 4-byte read-back
        tn = float(t_next.item())
        rt, ra = oracle.block_schedule(tr, dt_host)
        assert tn == rt and np.array_equal(active[:k].cpu().numpy(), ra)
        nb.hermite4_block_step(x, v, m, acc, jerk, t, active[:k], tn, w.eps2)
        xr, vr, ar, jr, tr = oracle.hermite4_block_step(xr, vr, w.m_j, ar, jr, tr, ra, rt, w.eps2)
        sizes.append(k)
    torch.cuda.synchronize()
    assert len(set(sizes)) == 3 and np.array_equal(t.cpu().numpy(), tr) and np.all(tr == 8.0 / 512)
    assert np.abs(x.cpu().numpy() - xr).max() < 1e-5 and np.abs(v.cpu().numpy() - vr).max() < 1e-5


def test_adaptive_block_step_run_with_all_three_calls(nb):
    """A whole block-time-step integration on the device: nb_block_schedule says who is due, nb_hermite4_block_step
    advances them, nb_block_step_size proposes each one's next step; the quantisation to the block grid (halve when the
    criterion asks for less, double only at commensurate times, dt_min <= dt <= dt_max) is the caller's, done here with
    torch on the device.  Properties: every clock ends exactly at t_end, several levels are in use, energy and momentum
    are conserved far better than the step sizes alone would suggest."""
    import torch
    n, eta = 1024, 0.01
    dt_min, dt_max, t_end = 2.0 ** -13, 2.0 ** -6, 2.0 ** -4
    w = wl.plummer_workload(n, 1.0 / 32, seed=31, with_velocities=True)
    x, v, m = dev(w.x_j.copy()), dev(w.v.copy()), dev(w.m_j)
    acc, jerk, _ = nb.force_jerk(x, v, x, v, m, w.eps2)
    t = torch.zeros(n, dtype=torch.float64, device="cuda")
    dt = torch.full((n,), 2.0 ** -10, dtype=torch.float64, device="cuda")
    steps, evaluated, levels_seen = 0, 0, set()
    while True:
        t_next, active, n_act = nb.block_schedule(t, dt)
        tn, k = float(t_next.item()), int(n_act.item())
        if tn > t_end:
            break
        idx = active[:k].long()
        a_old, j_old = acc[idx].contiguous(), jerk[idx].contiguous()
        h = (tn - t[idx]).float()
        nb.hermite4_block_step(x, v, m, acc, jerk, t, active[:k], tn, w.eps2)
        crit = nb.block_step_size(a_old, j_old, acc[idx].contiguous(), jerk[idx].contiguous(), h, eta).double()
        old = dt[idx]
        new = old.clone()
        for _ in range(4):                                                  # halve while the criterion asks for less
            new = torch.where((crit < new) & (new > dt_min), new / 2, new)
        may_double = (crit >= 2 * old) & (2 * old <= dt_max) & (torch.remainder(torch.full_like(old, tn), 2 * old) == 0)
        new = torch.where(may_double, 2 * old, new)
        dt[idx] = new
        steps += 1
        evaluated += k
        levels_seen.update(torch.unique(new).tolist())
        assert steps < 5000
    torch.cuda.synchronize()
    assert torch.all(t == t_end).item()                                     # everybody arrives exactly
    assert len(levels_seen) >= 3 and evaluated < steps * n                  # a real hierarchy, real savings
    gx, gv = x.cpu().numpy(), v.cpu().numpy()
    _, _, e0 = oracle.energy(w.x_j, w.v, w.m_j, w.eps2)
    _, _, e1 = oracle.energy(gx, gv, w.m_j, w.eps2)
    assert abs(e1 - e0) / abs(e0) < 2e-6
    p0 = (w.m_j[:, None] * w.v.astype(np.float64)).sum(0)
    p1 = (w.m_j[:, None] * gv.astype(np.float64)).sum(0)
    assert np.abs(p1 - p0).max() < 1e-6
    print(f"adaptive block run: {steps} block steps, {evaluated} particle evaluations of {steps * n}, "
          f"levels {sorted(levels_seen)}, dE/E = {abs(e1 - e0) / abs(e0):.2e}")


@pytest.mark.parametrize("n", [4, 5000, 70001])
def test_non_finite_due_times_are_never_selected(nb, n):
    """include/nbody_b200.h: "Non-finite due times are never selected (all non-finite: t_next = +inf, n_act = 0)" --
    parked particles (dt = +inf), NaN and -inf clocks, inf - inf; bit-exact against the oracle's definition."""
    inf, nan = float("inf"), float("nan")
    t, dt = clocks(n, seed=7 + n)
    rng = np.random.default_rng(n)
    for value, count in ((inf, n // 3), (nan, max(1, n // 50)), (-inf, max(1, n // 70))):
        who = rng.choice(n, count, replace=False)
        (dt if value == inf else t)[who] = value
    t[0], dt[0] = inf, -inf                                             # inf + (-inf) = NaN
    t_next, active = gpu_schedule(nb, t, dt)
    rt, ra = oracle.block_schedule(t, dt)
    assert np.isfinite(rt) and t_next == rt and np.array_equal(active, ra) and active.size > 0
    due = t[active] + dt[active]
    assert np.all(np.isfinite(due)) and np.all(due == rt)
    # nobody has a finite due time: t_next = +inf, nobody due
    for tt, dd in ((np.zeros(n), np.full(n, inf)), (np.full(n, nan), np.ones(n)), (np.full(n, -inf), np.ones(n))):
        t_next, active = gpu_schedule(nb, tt, dd)
        assert t_next == inf and active.size == 0
