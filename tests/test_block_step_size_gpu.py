"""nb_block_step_size (the Aarseth criterion that decides a particle's block level): the value feeds an integer decision,
so both sides compute it in FP32 with individually rounded operations and the comparison is BIT-EXACT."""
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


def gpu(nb, a0, j0, a1, j1, h, eta):
    import torch
    out = nb.block_step_size(dev(a0), dev(j0), dev(a1), dev(j1), dev(h), eta)
    torch.cuda.synchronize()
    return out.cpu().numpy()


def bits(z):
    return np.ascontiguousarray(z, dtype=np.float32).view(np.uint32)


@pytest.mark.parametrize("n,seed", [(1, 0), (255, 1), (256, 2), (257, 3), (5000, 4), (65536, 5)])
def test_bit_exact_on_a_plummer_sphere(nb, n, seed):
    """(a0, j0) at the start state, (a1, j1) after a drift over each particle's own h: all four from the oracle,
    rounded to FP32 -- realistic magnitudes and correlations, nothing from the CUDA path."""
    w = wl.plummer_workload(max(n, 2), 1.0 / 64, seed=50 + seed, with_velocities=True)
    x, v, m = w.x_j[:n], w.v[:n], w.m_j
    h = (2.0 ** -(6.0 + wl.block_levels(n, seed))).astype(np.float32)
    a0, j0, _ = oracle.force_jerk(x, v, w.x_j, w.v, m, w.eps2)
    x1 = (x.astype(np.float64) + v.astype(np.float64) * h[:, None]).astype(np.float32)
    a1, j1, _ = oracle.force_jerk(x1, v, w.x_j, w.v, m, w.eps2)
    args = [z.astype(np.float32) for z in (a0, j0, a1, j1)]
    got = gpu(nb, *args, h, 0.02)
    want = oracle.block_step_size(*args, h, 0.02)
    assert got.dtype == np.float32 and np.array_equal(bits(got), bits(want))
    assert np.isfinite(got).all() and (got > 0).all()
    # the decision it feeds: the block level (power-of-two quantisation) is the same integer on both sides
    assert np.array_equal(np.floor(np.log2(got.astype(np.float64))), np.floor(np.log2(want.astype(np.float64))))


@pytest.mark.parametrize("seed", range(6))
def test_bit_exact_on_random_inputs_over_a_wide_range(nb, seed):
    rng = np.random.default_rng(60 + seed)
    n = int(rng.integers(1, 20000))
    scale = 10.0 ** rng.uniform(-6, 6, size=(4, n, 1))
    a0, j0, a1, j1 = ((rng.normal(size=(n, 3)) * scale[k]).astype(np.float32) for k in range(4))
    h = (2.0 ** -rng.integers(0, 16, n).astype(np.float64)).astype(np.float32)
    if seed % 2:
        h = rng.uniform(1e-4, 1.0, n).astype(np.float32)                # steps that are not powers of two
    eta = float(np.float32(10.0 ** rng.uniform(-3, -1)))
    got = gpu(nb, a0, j0, a1, j1, h, eta)
    want = oracle.block_step_size(a0, j0, a1, j1, h, eta)
    assert np.array_equal(bits(got), bits(want))


def test_degenerate_inputs_follow_ieee(nb):
    """Constant acceleration (a2' = a3 = 0, j = 0): 0/0 -> NaN on both sides; constant jerk: bot = 0, top > 0 -> +inf."""
    a = np.array([[1.0, 2.0, 3.0], [1.0, 0.0, 0.0]], dtype=np.float32)
    j = np.array([[0.0, 0.0, 0.0], [0.5, 0.0, 0.0]], dtype=np.float32)
    h = np.array([0.25, 0.25], dtype=np.float32)
    a1 = a + j * h[:, None]
    got = gpu(nb, a, j, a1, j, h, 0.01)
    want = oracle.block_step_size(a, j, a1, j, h, 0.01)
    assert np.isnan(got[0]) and np.isnan(want[0]) and np.isposinf(got[1]) and np.isposinf(want[1])
    assert nb.last_launch_count() == 1


@pytest.mark.parametrize("n,seed,lev0", [(5000, 4, 3), (5000, 4, 9), (65536, 5, 6)])
def test_against_the_plain_fp64_definition(nb, n, seed, lev0):
    """The kernel against oracle.block_step_size_f64 -- the Aarseth formula in plain FP64 (include/nbody_b200.h) -- by
    tolerance, beside the bit-exact test against the FP32 definition: so the CUDA path is not held only against a
    mirror of its own arithmetic.  Inputs: a Plummer sphere, (a0, j0) at the start, (a1, j1) at each particle's Hermite-
    predicted state after its own h (all four from the oracle, rounded to FP32).  Tolerance: the formula has ~25
    FP32 roundings (2^-24 each) and one cancellation, a0 - a1, which is exact on FP32 inputs of equal exponent
    (|da| / |a| >= 1e-4 here, asserted); 1e-5 relative leaves a factor 10 over the 1e-6 measured with the FP32 oracle
    on the CPU."""
    w = wl.plummer_workload(n, 1.0 / 64, seed=50 + seed, with_velocities=True)
    x, v, m = w.x_j.astype(np.float64), w.v.astype(np.float64), w.m_j
    h = (2.0 ** -(float(lev0) + wl.block_levels(n, seed))).astype(np.float32)
    a0, j0, _ = oracle.force_jerk(w.x_j, w.v, w.x_j, w.v, m, w.eps2)
    hh = h.astype(np.float64)[:, None]
    x1 = (x + v * hh + 0.5 * a0 * hh ** 2 + j0 * hh ** 3 / 6.0).astype(np.float32)
    v1 = (v + a0 * hh + 0.5 * j0 * hh ** 2).astype(np.float32)
    a1, j1, _ = oracle.force_jerk(x1, v1, w.x_j, w.v, m, w.eps2)
    args = [z.astype(np.float32) for z in (a0, j0, a1, j1)]
    da = np.linalg.norm(args[0].astype(np.float64) - args[2], axis=1) / np.linalg.norm(args[0], axis=1)
    assert da.min() >= 1e-4                                             # well conditioned: the stated premise
    got = gpu(nb, *args, h, 0.02).astype(np.float64)
    want = oracle.block_step_size_f64(*args, h, np.float32(0.02))
    rel = np.abs(got / want - 1.0)
    assert rel.max() <= 1e-5, (rel.max(), int(rel.argmax()))
    assert np.sqrt(np.mean(rel * rel)) <= 1e-6
