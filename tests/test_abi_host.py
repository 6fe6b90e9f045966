"""CPU-only checks of the C-ABI library and its host logic: the shared library loads, exports every symbol
include/nbody_b200.h declares, validates arguments before touching CUDA, fails loudly (never silently succeeds)
without a device, and the launch planner is a sane pure function.  No compute calls are made here."""
import ctypes
import os
import re

import pytest

import paper_astro_ph_0703100_b200 as nb

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    names = set()
    for header in ("nbody_b200.h", "nb_debug.h"):
        text = open(os.path.join(ROOT, "include", header)).read()
        text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
        names |= set(re.findall(r"\b(nb_[a-z0-9_]+)\s*\(", text))
    return sorted(names)


def test_library_exports_every_declared_symbol():
    names = declared_functions()
    assert {"nb_force", "nb_force_host", "nb_leapfrog_kdk", "nb_plan_query", "nb_status_string", "nb_version"} <= set(names)
    lib = nb.lib()
    for name in names:
        assert hasattr(lib, name), f"{name} is declared in include/nbody_b200.h but not exported"
    assert nb.version() >= 100


def test_status_strings():
    for code, word in ((0, "NB_OK"), (1, "INVALID"), (2, "CUDA"), (3, "ALLOC"), (4, "UNSUPPORTED"), (5, "LIMIT")):
        assert word in nb.status_string(code)
    assert "unknown" in nb.status_string(99)


def test_argument_validation_happens_before_any_cuda_call():
    lib = nb.lib()
    buf = (ctypes.c_float * 12)()
    p = ctypes.addressof(buf)
    assert lib.nb_force(-1, p, 1, p, p, 0.1, p, None, None) == 1
    assert lib.nb_force(1, p, 2 ** 31, p, p, 0.1, p, None, None) == 1
    assert lib.nb_force(2 ** 31 - 4096, p, 1, p, p, 0.1, p, None, None) == 1      # largest count is 2^31 - 4097
    assert lib.nb_force(1, None, 1, p, p, 0.1, p, None, None) == 1
    assert lib.nb_force(1, p, 1, p, None, 0.1, p, None, None) == 1
    assert lib.nb_force(1, p, 1, p, p, -0.5, p, None, None) == 1
    assert lib.nb_force(1, p, 1, p, p, float("nan"), p, None, None) == 1
    assert lib.nb_force_host(1, p, 1, p, p, float("inf"), p, None) == 1
    assert lib.nb_leapfrog_kdk(4, p, p, p, 0.1, float("nan"), 1, p, None, None) == 1
    assert lib.nb_leapfrog_kdk(4, p, p, p, 0.1, 0.1, -1, p, None, None) == 1
    assert lib.nb_leapfrog_kdk(4, None, p, p, 0.1, 0.1, 1, p, None, None) == 1
    out = (ctypes.c_int64 * 8)()
    assert lib.nb_plan_query(0, 5, 148, out) == 1
    assert lib.nb_plan_query(5, 5, 148, None) == 1
    # the widened entry points validate the same way
    assert lib.nb_force_jerk(1, p, None, 1, p, p, p, 0.1, p, p, None, None) == 1
    assert lib.nb_force_jerk(1, p, p, 1, p, p, p, -1.0, p, p, None, None) == 1
    assert lib.nb_force_jerk_host(1, p, p, 1, p, p, p, 0.1, p, None, None) == 1
    assert lib.nb_hermite4(4, p, p, p, 0.1, float("inf"), 1, p, p, None, None) == 1
    assert lib.nb_hermite4(4, p, p, p, 0.1, 0.1, 1, p, None, None, None) == 1
    assert lib.nb_hermite4_block_step(4, p, p, p, p, p, p, 5, p, 0.5, 0.1, None) == 1        # n_act > n
    assert lib.nb_hermite4_block_step(4, p, p, p, p, p, None, 2, p, 0.5, 0.1, None) == 1     # no clocks
    assert lib.nb_hermite4_block_step(4, p, p, p, p, p, p, 2, None, 0.5, 0.1, None) == 1     # no active list
    assert lib.nb_hermite4_block_step(4, p, p, p, p, p, p, 2, p, float("nan"), 0.1, None) == 1
    assert lib.nb_hermite4_block_step(4, p, p, p, p, p, p, 2, p, 0.5, -0.1, None) == 1
    assert lib.nb_block_schedule(4, p, None, p, p, p, None) == 1
    assert lib.nb_block_schedule(4, p, p, None, p, p, None) == 1
    assert lib.nb_block_schedule(-1, p, p, p, p, p, None) == 1
    assert lib.nb_block_step_size(4, p, p, p, p, p, 0.0, p, None) == 1                       # eta must be > 0
    assert lib.nb_block_step_size(4, p, p, None, p, p, 0.01, p, None) == 1
    assert lib.nb_force_batched(-1, p, p, 1, p, 1, p, p, 0.1, p, None, None) == 1
    assert lib.nb_force_batched(2, None, p, 1, p, 1, p, p, 0.1, p, None, None) == 1
    assert lib.nb_force_eps_i(1, p, None, 1, p, p, p, None, None) == 1
    assert lib.nb_force_packed(1, p, 1, None, 0.1, p, None, None) == 1
    assert lib.nb_force_packed(1, p, 1, p + 4, 0.1, p, None, None) == 1          # xm_j must be 16-byte aligned
    assert lib.nb_pack_j(1, p, None, p, None) == 1
    assert lib.nb_cunbody_force(p, None, p, 1, 1, None) == 1
    assert lib.nb_cunbody_force_jerk_pot(None, p, p, 1, 1, None) == 1
    assert lib.nb_cunbody_lennard_jones(None, p, p, 1, 1, None) == 1
    assert lib.nb_cunbody_lennard_jones(p, p, p, -1, 1, None) == 1
    assert lib.nb_plan_query_jerk(5, -5, 148, out) == 1


def test_without_a_device_every_compute_entry_reports_an_error():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    lib = nb.lib()
    buf = (ctypes.c_float * 64)()
    p = ctypes.addressof(buf)
    off = (ctypes.c_int32 * 2)(0, 1)
    po = ctypes.addressof(off)
    for st in (lib.nb_force(1, p, 1, p, p, 0.1, p, None, None),
               lib.nb_force_jerk(1, p, p, 1, p, p, p, 0.1, p, p, None, None),
               lib.nb_force_batched(1, po, po, 1, p, 1, p, p, 0.1, p, None, None),
               lib.nb_force_eps_i(1, p, p, 1, p, p, p, None, None),
               lib.nb_force_packed(1, p, 1, p, 0.1, p, None, None),
               lib.nb_leapfrog_kdk(1, p, p, p, 0.1, 0.1, 1, p, None, None),
               lib.nb_hermite4(1, p, p, p, 0.1, 0.1, 1, p, p, None, None),
               lib.nb_hermite4_block_step(1, p, p, p, p, p, p, 1, p, 0.5, 0.1, None),
               lib.nb_block_schedule(1, p, p, p, p, p, None),
               lib.nb_block_step_size(1, p, p, p, p, p, 0.01, p, None),
               lib.nb_cunbody_force(p, p, p, 1, 1, None)):
        assert st in (2, 4), "without a B200 the library must report an error, not compute on the CPU"


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    lib = nb.lib()
    buf = (ctypes.c_float * 12)()
    p = ctypes.addressof(buf)
    st = lib.nb_force_host(1, p, 1, p, p, 0.1, p, None)
    assert st in (2, 4), "without a B200 the library must report an error, not compute on the CPU"


@pytest.mark.parametrize("n_i,n_j", [(1, 1), (1, 777), (31, 1000), (512, 65536), (2048, 2048), (65536, 65536),
                                      (131072, 131072), (1048576, 1048576), (2 ** 31 - 4097, 9)])
def test_planner_invariants(n_i, n_j):
    p = nb.plan_query(n_i, n_j, 148)
    assert p["K"] in (2, 4, 8) and p["WI"] * p["WJ"] == 8 and p["WJ"] in (1, 2, 4, 8)
    assert p["tile_i"] == 32 * p["K"] * p["WI"]
    assert p["tiles_i"] * p["tile_i"] >= n_i > (p["tiles_i"] - 1) * p["tile_i"]
    assert 1 <= p["S"] <= 2048 and p["S"] * p["WJ"] <= max(1, n_j)
    assert p["tile_j"] * 16 * p["stages"] * p["WJ"] <= 200 * 1024            # fits shared memory
    assert p == nb.plan_query(n_i, n_j, 148)                                  # pure function
    assert nb.plan_query(n_i, n_j, 0) == p                                    # sm_count <= 0 means 148


def test_planner_fills_the_machine_for_the_bench_config():
    p = nb.plan_query(131072, 131072, 148)
    ctas = p["tiles_i"] * p["S"]
    assert ctas >= 148 and p["K"] == 8
    waves = ctas / 148.0
    assert waves / -(-ctas // 148) > 0.9                                       # < 10 % wave-quantisation loss


def test_fast_planner_is_the_exhaustive_search_and_costs_microseconds():
    """csrc/nb_plan.h: make_plan visits only the S where the cost's minimum can lie; its choice is DEFINED by the
    exhaustive search over every (K, WJ, S) (nb_debug_plan_exhaustive) and must equal it -- and an unseen shape must cost
    the host a few microseconds, not the 60-220 us of the exhaustive search (a small block step lasts ~20 us)."""
    import time
    import numpy as np
    rng = np.random.default_rng(5)
    sizes = [1, 2, 7, 31, 32, 33, 100, 255, 256, 257, 512, 1000, 2048, 4096, 5000, 16384, 20480, 65536, 131072, 1048576, 20000000]
    shapes = [(a, b) for a in sizes for b in sizes]
    shapes += [(int(np.exp(rng.uniform(0, 16.5))) + 1, int(np.exp(rng.uniform(0, 16.5))) + 1) for _ in range(600)]
    for jerk in (False, True):
        query = nb.plan_query_jerk if jerk else nb.plan_query
        for n_i, n_j in shapes:
            assert query(n_i, n_j, 148) == nb.debug_plan_exhaustive(n_i, n_j, 148, jerk=jerk), (n_i, n_j, jerk)
    lib = nb.lib()
    out = (ctypes.c_int64 * 8)()
    def per_shape(fn):                                        # best of 3 passes: a loaded host must not fail the bound
        best = float("inf")
        for _ in range(3):
            t0 = time.perf_counter()
            for n_i, n_j in shapes:                           # every shape differs: nothing a cache could serve
                fn(n_i, n_j, 148, out)
            best = min(best, (time.perf_counter() - t0) / len(shapes))
        return best
    per_call, per_small = per_shape(lib.nb_plan_query), per_shape(lib.nb_plan_query_small)
    # ~3-5 us + ~0.5 us of ctypes; the small-i-set planner scores ~600 decompositions (~10 us), and its table is keyed by
    # n_i rounded up to a multiple of 8
    assert per_call < 8e-6 and per_small < 20e-6, (per_call, per_small)


def test_small_planner_invariants():
    for n_i, n_j in [(1, 1), (1, 777), (16, 16384), (512, 65536), (2048, 2048), (2048, 65536), (100, 10 ** 6), (3, 5)]:
        p = nb.plan_query_small(n_i, n_j, 148)
        assert (p["KI"], p["LJ"]) in ((2, 1), (1, 1), (1, 2), (1, 4)) and p["WJ"] in (1, 2, 4, 8, 16) and p["NW"] in (8, 16) and p["WJ"] <= p["NW"]
        assert p["tile_i"] == (p["NW"] // p["WJ"]) * p["KI"] * (32 // p["LJ"])
        assert p["tiles_i"] * p["tile_i"] >= n_i > (p["tiles_i"] - 1) * p["tile_i"]
        assert p["CS"] in (1, 2, 4, 8) and p["S"] % p["CS"] == 0 and p["tile_i"] % p["CS"] == 0 and 1 <= p["S"] <= 2048
        assert p == nb.plan_query_small(n_i, n_j, 148)
        q = nb.plan_query_small((n_i + 7) // 8 * 8, n_j, 148)               # the plan depends on n_i through ceil(n_i / 8) only
        assert {k: v for k, v in p.items() if k != "default"} == {k: v for k, v in q.items() if k != "default"}


def test_small_jerk_planner_invariants():
    for n_i, n_j in [(1, 1), (1, 777), (16, 16384), (512, 65536), (2048, 2048), (2048, 65536), (100, 10 ** 6), (3, 5), (4096, 1024)]:
        p = nb.plan_query_small_jerk(n_i, n_j, 148)
        assert (p["NW"], p["LJ"], p["WJ"]) in ((16, 1, 2), (16, 1, 4), (16, 1, 8), (16, 1, 16), (8, 2, 8), (8, 4, 8)) and p["KI"] == 1
        assert p["tile_i"] == (p["NW"] // p["WJ"]) * (32 // p["LJ"])
        assert p["tiles_i"] * p["tile_i"] >= n_i > (p["tiles_i"] - 1) * p["tile_i"]
        assert p["CS"] in (1, 2, 4, 8) and p["S"] % p["CS"] == 0 and p["tile_i"] % p["CS"] == 0 and 1 <= p["S"] <= 2048
        assert p["default_steps"] == int(n_i <= 4096 and (n_i * n_j <= 2 ** 22 or (n_i <= 512 and n_i * n_j <= 2 ** 23)))
        assert p["default"] == int(n_i <= 4096 and (n_i * n_j <= 2 ** 25 or (n_i <= 1024 and n_i * n_j <= 2 ** 26) or
                                                    (n_i <= 256 and n_i * n_j <= 2 ** 28) or (n_i <= 32 and n_i * n_j <= 2 ** 29)))
        assert p == nb.plan_query_small_jerk(n_i, n_j, 148)


def test_debug_switches_parse_and_reject():
    assert nb.lib().nb_debug_set(b"NB_PLAN", b"8,8,1,3") == 0
    assert nb.lib().nb_debug_set(b"NB_PLAN", b"8,8,2,3") == 1           # WI * WJ != 8
    assert nb.lib().nb_debug_set(b"NB_PLAN", None) == 0
    assert nb.lib().nb_debug_set(b"NB_SMALL_PLAN", b"8,1,2,8,8,8") == 0
    assert nb.lib().nb_debug_set(b"NB_SMALL_PLAN", b"8,2,2,8,8,8") == 1   # LJ > 1 needs KI = 1
    assert nb.lib().nb_debug_set(b"NB_SMALL_PLAN", b"8,1,4,8,8,8") == 0   # tile 8, cluster 8
    assert nb.lib().nb_debug_set(b"NB_SMALL_PLAN", b"16,2,1,2,144,8") == 0
    assert nb.lib().nb_debug_set(b"NB_SMALL_PLAN", b"") == 0
    assert nb.lib().nb_debug_set(b"NB_SMALL_JERK_PLAN", b"16,1,8,18,2") == 0
    assert nb.lib().nb_debug_set(b"NB_SMALL_JERK_PLAN", b"16,1,1,18,2") == 1   # WJ = 1 is not instantiated for force + jerk
    assert nb.lib().nb_debug_set(b"NB_SMALL_JERK_PLAN", b"8,4,8,8,4") == 0
    assert nb.lib().nb_debug_set(b"NB_SMALL_JERK_PLAN", b"8,4,8,6,8") == 1     # S is not a multiple of the cluster size
    assert nb.lib().nb_debug_set(b"NB_SMALL_JERK_PLAN", None) == 0
    assert nb.lib().nb_debug_set(b"NB_SMALL_JERK", b"2") == 1
    assert nb.lib().nb_debug_set(b"NB_SMALL_PDL", b"0") == 0
    assert nb.lib().nb_debug_set(b"NB_MASK", b"nonsense") == 1
    assert nb.lib().nb_debug_set(b"NB_NO_SUCH_SWITCH", b"1") == 1
    assert nb.lib().nb_debug_set(None, b"1") == 1
    for key in (b"NB_MASK", b"NB_SMALL", b"NB_SMALL_MASK", b"NB_SMALL_PDL", b"NB_SMALL_JERK", b"NB_SMALL_JERK_PLAN", b"NB_FUSED_REDUCE", b"NB_DIRECT", b"NB_STEP_GRAPH", b"NB_HERMITE_FUSE", b"NB_BATCH_TILE"):
        assert nb.lib().nb_debug_set(key, None) == 0
