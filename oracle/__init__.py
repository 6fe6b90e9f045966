"""CPU oracle for the all-pairs softened gravity path -- TEST INFRASTRUCTURE, NOT PRODUCT.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  The product
(``paper_astro_ph_0703100_b200``) never imports it, and this package never imports the product.

The arithmetic lives in ``nbody_oracle.c`` (plain C, double precision; see its header for the
passages of PAPER.md each line follows).  This file only builds that C file with gcc and marshals
numpy arrays into it through ctypes -- with two exceptions written out in numpy below: ``block_schedule`` (a minimum and
an equality test, index work) and ``block_step_size`` (a criterion that feeds an integer decision, so it is
defined in the kernel's precision, FP32, one rounded operation at a time).  Parity unpinned: nothing in this package.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading
from typing import Optional, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "nbody_oracle.c")
_SO = os.path.join(_HERE, "libnbody_oracle.so")
_lock = threading.Lock()
_lib = None

GCC_FLAGS = ["-O2", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared", "-std=c99", "-Wall"]


def build(force: bool = False) -> str:
    """Compile nbody_oracle.c -> libnbody_oracle.so (in-tree) if missing or stale."""
    with _lock:
        stale = (not os.path.exists(_SO)) or os.path.getmtime(_SO) < os.path.getmtime(_SRC)
        if force or stale:
            tmp = _SO + f".tmp{os.getpid()}"
            subprocess.run(["gcc", *GCC_FLAGS, "-o", tmp, _SRC, "-lm"], check=True)
            os.replace(tmp, _SO)
    return _SO


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        i64, f32, f64 = ctypes.c_int64, ctypes.c_float, ctypes.c_double
        p = ctypes.c_void_p
        lib.oracle_force_f64.argtypes = [i64, p, i64, p, p, f64, p, p]
        lib.oracle_force_f64.restype = ctypes.c_int
        lib.oracle_force_f32.argtypes = [i64, p, i64, p, p, f32, p, p]
        lib.oracle_force_f32.restype = ctypes.c_int
        lib.oracle_energy_f32.argtypes = [i64, p, p, p, f32, p]
        lib.oracle_energy_f32.restype = ctypes.c_int
        lib.oracle_leapfrog_kdk_f64.argtypes = [i64, p, p, p, f64, f64, i64, p, p]
        lib.oracle_leapfrog_kdk_f64.restype = ctypes.c_int
        lib.oracle_force_jerk_f64.argtypes = [i64, p, p, i64, p, p, p, f64, p, p, p]
        lib.oracle_force_jerk_f64.restype = ctypes.c_int
        lib.oracle_force_jerk_f32.argtypes = [i64, p, p, i64, p, p, p, f32, p, p, p]
        lib.oracle_force_jerk_f32.restype = ctypes.c_int
        lib.oracle_force_eps_i_f64.argtypes = [i64, p, p, i64, p, p, p, p]
        lib.oracle_force_eps_i_f64.restype = ctypes.c_int
        lib.oracle_hermite4_f64.argtypes = [i64, p, p, p, f64, f64, i64, p, p, p]
        lib.oracle_hermite4_f64.restype = ctypes.c_int
        lib.oracle_hermite4_block_step_f64.argtypes = [i64, p, p, p, p, p, p, i64, p, f64, f64]
        lib.oracle_hermite4_block_step_f64.restype = ctypes.c_int
        lib.oracle_lj_f64.argtypes = [i64, p, i64, p, p]
        lib.oracle_lj_f64.restype = ctypes.c_int
        lib.oracle_num_threads.restype = ctypes.c_int
        lib.oracle_set_num_threads.argtypes = [ctypes.c_int]
        _lib = lib
    return _lib


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def set_num_threads(n: int) -> None:
    _load().oracle_set_num_threads(int(n))


def _c(a: np.ndarray, dtype) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=dtype)


def _ptr(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def force(x_i: np.ndarray, x_j: np.ndarray, m_j: np.ndarray, eps2: float,
          want_pot: bool = True) -> Tuple[np.ndarray, Optional[np.ndarray]]:
    """Eq. (1) and phi in double.  float32 inputs are promoted exactly; float64 inputs are used as is.

    Returns (acc float64 [n_i,3], pot float64 [n_i] or None).
    """
    f32 = (x_i.dtype == np.float32 and x_j.dtype == np.float32 and m_j.dtype == np.float32)
    dt = np.float32 if f32 else np.float64
    xi, xj, mj = _c(x_i, dt).reshape(-1, 3), _c(x_j, dt).reshape(-1, 3), _c(m_j, dt).reshape(-1)
    n_i, n_j = xi.shape[0], xj.shape[0]
    if mj.shape[0] != n_j:
        raise ValueError("m_j length != n_j")
    acc = np.zeros((n_i, 3), dtype=np.float64)
    pot = np.zeros(n_i, dtype=np.float64) if want_pot else None
    fn = _load().oracle_force_f32 if f32 else _load().oracle_force_f64
    rc = fn(n_i, _ptr(xi), n_j, _ptr(xj), _ptr(mj), float(eps2), _ptr(acc), _ptr(pot))
    if rc != 0:
        raise ValueError(f"oracle_force returned {rc}")
    return acc, pot


def force_jerk(x_i: np.ndarray, v_i: np.ndarray, x_j: np.ndarray, v_j: np.ndarray, m_j: np.ndarray, eps2: float,
               want_pot: bool = True):
    """Force + jerk + potential of Fig. A.4 in double.  float32 inputs are promoted exactly.

    Returns (acc [n_i,3], jerk [n_i,3], pot [n_i] or None), all float64.
    """
    arrs = (x_i, v_i, x_j, v_j, m_j)
    f32 = all(a.dtype == np.float32 for a in arrs)
    dt = np.float32 if f32 else np.float64
    xi, vi = _c(x_i, dt).reshape(-1, 3), _c(v_i, dt).reshape(-1, 3)
    xj, vj, mj = _c(x_j, dt).reshape(-1, 3), _c(v_j, dt).reshape(-1, 3), _c(m_j, dt).reshape(-1)
    n_i, n_j = xi.shape[0], xj.shape[0]
    if vi.shape[0] != n_i or vj.shape[0] != n_j or mj.shape[0] != n_j:
        raise ValueError("array lengths differ")
    acc = np.zeros((n_i, 3), dtype=np.float64)
    jerk = np.zeros((n_i, 3), dtype=np.float64)
    pot = np.zeros(n_i, dtype=np.float64) if want_pot else None
    fn = _load().oracle_force_jerk_f32 if f32 else _load().oracle_force_jerk_f64
    rc = fn(n_i, _ptr(xi), _ptr(vi), n_j, _ptr(xj), _ptr(vj), _ptr(mj), float(eps2), _ptr(acc), _ptr(jerk), _ptr(pot))
    if rc != 0:
        raise ValueError(f"oracle_force_jerk returned {rc}")
    return acc, jerk, pot


def force_eps_i(x_i: np.ndarray, eps2_i: np.ndarray, x_j: np.ndarray, m_j: np.ndarray, want_pot: bool = True):
    """Row f3: Eq. (1) and phi with one eps^2 per i-particle (Fig. A.1).  Inputs (float32 or
    float64) are promoted exactly to double.  Returns (acc [n_i,3], pot [n_i] or None) in float64."""
    xi, xj = _c(x_i, np.float64).reshape(-1, 3), _c(x_j, np.float64).reshape(-1, 3)
    e2, mj = _c(eps2_i, np.float64).reshape(-1), _c(m_j, np.float64).reshape(-1)
    n_i, n_j = xi.shape[0], xj.shape[0]
    if e2.shape[0] != n_i or mj.shape[0] != n_j:
        raise ValueError("array lengths differ")
    acc = np.zeros((n_i, 3), dtype=np.float64)
    pot = np.zeros(n_i, dtype=np.float64) if want_pot else None
    rc = _load().oracle_force_eps_i_f64(n_i, _ptr(xi), _ptr(e2), n_j, _ptr(xj), _ptr(mj), _ptr(acc), _ptr(pot))
    if rc != 0:
        raise ValueError(f"oracle_force_eps_i returned {rc}")
    return acc, pot


def lennard_jones(p_xi: np.ndarray, p_xj: np.ndarray) -> np.ndarray:
    """Row f3, reading R19: 12-6 Lennard-Jones with Lorentz-Berthelot mixing, all pairs.  Rows
    p_xi [n_i, 5] = (x, y, z, sigma_i / 2, sqrt(eps_i)), p_xj [n_j, 5] likewise (float32 or float64, promoted exactly
    to double).  Returns p_fi [n_i, 4] = (Fx, Fy, Fz, U) in float64: the force ON i and the sum of its pair energies."""
    xi, xj = _c(p_xi, np.float64).reshape(-1, 5), _c(p_xj, np.float64).reshape(-1, 5)
    out = np.zeros((xi.shape[0], 4), dtype=np.float64)
    rc = _load().oracle_lj_f64(xi.shape[0], _ptr(xi), xj.shape[0], _ptr(xj), _ptr(out))
    if rc != 0:
        raise ValueError(f"oracle_lj returned {rc}")
    return out


def force_batched(i_offsets: np.ndarray, j_offsets: np.ndarray, x_i: np.ndarray, x_j: np.ndarray, m_j: np.ndarray,
                  eps2: float):
    """Row f2: Eq. (1) and phi for independent sub-problems b = (i in [i_offsets[b], i_offsets[b+1]),
    j in [j_offsets[b], j_offsets[b+1])) -- literally one ``force`` call per sub-problem (PAPER.md:246, 355-359:
    the host tree code calls the force routine once per interaction list).  i-particles outside every
    sub-problem keep a = 0, phi = 0."""
    n_i = np.asarray(x_i).reshape(-1, 3).shape[0]
    acc = np.zeros((n_i, 3), dtype=np.float64)
    pot = np.zeros(n_i, dtype=np.float64)
    for b in range(len(i_offsets) - 1):
        i0, i1, j0, j1 = int(i_offsets[b]), int(i_offsets[b + 1]), int(j_offsets[b]), int(j_offsets[b + 1])
        if i1 > i0:
            acc[i0:i1], pot[i0:i1] = force(x_i[i0:i1], x_j[j0:j1], m_j[j0:j1], eps2)
    return acc, pot


def energy(x: np.ndarray, v: np.ndarray, m: np.ndarray, eps2: float) -> Tuple[float, float, float]:
    """(T, W, E) in double from an FP32 state; W = 1/2 sum m_i phi_i with coincident pairs skipped."""
    xx, vv, mm = _c(x, np.float32).reshape(-1, 3), _c(v, np.float32).reshape(-1, 3), _c(m, np.float32).reshape(-1)
    out = np.zeros(3, dtype=np.float64)
    rc = _load().oracle_energy_f32(xx.shape[0], _ptr(xx), _ptr(vv), _ptr(mm), float(eps2), _ptr(out))
    if rc != 0:
        raise ValueError(f"oracle_energy returned {rc}")
    return float(out[0]), float(out[1]), float(out[2])


def leapfrog_kdk(x: np.ndarray, v: np.ndarray, m: np.ndarray, eps2: float, dt: float, n_steps: int):
    """Textbook KDK in double.  Returns (x, v, acc, pot) at the final time (inputs are not modified)."""
    xx = np.array(x, dtype=np.float64, order="C").reshape(-1, 3)
    vv = np.array(v, dtype=np.float64, order="C").reshape(-1, 3)
    mm = _c(m, np.float64).reshape(-1)
    n = xx.shape[0]
    acc = np.zeros((n, 3), dtype=np.float64)
    pot = np.zeros(n, dtype=np.float64)
    rc = _load().oracle_leapfrog_kdk_f64(n, _ptr(xx), _ptr(vv), _ptr(mm), float(eps2), float(dt), int(n_steps),
                                         _ptr(acc), _ptr(pot))
    if rc != 0:
        raise ValueError(f"oracle_leapfrog_kdk returned {rc}")
    return xx, vv, acc, pot


def hermite4(x: np.ndarray, v: np.ndarray, m: np.ndarray, eps2: float, dt: float, n_steps: int):
    """Shared-time-step 4th-order Hermite (predict-evaluate-correct) in double.  Returns (x, v, acc, jerk, pot);
    inputs are not modified."""
    xx = np.array(x, dtype=np.float64, order="C").reshape(-1, 3)
    vv = np.array(v, dtype=np.float64, order="C").reshape(-1, 3)
    mm = _c(m, np.float64).reshape(-1)
    n = xx.shape[0]
    acc = np.zeros((n, 3)); jerk = np.zeros((n, 3)); pot = np.zeros(n)
    rc = _load().oracle_hermite4_f64(n, _ptr(xx), _ptr(vv), _ptr(mm), float(eps2), float(dt), int(n_steps),
                                     _ptr(acc), _ptr(jerk), _ptr(pot))
    if rc != 0:
        raise ValueError(f"oracle_hermite4 returned {rc}")
    return xx, vv, acc, jerk, pot


def hermite4_block_step(x: np.ndarray, v: np.ndarray, m: np.ndarray, acc: np.ndarray, jerk: np.ndarray, t: np.ndarray,
                        active: np.ndarray, t_now: float, eps2: float):
    """One block step of the individual-time-step Hermite scheme in double (reading R20): everybody is
    predicted to t_now, the particles listed in ``active`` are evaluated against all and corrected.  Returns new
    (x, v, acc, jerk, t); inputs are not modified."""
    xx = np.array(x, dtype=np.float64, order="C").reshape(-1, 3)
    vv = np.array(v, dtype=np.float64, order="C").reshape(-1, 3)
    aa = np.array(acc, dtype=np.float64, order="C").reshape(-1, 3)
    jj = np.array(jerk, dtype=np.float64, order="C").reshape(-1, 3)
    tt = np.array(t, dtype=np.float64, order="C").reshape(-1)
    mm = _c(m, np.float64).reshape(-1)
    idx = _c(np.asarray(active), np.int32).reshape(-1)
    n = xx.shape[0]
    if not (vv.shape[0] == aa.shape[0] == jj.shape[0] == tt.shape[0] == mm.shape[0] == n):
        raise ValueError("array lengths differ")
    if np.unique(idx).size != idx.size:
        raise ValueError("active indices must be distinct")
    rc = _load().oracle_hermite4_block_step_f64(n, _ptr(xx), _ptr(vv), _ptr(mm), _ptr(aa), _ptr(jj), _ptr(tt),
                                                idx.size, _ptr(idx) if idx.size else None, float(t_now), float(eps2))
    if rc != 0:
        raise ValueError(f"oracle_hermite4_block_step returned {rc}")
    return xx, vv, aa, jj, tt


def block_schedule(t: np.ndarray, dt: np.ndarray):
    """The block-step scheduler's definition (reading R20): the next block time is the earliest due time
    t_next = min_k (t[k] + dt[k]) (one FP64 addition per particle), and the due particles are those whose due time
    EQUALS it, in ascending index order.  Due times that are not finite (+-inf, NaN) take no part: they are never the
    minimum and never due.  Returns (t_next, active int32 [n_act]); n = 0 or no finite due time gives (+inf, empty).
    Pins (tests/test_oracle_hermite_pins.py, "h9"): hand-worked cases, ties, a pure-Python loop."""
    tt = np.asarray(t, dtype=np.float64).reshape(-1)
    dd = np.asarray(dt, dtype=np.float64).reshape(-1)
    if tt.shape != dd.shape:
        raise ValueError("array lengths differ")
    if tt.size == 0:
        return float("inf"), np.zeros(0, dtype=np.int32)
    with np.errstate(invalid="ignore"):
        due = tt + dd                      # inf + (-inf) = NaN: not finite, takes no part
    finite = np.isfinite(due)              # reading R20: a non-finite due time (dt = +inf parks a particle) is never selected
    if not finite.any():
        return float("inf"), np.zeros(0, dtype=np.int32)
    t_next = float(due[finite].min())
    return t_next, np.nonzero(finite & (due == t_next))[0].astype(np.int32)


def block_step_size(a0: np.ndarray, j0: np.ndarray, a1: np.ndarray, j1: np.ndarray, h: np.ndarray, eta: float) -> np.ndarray:
    """The Aarseth step-size criterion of the block Hermite scheme (textbook, reading R20; Makino &
    Aarseth 1992), from the two evaluations (a0, j0) at t and (a1, j1) at t + h of one particle:

        a2 = (-6 (a0 - a1) - h (4 j0 + 2 j1)) / h^2        a3 = (12 (a0 - a1) + 6 h (j0 + j1)) / h^3     (at t)
        a2' = a2 + h a3                                     (second derivative at t + h; a3 is constant)
        dt = sqrt( eta (|a1| |a2'| + |j1|^2) / (|j1| |a3| + |a2'|^2) )

    The result feeds an integer decision (the block level), so the definition fixes the precision and the order:
    every operation below is ONE IEEE FP32 operation (numpy float32 element-wise), in the order written; norms are
    sqrt((x x + y y) + z z).  Returns dt, float32 [n].  Pins (tests/test_oracle_hermite_pins.py, "h10"): cubic
    a(t) (the interpolant is exact), the circular orbit's sqrt(eta)/omega with its h^2 convergence."""
    f = np.float32
    a0, j0, a1, j1 = (np.ascontiguousarray(z, dtype=f).reshape(-1, 3) for z in (a0, j0, a1, j1))
    h = np.ascontiguousarray(h, dtype=f).reshape(-1, 1)
    eta = f(eta)
    old = np.seterr(over="ignore", divide="ignore", invalid="ignore")     # IEEE inf / NaN are part of the definition
    da = a0 - a1
    s1 = f(4) * j0 + f(2) * j1
    h2 = h * h
    a2 = -(f(6) * da + h * s1) / h2
    s2 = j0 + j1
    h3 = h2 * h
    a3 = (f(12) * da + (f(6) * h) * s2) / h3
    a2 = a2 + h * a3

    def sq(z):
        return (z[:, 0] * z[:, 0] + z[:, 1] * z[:, 1]) + z[:, 2] * z[:, 2]
    a1sq, j1sq, a2sq, a3sq = sq(a1), sq(j1), sq(a2), sq(a3)
    top = np.sqrt(a1sq) * np.sqrt(a2sq) + j1sq
    bot = np.sqrt(j1sq) * np.sqrt(a3sq) + a2sq
    out = np.sqrt(eta * (top / bot))
    np.seterr(**old)
    assert out.dtype == np.float32
    return out


def block_step_size_f64(a0: np.ndarray, j0: np.ndarray, a1: np.ndarray, j1: np.ndarray, h: np.ndarray, eta: float) -> np.ndarray:
    """The same Aarseth criterion as block_step_size, written out plainly in FP64 (the formula of
    include/nbody_b200.h "nb_block_step_size" / Makino & Aarseth 1992, no prescribed rounding or order):

        a2 = (-6 (a0 - a1) - h (4 j0 + 2 j1)) / h^2;  a3 = (12 (a0 - a1) + 6 h (j0 + j1)) / h^3;  a2' = a2 + h a3
        dt = sqrt( eta (|a1| |a2'| + |j1|^2) / (|j1| |a3| + |a2'|^2) )

    The FP32 definition above exists because the value feeds an integer decision; this one is the plain definition the
    CUDA path is ALSO held against, by tolerance, on well-conditioned inputs (tests/test_block_step_size_gpu.py), so
    that the kernel is not checked only against an FP32 mirror of its own arithmetic.  Returns dt, float64 [n].
    Pins (tests/test_oracle_hermite_pins.py, "h10"): cubic a(t) to 1e-13, the circular orbit, the scaling laws, and
    agreement with the FP32 definition to FP32 rounding."""
    a0, j0, a1, j1 = (np.ascontiguousarray(z, dtype=np.float64).reshape(-1, 3) for z in (a0, j0, a1, j1))
    h = np.ascontiguousarray(h, dtype=np.float64).reshape(-1, 1)
    old = np.seterr(over="ignore", divide="ignore", invalid="ignore")
    a2 = (-6.0 * (a0 - a1) - h * (4.0 * j0 + 2.0 * j1)) / h ** 2
    a3 = (12.0 * (a0 - a1) + 6.0 * h * (j0 + j1)) / h ** 3
    a2 = a2 + h * a3

    def norm(z):
        return np.sqrt(np.sum(z * z, axis=1))
    out = np.sqrt(float(eta) * (norm(a1) * norm(a2) + norm(j1) ** 2) / (norm(j1) * norm(a3) + norm(a2) ** 2))
    np.seterr(**old)
    return out


def error_metrics(acc_test: np.ndarray, acc_ref: np.ndarray, pot_test: Optional[np.ndarray] = None,
                  pot_ref: Optional[np.ndarray] = None) -> dict:
    """Eq. (3): e_i = |a_test,i - a_ref,i| / |a_ref,i|; max and RMS over i; same for phi."""
    a_t = np.asarray(acc_test, dtype=np.float64)
    a_r = np.asarray(acc_ref, dtype=np.float64)
    e = np.linalg.norm(a_t - a_r, axis=1) / np.linalg.norm(a_r, axis=1)
    out = {"acc_max": float(e.max()), "acc_rms": float(np.sqrt(np.mean(e * e)))}
    if pot_test is not None and pot_ref is not None:
        p = np.abs(np.asarray(pot_test, dtype=np.float64) - pot_ref) / np.abs(pot_ref)
        out["pot_max"] = float(p.max())
        out["pot_rms"] = float(np.sqrt(np.mean(p * p)))
    return out
