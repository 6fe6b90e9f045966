"""Seeded synthetic inputs for the five BASELINE.json configs (C0..C4).

This module only *draws particles*.  It holds none of the method's arithmetic (no pair
force, no potential, no integrator) and is the one module that both the CUDA path's tests /
bench and the CPU oracle's tests read, so that both sides see bit-identical FP32 arrays.

Why synthetic: the paper measured on equal-mass Plummer spheres built with the NEMO toolbox's
``mkplummer`` (section 3.3; Tables 2-3).  NEMO is a third-party
package that is not in this image; the generators below stand in for it, taking the workload's
*shape* (equal-mass Plummer sphere, N = 2048 ... 131072) and BASELINE.json's parameters.
The recipe is stated in DESIGN.md section "Input recipe".

All sampling is done in float64 with ``numpy.random.Generator(PCG64(seed))``, whole arrays in
the order stated below, then cast once to float32.  Units: G = 1, total mass 1, Plummer scale
a = 1.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional

import numpy as np

# Mass fraction of the a = 1 Plummer model inside r = 10a: M(r) = r^3 (1 + r^2)^(-3/2).
PLUMMER_MT_10A = 1000.0 / 101.0 ** 1.5


def _rng(seed: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(seed))


def _isotropic(radius: np.ndarray, u_z: np.ndarray, u_phi: np.ndarray) -> np.ndarray:
    """Vectors of length ``radius`` with isotropic directions from two uniform arrays."""
    z = (1.0 - 2.0 * u_z) * radius
    rho = np.sqrt(np.maximum(radius * radius - z * z, 0.0))
    phi = 2.0 * np.pi * u_phi
    return np.stack([rho * np.cos(phi), rho * np.sin(phi), z], axis=1)


def plummer_positions(n: int, rng: np.random.Generator, r_max_mass_fraction: float = PLUMMER_MT_10A):
    """Plummer sphere (a = 1) positions by inverse-CDF radius, truncated at 10a.

    Draw order: X1, X2, X3 ~ U(0,1), three arrays of length n.  X = X1 * M_T restricts the
    enclosed-mass fraction to r <= 10a; r = (X^(-2/3) - 1)^(-1/2).
    Returns (positions float64 [n,3], radii float64 [n]).
    """
    x1 = rng.random(n)
    x2 = rng.random(n)
    x3 = rng.random(n)
    frac = np.maximum(x1 * r_max_mass_fraction, 1e-300)
    r = 1.0 / np.sqrt(frac ** (-2.0 / 3.0) - 1.0)
    return _isotropic(r, x2, x3), r


def plummer_velocities(r: np.ndarray, rng: np.random.Generator) -> np.ndarray:
    """Aarseth-Henon-Wielen rejection sampling of isotropic Plummer velocities (a = 1, G = M = 1).

    For each particle draw (X4, X5) until 0.1*X5 < X4^2 (1 - X4^2)^(7/2); speed
    V = X4 * sqrt(2) * (1 + r^2)^(-1/4).  Vectorised: each round redraws only the rejected
    entries (round k draws its X4 array, then its X5 array), then two direction arrays.
    """
    n = r.shape[0]
    q = np.zeros(n)
    todo = np.arange(n)
    while todo.size:
        x4 = rng.random(todo.size)
        x5 = rng.random(todo.size)
        ok = 0.1 * x5 < x4 * x4 * (1.0 - x4 * x4) ** 3.5
        q[todo[ok]] = x4[ok]
        todo = todo[~ok]
    speed = q * np.sqrt(2.0) * (1.0 + r * r) ** -0.25
    u_z = rng.random(n)
    u_phi = rng.random(n)
    return _isotropic(speed, u_z, u_phi)


def uniform_sphere_positions(n: int, rng: np.random.Generator, radius: float = 1.0) -> np.ndarray:
    """Uniform-density ball: r = R * X1^(1/3), isotropic direction from X2, X3."""
    x1 = rng.random(n)
    x2 = rng.random(n)
    x3 = rng.random(n)
    return _isotropic(radius * np.cbrt(x1), x2, x3)


def lognormal_masses(n: int, rng: np.random.Generator) -> np.ndarray:
    """exp(N(0,1)) normalised (in float64) to total mass 1."""
    g = rng.standard_normal(n)
    m = np.exp(g)
    return m / m.sum()


@dataclass
class Workload:
    """One force call's (or one integration's) inputs, FP32, C-contiguous."""
    name: str
    x_j: np.ndarray                 # float32 [n_j, 3]
    m_j: np.ndarray                 # float32 [n_j]
    eps2: float                     # epsilon^2, exactly representable in FP32
    x_i: Optional[np.ndarray] = None  # float32 [n_i, 3]; None => i-set is the j-set (aliased)
    v: Optional[np.ndarray] = None    # float32 [n, 3] (C4 only)
    dt: Optional[float] = None
    n_steps: Optional[int] = None
    i_index: Optional[np.ndarray] = None  # int64 [n_i] indices into the j-set (C2 only)
    seed: int = 0
    meta: dict = field(default_factory=dict)

    @property
    def n_j(self) -> int:
        return int(self.x_j.shape[0])

    @property
    def n_i(self) -> int:
        return int(self.x_j.shape[0] if self.x_i is None else self.x_i.shape[0])

    @property
    def xi(self) -> np.ndarray:
        return self.x_j if self.x_i is None else self.x_i

    @property
    def pairs(self) -> int:
        return self.n_i * self.n_j


def _f32(a: np.ndarray) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float32)


def plummer_workload(n: int, eps: float, seed: int, name: str = "plummer", with_velocities: bool = False,
                     dt: Optional[float] = None, n_steps: Optional[int] = None) -> Workload:
    rng = _rng(seed)
    pos, r = plummer_positions(n, rng)
    m = np.full(n, 1.0 / n)
    v = plummer_velocities(r, rng) if with_velocities else None
    return Workload(name=name, x_j=_f32(pos), m_j=_f32(m), eps2=float(np.float32(eps * eps)),
                    v=None if v is None else _f32(v), dt=dt, n_steps=n_steps, seed=seed,
                    meta={"model": "plummer a=1 truncated at 10a", "eps": eps})


def subset_workload(n_j: int, n_i: int, eps: float, seed: int, name: str = "subset") -> Workload:
    """Active-subset call: positions first, then n_i indices without replacement (C2 recipe)."""
    rng = _rng(seed)
    pos, _ = plummer_positions(n_j, rng)
    idx = rng.choice(n_j, n_i, replace=False)
    x_j = _f32(pos)
    return Workload(name=name, x_j=x_j, m_j=_f32(np.full(n_j, 1.0 / n_j)), eps2=float(np.float32(eps * eps)),
                    x_i=np.ascontiguousarray(x_j[idx]), i_index=idx.astype(np.int64), seed=seed,
                    meta={"model": "plummer a=1 truncated at 10a; i = random subset of j", "eps": eps})


def uniform_sphere_workload(n: int, eps: float, seed: int, name: str = "uniform") -> Workload:
    rng = _rng(seed)
    pos = uniform_sphere_positions(n, rng)
    m = lognormal_masses(n, rng)
    return Workload(name=name, x_j=_f32(pos), m_j=_f32(m), eps2=float(np.float32(eps * eps)), seed=seed,
                    meta={"model": "uniform sphere R=1, log-normal masses", "eps": eps})


CONFIG_NAMES = ("C0", "C1", "C2", "C3", "C4")


def config(k: int, scale: float = 1.0) -> Workload:
    """BASELINE.json configs[k].  ``scale`` < 1 shrinks N (tests only; the bench uses scale = 1)."""
    def s(n: int) -> int:
        return max(8, int(round(n * scale)))
    if k == 0:
        return plummer_workload(s(2048), 1.0 / 64, seed=0, name="C0")
    if k == 1:
        return plummer_workload(s(131072), 1.0 / 256, seed=1, name="C1")
    if k == 2:
        return subset_workload(s(65536), min(512, s(65536)), 1.0 / 128, seed=2, name="C2")
    if k == 3:
        return uniform_sphere_workload(s(1048576), 1.0 / 1024, seed=3, name="C3")
    if k == 4:
        return plummer_workload(s(65536), 1.0 / 128, seed=4, name="C4", with_velocities=True,
                                dt=1.0 / 512, n_steps=1000)
    raise ValueError(f"no config {k}")


# ---------------------------------------------------------------------------------------------
# Row f2: interaction lists of a host tree code (section
# 4.4: "the force calculation on several thousands particles", Barnes' modified tree algorithm).
# The paper gives no tree and no list statistics beyond "several thousands"; the recipe below only
# reproduces the SHAPE of such a call sequence -- many groups of a few tens to a few hundred
# i-particles, each with its own list of a few thousand j-particles (its own members, near
# neighbours taken directly, and heavier pseudo-particles standing for far cells).
@dataclass
class BatchedWorkload:
    name: str
    i_offsets: np.ndarray           # int32 [n_batch + 1]
    j_offsets: np.ndarray           # int32 [n_batch + 1]
    x_i: np.ndarray                 # float32 [n_i_total, 3]
    x_j: np.ndarray                 # float32 [n_j_total, 3]
    m_j: np.ndarray                 # float32 [n_j_total]
    eps2: float
    seed: int = 0
    meta: dict = field(default_factory=dict)

    @property
    def n_batch(self) -> int:
        return int(self.i_offsets.shape[0] - 1)

    @property
    def pairs(self) -> int:
        ni = np.diff(self.i_offsets).astype(np.int64)
        nj = np.diff(self.j_offsets).astype(np.int64)
        return int((ni * nj).sum())


def tree_list_workload(n_particles: int, group_min: int, group_max: int, list_min: int, list_max: int, eps: float,
                       seed: int, name: str = "tree-lists", max_groups: Optional[int] = None) -> BatchedWorkload:
    """Groups = runs of consecutive particles of a Plummer sphere sorted along a 3-D grid order.

    Draw order: Plummer positions (X1, X2, X3); group sizes (uniform integers, cut to cover the
    sorted particles); then per group: list length (uniform integer), the indices of the direct
    neighbours (``rng.choice`` over all particles, without replacement), the cell positions
    (a fresh Plummer draw) and the cell occupation numbers (uniform integers 2..64; a cell's mass
    is that many particle masses).  One third of a list (rounded down) are cells.
    """
    rng = _rng(seed)
    pos, _ = plummer_positions(n_particles, rng)
    cell = np.floor((pos + 10.0) * (64.0 / 20.0)).astype(np.int64).clip(0, 63)
    order = np.lexsort((cell[:, 2], cell[:, 1], cell[:, 0]))
    pos = pos[order]
    m = 1.0 / n_particles
    sizes = []
    left = n_particles
    while left > 0 and (max_groups is None or len(sizes) < max_groups):
        g = int(min(left, rng.integers(group_min, group_max + 1)))
        sizes.append(g)
        left -= g
    i_off = np.concatenate([[0], np.cumsum(sizes)])
    xi_parts, xj_parts, mj_parts, lens = [], [], [], []
    for b, g in enumerate(sizes):
        own = np.arange(i_off[b], i_off[b + 1])
        n_list = int(rng.integers(list_min, list_max + 1))
        n_cells = n_list // 3
        n_near = max(0, n_list - n_cells - g)
        near = rng.choice(n_particles, n_near, replace=False)
        cells, _ = plummer_positions(n_cells, rng)
        occ = rng.integers(2, 65, n_cells)
        xi_parts.append(pos[own])
        xj_parts.append(np.concatenate([pos[own], pos[near], cells]))
        mj_parts.append(np.concatenate([np.full(g + n_near, m), occ * m]))
        lens.append(g + n_near + n_cells)
    j_off = np.concatenate([[0], np.cumsum(lens)])
    return BatchedWorkload(name=name, i_offsets=i_off.astype(np.int32), j_offsets=j_off.astype(np.int32),
                           x_i=_f32(np.concatenate(xi_parts)), x_j=_f32(np.concatenate(xj_parts)),
                           m_j=_f32(np.concatenate(mj_parts)), eps2=float(np.float32(eps * eps)), seed=seed,
                           meta={"model": "plummer a=1 truncated at 10a, grid-sorted groups with own + near + cell lists",
                                 "eps": eps, "groups": len(sizes)})


def lj_fluid_rows(n: int, density: float, jitter: float, seed: int) -> np.ndarray:
    """Row f3 (Lennard-Jones pipeline): n particles on a jittered simple-cubic lattice of number density ``density``
    (reduced units, sigma ~ 1) -- a dense fluid without overlaps -- with per-particle sigma in [0.9, 1.1] and eps in
    [0.5, 1.5].  Returns float32 rows [n, 5] = (x, y, z, sigma / 2, sqrt(eps)), the record format of
    nb_cunbody_lennard_jones.  ``jitter`` is the maximum displacement in units of the lattice spacing."""
    rng = _rng(seed)
    side = int(np.ceil(n ** (1.0 / 3.0)))
    a = density ** (-1.0 / 3.0)
    g = np.stack(np.meshgrid(*[np.arange(side, dtype=np.float64)] * 3, indexing="ij"), -1).reshape(-1, 3)
    pick = rng.permutation(g.shape[0])[:n]
    x = (g[pick] + rng.uniform(-jitter, jitter, (n, 3))) * a
    sigma = rng.uniform(0.9, 1.1, n)
    eps = rng.uniform(0.5, 1.5, n)
    return _f32(np.concatenate([x, 0.5 * sigma[:, None], np.sqrt(eps)[:, None]], axis=1))


def block_levels(n: int, seed: int, n_levels: int = 3) -> np.ndarray:
    """Seeded block-time-step levels for the active-subset integration (row f4): particle k steps with dt * 2**level[k].
    Half of the particles sit on the finest level, the rest are spread evenly over the coarser ones (block-step runs
    of a Plummer sphere keep most particles on few levels).  Holds no arithmetic of the method: who is due at
    sub-step s is ``s % 2**level == 0``, evaluated by the caller."""
    rng = _rng(seed)
    p = np.full(n_levels, 0.5 / max(n_levels - 1, 1))
    p[0] = 0.5 if n_levels > 1 else 1.0
    return rng.choice(n_levels, size=n, p=p).astype(np.int32)
