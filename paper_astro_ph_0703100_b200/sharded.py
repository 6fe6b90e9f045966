"""Row f4: multi-GPU i-sharding of the force evaluation and of the leapfrog.

The i-particles are independent (Eq. (1): every a_i is its own sum over j), so G ranks each own
a contiguous slice of the particles, and the only exchange step of the path is re-creating the j-set:

    1. every rank packs its slice into 16-byte (x, y, z, m) records          [local, O(n/G), nb_pack_j]
    2. ONE all-gather of those records (NCCL over NVLink 5 / NVSwitch)       [16 B x n per force call]
    3. every rank evaluates its own i-slice against all n records            [local, O(n^2/G), nb_force_packed]

No reduction is needed (a j-partition would need a reduce-scatter of 16 B x n_i and buys nothing).  Slices are
ceil(n/G) long; the last ranks' slices are padded with zero-mass records, which add nothing to a or phi.  In a time
integration every rank owns its slice of (x, v): `sharded_leapfrog_kdk` runs nb_kick_drift / nb_kick on the slice and
one all-gather of the updated records per step.

This module is plumbing only: ``torch.distributed`` moves the records, the library's kernels do every step of the
arithmetic.  The kernels are passed in as a ``Kernels`` bundle so that the host logic (slicing, padding, gather order,
step sequence) can be tested with gloo on CPU ranks, where the tests inject CPU stand-ins; the default bundle is the
CUDA library (``binding``) and there is no fallback.

The exchange: with the NCCL backend the records are gathered device to device; with the gloo backend and CUDA tensors
(the only way to run two ranks on ONE GPU, as the GPU tests do: NCCL refuses two ranks on the same device) the packed
slice is staged through host memory.  The kernels are the same in both cases.
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Callable, Optional, Tuple


@dataclass
class Kernels:
    """The library calls the sharded drivers make (same signatures as ``binding``)."""
    pack_j: Callable            # (x [k,3], m [k], xm_out [>=k,4]) -> xm_out
    force_packed: Callable      # (x_i [k,3], xm_j [n,4], eps2, acc_out=None, pot_out=None, want_pot=True) -> (acc, pot)
    kick_drift: Callable        # (x, v, acc, h, n_kicks, dt) in place
    kick: Callable              # (v, acc, h) in place


def library_kernels() -> Kernels:
    from . import binding
    return Kernels(binding.pack_j, binding.force_packed, binding.kick_drift, binding.kick)


def shard_range(n: int, rank: int, world: int) -> Tuple[int, int]:
    """Contiguous slice [lo, hi) of n particles owned by ``rank``: ceil(n/world) each, the tail ranks get less."""
    per = -(-n // world)
    lo = min(n, rank * per)
    return lo, min(n, lo + per)


def gather_packed(x_local, m_local, n_total: int, group=None, kernels: Optional[Kernels] = None):
    """All-gathers the packed (x, y, z, m) records of every rank's slice.  Returns a [world * ceil(n/world), 4]
    tensor on the local device whose first n_total rows are the particles in global order; the padding rows of
    ragged tail slices have m = 0 and sit at the END of their rank's block, so the records of rank r start at
    r * ceil(n/world)."""
    import torch
    import torch.distributed as dist
    kernels = kernels or library_kernels()
    world = dist.get_world_size(group) if dist.is_initialized() else 1
    per = -(-n_total // world)
    local = torch.zeros((per, 4), dtype=x_local.dtype, device=x_local.device)   # float32 records on the device
    if x_local.shape[0] > 0:
        kernels.pack_j(x_local.contiguous(), m_local.contiguous(), local)      # row a1: the library's kernel
    if world == 1:
        return local
    if x_local.is_cuda and dist.get_backend(group) != "nccl":
        # two ranks on one device (tests), or no NCCL: stage the 16 B x n/G records through host memory
        host = torch.empty((world * per, 4), dtype=x_local.dtype)
        dist.all_gather_into_tensor(host, local.cpu(), group=group)
        return host.to(x_local.device)
    out = torch.empty((world * per, 4), dtype=x_local.dtype, device=x_local.device)
    dist.all_gather_into_tensor(out, local, group=group)
    return out


def sharded_force(x_local, m_local, n_total: int, eps2: float, group=None, want_pot: bool = True,
                  kernels: Optional[Kernels] = None):
    """Acceleration and potential of this rank's slice against ALL particles of all ranks.

    x_local [k, 3], m_local [k]: this rank's slice (k = shard_range(n_total, rank, world) length).
    Returns (acc [k, 3], pot [k] or None) for the local slice.  One collective: the all-gather of 16 B x n_total.
    """
    kernels = kernels or library_kernels()
    xm_all = gather_packed(x_local, m_local, n_total, group, kernels)
    return kernels.force_packed(x_local.contiguous(), xm_all, eps2, want_pot=want_pot)


def sharded_leapfrog_kdk(x_local, v_local, m_local, n_total: int, eps2: float, dt: float, n_steps: int, group=None,
                         kernels: Optional[Kernels] = None):
    """n_steps kick-drift-kick steps with the particles i-sharded over the ranks (nb_leapfrog_kdk's sequence, per slice):

        a = force(slice | all)                                  one all-gather
        repeat n_steps times:  v += a dt/2;  x += v dt;  a = force(slice | all);  v += a dt/2      one all-gather per step

    x_local, v_local [k, 3] are updated in place; returns (acc [k, 3], pot [k]) at the final time.  The closing half-kick
    of a step is fused with the opening half-kick of the next (two separately rounded FMAs), as in nb_leapfrog_kdk; phi is
    evaluated at the final time only.
    """
    kernels = kernels or library_kernels()
    h = 0.5 * dt
    acc, pot = sharded_force(x_local, m_local, n_total, eps2, group, want_pot=(n_steps == 0), kernels=kernels)
    for s in range(n_steps):
        kernels.kick_drift(x_local, v_local, acc, h, 1 if s == 0 else 2, dt)
        acc, pot = sharded_force(x_local, m_local, n_total, eps2, group, want_pot=(s + 1 == n_steps), kernels=kernels)
    if n_steps > 0:
        kernels.kick(v_local, acc, h)
    return acc, pot
