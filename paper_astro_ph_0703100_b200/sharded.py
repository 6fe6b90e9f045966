"""Row f4: multi-GPU i-sharding of the force evaluation.

The i-particles are independent (Eq. (1): every a_i is its own sum over j), so G ranks each own
a contiguous slice of the particles, and the only exchange step of the path is re-creating the j-set:

    1. every rank packs its slice into 16-byte (x, y, z, m) records          [local, O(n/G)]
    2. ONE all-gather of those records over NCCL (NVLink 5 / NVSwitch)       [16 B x n per force call]
    3. every rank evaluates its own i-slice against all n records with nb_force_packed   [local, O(n^2/G)]

No reduction is needed (a j-partition would need a reduce-scatter of 16 B x n_i and buys nothing).  Slices are
ceil(n/G) long; the last ranks' slices are padded with zero-mass records, which add nothing to a or phi.

This module is plumbing only: ``torch.distributed`` moves the records, the library's kernels do every step of the
arithmetic.  ``force_fn`` exists so that the host logic (slicing, padding, gather order) can be tested with gloo on
CPU ranks; on a GPU rank the default is ``binding.force_packed`` and there is no fallback.
"""
from __future__ import annotations

from typing import Callable, Optional, Tuple


def shard_range(n: int, rank: int, world: int) -> Tuple[int, int]:
    """Contiguous slice [lo, hi) of n particles owned by ``rank``: ceil(n/world) each, the tail ranks get less."""
    per = -(-n // world)
    lo = min(n, rank * per)
    return lo, min(n, lo + per)


def gather_packed(x_local, m_local, n_total: int, group=None):
    """All-gathers the packed (x, y, z, m) records of every rank's slice.  Returns a [world * ceil(n/world), 4]
    tensor on the local device whose first n_total rows are the particles in global order; the padding rows of
    ragged tail slices have m = 0 and sit at the END of their rank's block, so the records of rank r start at
    r * ceil(n/world)."""
    import torch
    import torch.distributed as dist
    world = dist.get_world_size(group) if dist.is_initialized() else 1
    per = -(-n_total // world)
    local = torch.zeros((per, 4), dtype=torch.float32, device=x_local.device)
    k = x_local.shape[0]
    if x_local.is_cuda:
        from . import binding
        binding.pack_j(x_local.contiguous(), m_local.contiguous(), local)     # row a1, the library's kernel
    else:                                                                      # CPU ranks: gloo tests of the host logic only
        local[:k, :3] = x_local
        local[:k, 3] = m_local
    if world == 1:
        return local
    out = torch.empty((world * per, 4), dtype=torch.float32, device=x_local.device)
    dist.all_gather_into_tensor(out, local, group=group)
    return out


def sharded_force(x_local, m_local, n_total: int, eps2: float, group=None, want_pot: bool = True,
                  force_fn: Optional[Callable] = None):
    """Acceleration and potential of this rank's slice against ALL particles of all ranks.

    x_local [k, 3], m_local [k]: this rank's slice (k = shard_range(n_total, rank, world) length).
    Returns (acc [k, 3], pot [k] or None) for the local slice.  One collective: the all-gather of 16 B x n_total.
    """
    xm_all = gather_packed(x_local, m_local, n_total, group)
    if force_fn is None:
        from . import binding
        force_fn = binding.force_packed
    return force_fn(x_local.contiguous(), xm_all, eps2, want_pot=want_pot)
