"""Worker for tests/test_sharded.py: the host logic of the i-sharded force (row f4) over gloo on CPU ranks.
The arithmetic is injected (force_fn = the CPU oracle) -- the product's default force_fn is the CUDA library."""
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402
import torch  # noqa: E402
import torch.distributed as dist  # noqa: E402

import oracle  # noqa: E402
from paper_astro_ph_0703100_b200 import sharded, workloads as wl  # noqa: E402


def oracle_force_packed(x_i, xm_j, eps2, want_pot=True):
    xm = xm_j.numpy()
    acc, pot = oracle.force(x_i.numpy(), np.ascontiguousarray(xm[:, :3]), np.ascontiguousarray(xm[:, 3]), eps2)
    return torch.from_numpy(acc), torch.from_numpy(pot)


if __name__ == "__main__":
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    n = int(sys.argv[1])
    w = wl.plummer_workload(n, 1.0 / 64, seed=13)                     # every rank draws the same seeded particles
    lo, hi = sharded.shard_range(n, rank, world)
    x_local, m_local = torch.from_numpy(w.x_j[lo:hi].copy()), torch.from_numpy(w.m_j[lo:hi].copy())
    acc, pot = sharded.sharded_force(x_local, m_local, n, w.eps2, force_fn=oracle_force_packed)
    # collect the slices on rank 0 and compare with the unsharded oracle
    per = -(-n // world)
    buf = torch.zeros((per, 4), dtype=torch.float64)
    buf[: hi - lo, :3] = acc
    buf[: hi - lo, 3] = pot
    out = [torch.zeros_like(buf) for _ in range(world)]
    dist.all_gather(out, buf)
    if rank == 0:
        full = torch.cat(out)[:n].numpy() if n % per == 0 or world == 1 else \
            np.concatenate([o.numpy()[: sharded.shard_range(n, r, world)[1] - sharded.shard_range(n, r, world)[0]]
                            for r, o in enumerate(out)])
        ref_acc, ref_pot = oracle.force(w.x_j, w.x_j, w.m_j, w.eps2)
        print(json.dumps({"world": world, "n": n, "slices": [sharded.shard_range(n, r, world) for r in range(world)],
                          "acc_max_abs_diff": float(np.abs(full[:, :3] - ref_acc).max()),
                          "pot_max_abs_diff": float(np.abs(full[:, 3] - ref_pot).max())}), flush=True)
    dist.barrier()
    dist.destroy_process_group()
