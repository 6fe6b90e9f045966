"""Worker for tests/test_sharded.py: the i-sharded force and leapfrog (row f4) at world size > 1 over gloo.

    _gloo_shard_worker.py <force|leapfrog> <cpu|cuda> <n> [n_steps]

cpu : the host logic (slices, padding, gather order, step sequence) with CPU stand-ins injected for the library's kernels
      (pack, force = the oracle, kick / drift in float64) -- the product's default kernels are the CUDA library.
cuda: every rank on cuda:0 (the metered box has one GPU and NCCL refuses two ranks on one device): the library's own
      kernels (nb_pack_j, nb_force_packed, nb_kick_drift, nb_kick) on each rank's slice, the packed records exchanged
      through host memory over gloo.  Ranks never wait on one another's kernels, only on the host-side collective.
"""
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


def cpu_kernels():
    def pack_j(x, m, xm_out):
        k = x.shape[0]
        xm_out[:k, :3] = x
        xm_out[:k, 3] = m
        return xm_out

    def force_packed(x_i, xm_j, eps2, acc_out=None, pot_out=None, want_pot=True):
        xm = xm_j.numpy()
        acc, pot = oracle.force(x_i.numpy().astype(np.float64), np.ascontiguousarray(xm[:, :3], dtype=np.float64), np.ascontiguousarray(xm[:, 3], dtype=np.float64), eps2)
        return torch.from_numpy(acc), (torch.from_numpy(pot) if want_pot else None)

    def kick_drift(x, v, acc, h, n_kicks, dt):
        for _ in range(n_kicks):
            v += acc * h
        x += v * dt

    def kick(v, acc, h):
        v += acc * h

    return sharded.Kernels(pack_j, force_packed, kick_drift, kick)


if __name__ == "__main__":
    mode, where, n = sys.argv[1], sys.argv[2], int(sys.argv[3])
    n_steps = int(sys.argv[4]) if len(sys.argv) > 4 else 0
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    w = wl.plummer_workload(n, 1.0 / 64, seed=13, with_velocities=True)   # every rank draws the same seeded particles
    lo, hi = sharded.shard_range(n, rank, world)
    if where == "cuda":
        assert torch.cuda.is_available(), "the cuda mode needs a device (no CPU fallback exists)"
        torch.cuda.set_device(0)
        dev, dtype, kernels = "cuda", torch.float32, None
        import paper_astro_ph_0703100_b200 as nb
        nb.lib()
    else:
        dev, dtype, kernels = "cpu", torch.float64, cpu_kernels()
    x = torch.from_numpy(w.x_j[lo:hi].copy()).to(dev, dtype)
    v = torch.from_numpy(w.v[lo:hi].copy()).to(dev, dtype)
    m = torch.from_numpy(w.m_j[lo:hi].copy()).to(dev, dtype)
    dt = 1.0 / 256
    if mode == "force":
        acc, pot = sharded.sharded_force(x, m, n, w.eps2, kernels=kernels)
    else:
        acc, pot = sharded.sharded_leapfrog_kdk(x, v, m, n, w.eps2, dt, n_steps, kernels=kernels)
    if where == "cuda":
        torch.cuda.synchronize()
    # collect the slices on every rank (gloo, host) and compare on rank 0 with the unsharded oracle
    per = -(-n // world)
    buf = torch.zeros((per, 10), dtype=torch.float64)
    k = hi - lo
    buf[:k, 0:3], buf[:k, 3:6], buf[:k, 6:9], buf[:k, 9] = x.cpu().double(), v.cpu().double(), acc.cpu().double(), pot.cpu().double()
    out = [torch.zeros_like(buf) for _ in range(world)]
    dist.all_gather(out, buf)
    if rank == 0:
        full = np.concatenate([o.numpy()[: sharded.shard_range(n, r, world)[1] - sharded.shard_range(n, r, world)[0]]
                               for r, o in enumerate(out)])
        res = {"world": world, "n": n, "mode": mode, "where": where,
               "slices": [sharded.shard_range(n, r, world) for r in range(world)]}
        if mode == "force":
            ref_acc, ref_pot = oracle.force(w.x_j, w.x_j, w.m_j, w.eps2)
            e = oracle.error_metrics(full[:, 6:9], ref_acc, full[:, 9], ref_pot)
            res.update(acc_max_abs_diff=float(np.abs(full[:, 6:9] - ref_acc).max()),
                       pot_max_abs_diff=float(np.abs(full[:, 9] - ref_pot).max()), **e)
        else:
            xr, vr, ar, pr = oracle.leapfrog_kdk(w.x_j, w.v, w.m_j, w.eps2, dt, n_steps)
            res.update(x_max_abs_diff=float(np.abs(full[:, 0:3] - xr).max()), v_max_abs_diff=float(np.abs(full[:, 3:6] - vr).max()),
                       acc_rel=float(np.abs(full[:, 6:9] - ar).max() / np.abs(ar).max()),
                       pot_rel=float(np.abs(full[:, 9] - pr).max() / np.abs(pr).max()))
        print(json.dumps(res), flush=True)
    dist.barrier()
    dist.destroy_process_group()
