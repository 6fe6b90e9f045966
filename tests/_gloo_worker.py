"""Worker for tests/test_bench_multirank.py: run under torch.distributed.run with the gloo backend (CPU)."""
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import torch.distributed as dist  # noqa: E402

import bench  # noqa: E402

if __name__ == "__main__":
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    # each rank reports different timings; the aggregate must use the max over ranks
    total_ms, e2e_ms = bench.reduce_max([10.0 + 5.0 * rank, 100.0 - 7.0 * rank], world)
    out = bench.replica_throughput(pairs_per_rank_step=1000.0, world=world, steps=4, total_ms=total_ms)
    if rank == 0:
        print(json.dumps({"world": world, "total_ms": total_ms, "e2e_ms": e2e_ms, "value": out}), flush=True)
    dist.barrier()
    dist.destroy_process_group()
