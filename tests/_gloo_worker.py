"""Worker of tests/test_bench_host.py: world-size-2 gloo run of bench.py's N>1 host logic
(replicas only: max-over-ranks time, whole-job aggregate, rank 0 reports)."""
import json
import os
import sys

import torch
import torch.distributed as dist

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import bench  # noqa: E402


def main():
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()

    def reduce_max(x):
        t = torch.tensor([x], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    # rank r "measured" (r + 1) ms for 1e9 units
    value, t = bench.aggregate(float(rank + 1), 1e9, world, reduce_max)
    dist.barrier()
    if rank == 0:
        print(json.dumps({"value": value, "ms": t, "world": world}), flush=True)
    dist.destroy_process_group()


if __name__ == "__main__":
    main()
