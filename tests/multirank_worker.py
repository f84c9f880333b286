"""Worker of test_bench_multirank.py: one rank of a world_size-2 gloo job exercising bench.py's rank logic on CPU."""
import json
import os
import sys

import torch.distributed as dist

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import bench  # noqa: E402

if __name__ == "__main__":
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    dist.barrier()
    ms = bench.max_over_ranks(10.0 * (rank + 1), world, device="cpu")      # rank r "measured" 10 (r + 1) ms
    value = bench.whole_job_value(world, cells=1000, steps=5, ms=ms)
    dist.barrier()
    if rank == 0:
        print(json.dumps({"ms": ms, "value": value, "world": world}))
    dist.destroy_process_group()
