"""Worker for test_bench_multirank.py: one rank of a world_size-2 gloo job on CPU that exercises
bench.py's rank plumbing (environment parsing, MAX-time / SUM-amount aggregation)."""
import json
import os
import sys

import torch
import torch.distributed as dist

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import bench  # noqa: E402

rank, world, local = bench.dist_env()
dist.init_process_group("gloo")
assert dist.get_rank() == rank and dist.get_world_size() == world
# rank r "measured" (10 + r) ms and (r + 1) * 1000 updates
ms, upd = bench.aggregate_over_ranks(torch, 10.0 + rank, (rank + 1) * 1000.0, "cpu")
dist.barrier()
if rank == 0:
    print(json.dumps({"ms": ms, "updates": upd, "world": world, "local": local}))
dist.destroy_process_group()
