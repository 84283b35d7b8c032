"""Worker for test_sharding_host.py: one rank of a world_size-2 gloo job on CPU that builds its shard of config 5
(37 cells) and checks, together with the other rank, that the two shards tile the slab."""
import json
import os
import sys

import numpy as np
import torch.distributed as dist

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import paper_2305_13555_b200 as P  # noqa: E402
from paper_2305_13555_b200.sharding import shard_problem  # noqa: E402
from workloads import make_problem  # noqa: E402

dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
p = make_problem(5, cells=37)
s = shard_problem(p, rank, world)
mine = {"range": list(s.cell_range), "bcs": [s.bc_left[0], s.bc_right[0]], "first_dx": float(s.sigma_t[0]), "last_dx": float(s.sigma_t[-1])}
got = [None] * world
dist.all_gather_object(got, mine)
if rank == 0:
    ranges = [g["range"] for g in got]
    edge = got[0]["last_dx"] == float(p.sigma_t[ranges[0][1] - 1]) and got[1]["first_dx"] == float(p.sigma_t[ranges[1][0]])
    print(json.dumps({"ranges": ranges, "cells_total": ranges[-1][1], "cut_bcs": [g["bcs"] for g in got], "edge_match": bool(edge),
                      "mailbox_bytes": P.shard_mailbox_bytes(p.n_angles, world)}))
dist.barrier()
dist.destroy_process_group()
