"""Worker for test_multirank_cpu.py: 2 ranks over gloo on 127.0.0.1 exercise bench.py's multi-rank host logic."""
import json
import os
import sys

import torch
import torch.distributed as dist

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402

rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo")
ms = bench.max_over_ranks(10.0 + 5.0 * rank, world, torch.device("cpu"))      # slowest rank wins
dist.barrier()
from paper_2606_02982_b200 import workload as wl  # noqa: E402
tier, out_len, expo = wl.make_requests(bench.rank_seed(rank), 2, 50)           # every rank its own traces
digest = int(out_len.astype("int64").sum())
all_d = [None] * world
dist.all_gather_object(all_d, digest)
if rank == 0:
    print(json.dumps({"ms": ms, "digests": all_d, "world": world}))
dist.destroy_process_group()
