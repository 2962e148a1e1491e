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
# every rank builds its own shard of the headline workload exactly as bench.run_ours does (configs[3] traces, seed per rank;
# no text sample here, so no characterizer is needed): weak scaling, no data-path exchange
c = bench.build_cfg3(2, 0, bench.rank_seed(rank), None)
assert c.n_inst == 2 * 20 and c.server.max_batch == 128 and c.server.kv_budget == 65536
digest = int(c.out_len.astype("int64").sum()) * 1_000_003 + int(c.arrival[-1])
all_d = [None] * world
dist.all_gather_object(all_d, digest)
if rank == 0:
    print(json.dumps({"ms": ms, "digests": all_d, "world": world}))
dist.destroy_process_group()
