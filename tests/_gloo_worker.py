"""worker of test_bench_multirank.py: two CPU ranks over gloo exercise bench.py's only cross-rank step"""
import json
import os
import sys

import torch.distributed as dist

sys.path.insert(0, os.path.join(os.path.dirname(os.path.abspath(__file__)), ".."))
import bench

rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo")
ms, e2e = bench.max_over_ranks([10.0 + rank, 50.0 - rank], world)
if rank == 0:
    json.dump({"ms": ms, "e2e": e2e, "value": bench.aggregate_value(1000, 4, world, ms)}, open(sys.argv[1], "w"))
dist.barrier()
dist.destroy_process_group()
