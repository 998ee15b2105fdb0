"""Worker of tests/test_multiproc.py: one of WORLD_SIZE CPU processes (gloo) exercising bench.py's multi-rank host logic."""
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import torch.distributed as dist

import bench

rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo")
dist.barrier()
ms = bench.max_over_ranks(10.0 * (rank + 1), dist, "cpu")          # rank r "measured" 10 (r + 1) ms
value = bench.whole_job_value(bench.STEP_FLOP, 4, world, ms)
dist.barrier()
if rank == 0:
    print(json.dumps({"ms": ms, "value": value, "world": world}), flush=True)
dist.destroy_process_group()
