"""Worker of tests/test_bench_dist.py: run under torch.distributed.run with 2 CPU ranks (gloo)."""
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import bench  # noqa: E402

world, rank, local = bench.dist_setup(int(os.environ["WORLD_SIZE"]))
assert world == 2
bench.barrier(world)
local_ms = [100.0, 140.0][rank]
ms_total, ms_step, value = bench.aggregate_replicas(world, local_ms, steps=20)
launches = bench.sum_over_ranks(world, 85 + rank)
bench.barrier(world)
if rank == 0:
    print("RESULT " + json.dumps(dict(ms_total=ms_total, ms_step=ms_step, value=value, launches=launches)))
import torch.distributed as dist  # noqa: E402
dist.destroy_process_group()
