"""Worker of tests/test_bench_multirank.py: one of WORLD_SIZE gloo ranks on the CPU."""
import json
import os
import sys

import torch
import torch.distributed as dist

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import bench  # noqa: E402

rank = int(os.environ["RANK"]); world = int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo")
ms = bench.max_over_ranks(10.0 + 5.0 * rank, torch.device("cpu"), world)   # slowest rank wins
dist.barrier()
if rank == 0:
    print(json.dumps({"ms": ms, "value": bench.whole_job_gdof_per_s(1000, 2, world, ms * 1e-3)}))
dist.destroy_process_group()
