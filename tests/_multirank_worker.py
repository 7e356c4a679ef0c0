"""Worker for tests/test_bench_multirank.py: two gloo ranks exercise bench.py's rank logic."""
import json
import os
import sys

import torch.distributed as dist

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import bench  # noqa: E402

dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
ms = bench.max_over_ranks(100.0 * (rank + 1), world, device="cpu")     # rank 1 is the slow one
dist.barrier()
if rank == 0:
    print(json.dumps({"world": world, "ms_max": ms, "value": bench.whole_job_value(1e6, 3, world, ms)}))
dist.destroy_process_group()
