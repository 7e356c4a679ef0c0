"""Worker for tests/test_sharded_cpu.py: gloo ranks run the exchange step of the j-sharded path
(paper_1207_2367_b200/sharded.py) on CPU.  The evaluation itself needs the GPU, so here each rank's
partial forces come from the oracle restricted to the rank's j-slice (masses outside the slice set
to zero contribute exactly nothing); the all-reduce must reproduce the oracle's full evaluation."""
import json
import os
import sys

import numpy as np
import torch
import torch.distributed as dist

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import oracle.nb_oracle as orc  # noqa: E402
from paper_1207_2367_b200.sharded import j_range  # noqa: E402
from workloads import mean_field_acc, plummer  # noqa: E402

dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
N = int(sys.argv[1])
pos, vel, m = plummer(N, seed=17)
accp = mean_field_acc(pos)
jb, je = j_range(N, rank, world)
ms = np.zeros_like(m)
ms[jb:je] = m[jb:je]
idx = np.arange(0, N, 7, dtype=np.int32)                       # the "active set"
part = np.stack(orc.force(pos, vel, accp, ms, 1e-3, idx))      # [3][n][3] partial acc, jerk, snap
buf = torch.from_numpy(np.ascontiguousarray(part.transpose(0, 2, 1)).reshape(-1).copy())  # [9][n]
dist.all_reduce(buf, op=dist.ReduceOp.SUM)
ranges = [None] * world
dist.all_gather_object(ranges, (jb, je))
full = np.stack(orc.force(pos, vel, accp, m, 1e-3, idx)).transpose(0, 2, 1).reshape(-1)
err = float(np.abs(buf.numpy() - full).max() / np.abs(full).max())
if rank == 0:
    print(json.dumps({"world": world, "ranges": ranges, "err": err, "n": int(idx.size)}))
dist.destroy_process_group()
