"""Run under torchrun with the gloo backend (CPU): exercises bench.py's N > 1 plumbing without a GPU."""
import json
import os
import sys

import torch
import torch.distributed as dist

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__)))))
import bench  # noqa: E402

dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
ms = 10.0 + 5.0 * rank                                  # rank r "measured" 10 + 5 r ms
ms_max = bench.max_over_ranks(ms, world, "cpu")
rate = bench.aggregate_rate(1000, world, 4, ms_max)
dist.barrier()
# one file per rank: two ranks printing to one captured stdout can interleave their lines
with open(os.path.join(os.environ["AGATE_MP_OUT"], f"rank{rank}.json"), "w") as f:
    json.dump({"rank": rank, "world": world, "ms_max": ms_max, "rate": rate}, f)
dist.destroy_process_group()
