"""Run under torchrun with the gloo backend (CPU): the halo-exchange schedule of paper_2503_20899_b200/slab.py.
Every rank owns a range of "planes" whose value is their global index; after one exchange its receive buffers must
hold the two planes below and above its range (wrapped if periodic), and the v_max all-reduce must give the maximum."""
import json
import os
import sys

import torch
import torch.distributed as dist

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__)))))
from paper_2503_20899_b200 import slab  # noqa: E402  (imports no CUDA code until an Agate context is made)

dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
out = {"rank": rank, "world": world, "cases": []}
for n, periodic in ((11, True), (11, False), (4 * world, True)):
    parts = slab.split(n, world)
    s0, cnt = parts[rank]
    width = 3                                             # elements per plane
    mine = torch.arange(s0, s0 + cnt, dtype=torch.float64).repeat_interleave(width).reshape(cnt, width)
    send_lo, send_hi = mine[:2].clone(), mine[-2:].clone()
    recv_lo = torch.full((2, width), -1.0, dtype=torch.float64)
    recv_hi = torch.full((2, width), -1.0, dtype=torch.float64)
    slab.exchange(send_lo, send_hi, recv_lo, recv_hi, rank, world, periodic)
    lo, hi = slab.neighbours(rank, world, periodic)
    want_lo = [(s0 - 2) % n, (s0 - 1) % n] if lo is not None else [-1, -1]
    want_hi = [(s0 + cnt) % n, (s0 + cnt + 1) % n] if hi is not None else [-1, -1]
    ok = (recv_lo[:, 0].tolist() == [float(v) for v in want_lo] and recv_hi[:, 0].tolist() == [float(v) for v in want_hi]
          and bool((recv_lo == recv_lo[:, :1]).all()) and bool((recv_hi == recv_hi[:, :1]).all()))
    out["cases"].append({"n": n, "periodic": periodic, "ok": ok, "recv_lo": recv_lo[:, 0].tolist(),
                         "recv_hi": recv_hi[:, 0].tolist(), "parts": parts})
v = torch.tensor([1.0 + 0.25 * rank], dtype=torch.float64)
dist.all_reduce(v, op=dist.ReduceOp.MAX)
out["vmax"] = float(v.item())
dist.barrier()
with open(os.path.join(os.environ["AGATE_MP_OUT"], f"slab_rank{rank}.json"), "w") as f:
    json.dump(out, f)
dist.destroy_process_group()
