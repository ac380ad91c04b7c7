"""Slab decomposition plumbing (NEXT-4; include/agate.h "slab decomposition").

Argument marshalling and message passing only: every kernel of the path runs inside libagate.so.  A rank owns the
planes [start, start + count) of the grid's last active dimension, holds an ordinary `Agate` context over them with
its cut faces marked (`agate_set_slab`), and per Runge-Kutta stage exchanges the two ghost layers of each cut face
with its neighbours between `agate_stage_pre` and `agate_stage_post`.  Per step one all-reduce(max) of one double
gives the common v_max, hence dt (A7).  Messages travel through `torch.distributed` (NCCL over NVLink on GPUs; the
CPU tests of the schedule use gloo), or as plain device copies when one process holds both sides of a face.
"""
from __future__ import annotations


def split(n: int, world: int):
    """Contiguous, near-equal plane ranges: [(start, count)] per rank; every rank gets at least the two layers its
    neighbours need as ghosts."""
    if world < 1 or n < 2 * world:
        raise ValueError(f"cannot cut {n} planes into {world} slabs of at least 2")
    base, extra = divmod(n, world)
    out, s = [], 0
    for r in range(world):
        c = base + (1 if r < extra else 0)
        out.append((s, c))
        s += c
    return out


def neighbours(rank: int, world: int, periodic: bool):
    """(lower, upper) rank across the low / high cut face, None where the slab ends at an open domain boundary."""
    lo = rank - 1 if rank > 0 else (world - 1 if periodic else None)
    hi = rank + 1 if rank < world - 1 else (0 if periodic else None)
    return lo, hi


def exchange(send_lo, send_hi, recv_lo, recv_hi, rank: int, world: int, periodic: bool, group=None):
    """One halo exchange: send_hi -> the upper neighbour's recv_lo, send_lo -> the lower neighbour's recv_hi.
    Tensors may live on any device the process group's backend serves.  Runs on torch's CURRENT stream (wrap the call
    in `torch.cuda.stream(ctx.stream)`), so it is ordered between the context's pack and unpack copies.  With one
    rank and a periodic dimension the slab is its own neighbour: two device copies."""
    import torch
    lo, hi = neighbours(rank, world, periodic)
    if world == 1:
        if hi is not None:
            recv_lo.copy_(send_hi, non_blocking=True)
            recv_hi.copy_(send_lo, non_blocking=True)
        return
    import torch.distributed as dist
    ops = []
    # two ranks with a periodic dimension: both faces go to the same peer; tags keep the two messages apart where the
    # backend matches by tag (gloo), order does where it matches by order (NCCL): sends and receives are listed in
    # the same face order on both sides
    if hi is not None:
        ops.append(dist.P2POp(dist.isend, send_hi, hi, group=group, tag=1))
    if lo is not None:
        ops.append(dist.P2POp(dist.isend, send_lo, lo, group=group, tag=2))
    if lo is not None:
        ops.append(dist.P2POp(dist.irecv, recv_lo, lo, group=group, tag=1))
    if hi is not None:
        ops.append(dist.P2POp(dist.irecv, recv_hi, hi, group=group, tag=2))
    if ops:
        for w in dist.batch_isend_irecv(ops):
            w.wait()              # NCCL: the current stream waits, the host does not


class SlabStepper:
    """One rank's slab: an Agate context with its cut faces marked, its four halo buffers, and the step loop."""

    def __init__(self, ctx, rank: int, world: int, periodic: bool, group=None):
        self.ctx, self.rank, self.world, self.periodic, self.group = ctx, rank, world, periodic, group
        lo, hi = neighbours(rank, world, periodic)
        ctx.set_slab(lo is not None, hi is not None)
        self.cut_lo, self.cut_hi = lo is not None, hi is not None
        self.send_lo, self.send_hi, self.recv_lo, self.recv_hi = ctx.halo_buffers()
        self.rk = int(ctx.cfg.rk)
        self._fused_valid = False
        try:
            self._vmax = ctx.vmax_tensor()              # None: this kernel keeps no fused v_max (1-D grids, CGL)
        except Exception:
            self._vmax = None

    def reset(self):
        """Call after ctx.set_state(): the next step takes v_max from the reduction pass, not from a previous step."""
        self._fused_valid = False

    def _allreduce_vmax(self):
        import torch
        ctx = self.ctx
        if self._fused_valid and self._vmax is not None:
            # the last stage of the previous step left this slab's v_max on the device: all-reduce it in place
            if self.world > 1:
                import torch.distributed as dist
                with torch.cuda.stream(ctx.stream):
                    dist.all_reduce(self._vmax, op=dist.ReduceOp.MAX, group=self.group)
            return
        vm = ctx.get_vmax()                             # first step after set_state, or a kernel without the fused A7
        if self.world > 1:
            import torch.distributed as dist
            t = torch.tensor([vm], dtype=torch.float64, device=ctx.device)
            dist.all_reduce(t, op=dist.ReduceOp.MAX, group=self.group)
            vm = float(t.item())
        ctx.set_vmax(vm)

    def step(self):
        import torch
        ctx = self.ctx
        self._allreduce_vmax()
        ctx.step_begin(0.0)
        for s in range(self.rk):
            ctx.stage_pre(s, self.send_lo if self.cut_lo else None, self.send_hi if self.cut_hi else None)
            with torch.cuda.stream(ctx.stream):
                exchange(self.send_lo, self.send_hi, self.recv_lo, self.recv_hi, self.rank, self.world, self.periodic,
                         self.group)
            ctx.stage_post(s, self.recv_lo if self.cut_lo else None, self.recv_hi if self.cut_hi else None)
        self._fused_valid = True
