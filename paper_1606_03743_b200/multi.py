"""Multi-GPU plumbing of the bemcub path: one process per GPU,
the mesh replicated, FIELD POINTS (eval) or MATRIX ROWS (assemble) sharded by contiguous ranges.
The data path has no exchange step, hence no collective: every rank evaluates its own range with
the full element list (field points are independent, element contributions add).
`torch.distributed` is used only for the barrier, the max-over-ranks timing and, when the caller
wants the whole result on one rank, a gather of the outputs.

For a handful of field points (a tracker's calls, L32) the other natural sharding is by ELEMENTS:
every rank holds a contiguous range of the mesh, evaluates the same field points against it, and the
per-point sums (32 bytes per field point) are added over the ranks - the one exchange step this path
has, and a tiny one.  `sum_in_rank_order` does it as an all-gather followed by a sum in rank order, so
every rank ends with the same bits whatever the backend's reduction order.

No arithmetic of the method lives here beyond that sum.  Works with any backend (`nccl` on GPUs, `gloo` in the
CPU tests).
"""
from __future__ import annotations

from .synth import shard_range


def world():
    """(rank, world_size) of the default process group, (0, 1) without one."""
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        return dist.get_rank(), dist.get_world_size()
    return 0, 1


def my_range(total: int) -> tuple[int, int]:
    """This rank's contiguous [lo, hi) of `total` field points / matrix rows."""
    rank, ws = world()
    return shard_range(total, rank, ws)


def max_over_ranks(value: float, device=None) -> float:
    """Timing rule of the bench contract: a step takes as long as its slowest rank."""
    import torch
    import torch.distributed as dist
    rank, ws = world()
    if ws == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, device=None) -> float:
    """Units processed by the whole job (weak scaling: every rank brings its own units)."""
    import torch
    import torch.distributed as dist
    rank, ws = world()
    if ws == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def gather_rows(local, total: int, dst: int = 0):
    """Concatenates the per-rank blocks `local` ([hi-lo, ...] tensors, rank order = row order) of a
    result with `total` rows on rank `dst`; returns None elsewhere.  Ranges may differ by one row, so
    blocks are padded to the largest before the gather."""
    import torch
    import torch.distributed as dist
    rank, ws = world()
    if ws == 1:
        return local
    sizes = [shard_range(total, r, ws) for r in range(ws)]
    big = max(hi - lo for lo, hi in sizes)
    pad = torch.zeros((big,) + tuple(local.shape[1:]), dtype=local.dtype, device=local.device)
    pad[: local.shape[0]] = local
    bufs = [torch.empty_like(pad) for _ in range(ws)] if rank == dst else None
    dist.gather(pad, bufs, dst=dst)
    if rank != dst:
        return None
    return torch.cat([b[: hi - lo] for b, (lo, hi) in zip(bufs, sizes)], dim=0)


def sum_in_rank_order(local):
    """Element-sharded evaluation: `local` = this rank's partial Phi / E sums for the SAME field points
    (any shape, same on every rank).  Returns their sum over the ranks, added in rank order, on every rank."""
    import torch
    import torch.distributed as dist
    rank, ws = world()
    if ws == 1:
        return local
    bufs = [torch.empty_like(local) for _ in range(ws)]
    dist.all_gather(bufs, local.contiguous())
    total = bufs[0].clone()
    for b in bufs[1:]:
        total += b
    return total
