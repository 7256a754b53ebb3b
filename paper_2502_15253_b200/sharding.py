"""Multi-GPU layer of the hot path: shard the batch of parameter points across ranks.

SURVEY.md 8(e): the path shards BY PARAMETER POINT.  Every rank holds the
whole event store and evaluates a contiguous slice of the batch with its own libphylino context;
no floating-point reduction crosses ranks and nothing is summed across them.  A slice is a batch of
another size, so the library may cut its work differently (unit length, schedule, sub-stream split:
which events a lane sums in fp64 before the exact integer accumulation): the gathered rows agree with
the one-GPU call to rounding -- <= 1e-13 relative per bin, <= 1e-9 in the NLL, measured with the real
library in tests/test_gpu_schedules.py::test_point_shards_agree_with_the_unsharded_batch -- not bit
for bit, and each slice meets the parity bars against the CPU reference on its own.  Reruns of the same split are
bit-identical.
The only exchange is an all-gather of the per-point results (`nll[P]`, or `hist[P x bins]`),
done with `torch.distributed` (NCCL on GPUs; gloo in the CPU tests).  There is no data-path
collective inside the kernels and nothing here computes: this module only slices, pads and gathers.
"""
from __future__ import annotations

from typing import Callable, Optional, Tuple

import torch
import torch.distributed as dist


def shard_points(n_points: int, world: int, rank: int) -> Tuple[int, int]:
    """Contiguous balanced slice [lo, hi) of a batch of n_points for `rank` of `world`:
    the first n_points % world ranks hold one point more.  Empty slices are legal (P < world)."""
    if n_points < 0 or world < 1 or not (0 <= rank < world):
        raise ValueError(f"shard_points({n_points}, {world}, {rank})")
    base, extra = divmod(n_points, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def shard_sizes(n_points: int, world: int):
    return [shard_points(n_points, world, r)[1] - shard_points(n_points, world, r)[0] for r in range(world)]


def all_gather_points(local: torch.Tensor, n_points: int, group: Optional[dist.ProcessGroup] = None) -> torch.Tensor:
    """Gather per-point rows (`local` = this rank's slice, shape [n_local, ...]) into the full
    [n_points, ...] tensor on every rank.  Slices differ by at most one row, so every rank pads
    to the largest slice, one all_gather moves the padded blocks, and the padding is cut off."""
    if not (dist.is_available() and dist.is_initialized()):
        if local.shape[0] != n_points:
            raise ValueError("single process: the local slice must be the whole batch")
        return local
    world, rank = dist.get_world_size(group), dist.get_rank(group)
    sizes = shard_sizes(n_points, world)
    if local.shape[0] != sizes[rank]:
        raise ValueError(f"rank {rank}: slice has {local.shape[0]} rows, expected {sizes[rank]}")
    width = max(sizes)
    tail = tuple(local.shape[1:])
    padded = torch.zeros((width,) + tail, dtype=local.dtype, device=local.device)
    padded[: sizes[rank]] = local
    blocks = [torch.empty_like(padded) for _ in range(world)]
    dist.all_gather(blocks, padded, group=group)
    return torch.cat([b[:n] for b, n in zip(blocks, sizes)], dim=0)


def sharded_eval(evaluate: Callable[[torch.Tensor], torch.Tensor], params: torch.Tensor,
                 group: Optional[dist.ProcessGroup] = None) -> torch.Tensor:
    """Evaluate `evaluate(params[lo:hi])` on this rank's slice of the batch and gather the rows of
    every rank.  `evaluate` is the caller's bound call into the library, e.g.
    `lambda p: ph.nll(p, data)` or `ph.spectra`; it must return one row per point."""
    n_points = params.shape[0]
    if dist.is_available() and dist.is_initialized():
        world, rank = dist.get_world_size(group), dist.get_rank(group)
    else:
        world, rank = 1, 0
    lo, hi = shard_points(n_points, world, rank)
    local = evaluate(params[lo:hi].contiguous())
    if local.shape[0] != hi - lo:
        raise ValueError("evaluate() must return one row per parameter point")
    return all_gather_points(local, n_points, group)
