"""Pose sharding across ranks: poses are independent units and the packed
scene is tiny, so every rank holds the whole scene (one psdf_create_scene per device) and a
contiguous slice of the poses.  There is NO collective on the data path; the only
collectives are the optional all-gather of the results for a single consumer and the
max-over-ranks reduction of the step time in bench.py.  Host logic only: no PSDF
arithmetic lives here.  Works with any torch.distributed backend (nccl on GPUs, gloo in
the CPU tests).
"""
from __future__ import annotations

from typing import Callable, Optional, Tuple

import numpy as np


def shard_range(n: int, rank: int, world: int) -> Tuple[int, int]:
    """Contiguous slice [begin, end) of n poses owned by `rank`; sizes differ by at most one,
    the first n % world ranks take the extra pose.  Empty slices are legal (n < world)."""
    if world < 1 or not (0 <= rank < world) or n < 0:
        raise ValueError(f"bad shard request n={n} rank={rank} world={world}")
    base, extra = divmod(n, world)
    begin = rank * base + min(rank, extra)
    return begin, begin + base + (1 if rank < extra else 0)


def max_over_ranks(seconds, group=None, device: Optional[str] = None):
    """MAX-reduce of per-rank timings (a float or a sequence of floats); identity when
    torch.distributed is not initialised.  Returns a list of floats."""
    import torch
    import torch.distributed as dist
    vals = [float(seconds)] if np.isscalar(seconds) else [float(s) for s in seconds]
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return vals
    if device is None:
        device = "cuda" if dist.get_backend(group) == "nccl" else "cpu"
    t = torch.tensor(vals, dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return [float(x) for x in t.cpu()]


def eval_sharded(evaluate: Callable, poses, group=None, gather: bool = True):
    """Evaluates this rank's slice of `poses` [N,3] (torch tensor, same on every rank) with
    `evaluate(poses_slice) -> (value[n], grad[n,3])` (e.g. a bound Scene.eval) and, if
    `gather`, all-gathers the packed [N,4] = (value, grad) rows so that every rank returns
    the full (value[N], grad[N,3]); otherwise returns the local slice and its range.
    Uneven slices are padded to the largest one for the collective and trimmed after."""
    import torch
    import torch.distributed as dist
    on = dist.is_available() and dist.is_initialized()
    world = dist.get_world_size(group) if on else 1
    rank = dist.get_rank(group) if on else 0
    n = int(poses.shape[0])
    b, e = shard_range(n, rank, world)
    value, grad = evaluate(poses[b:e])
    if not gather:
        return value, grad, (b, e)
    if world == 1:
        return value, grad
    cap = -(-n // world) if n else 0
    packed = torch.zeros((cap, 4), dtype=value.dtype, device=value.device)
    packed[: e - b, 0] = value
    packed[: e - b, 1:] = grad
    if value.is_cuda:
        out = torch.empty((world * cap, 4), dtype=value.dtype, device=value.device)
        dist.all_gather_into_tensor(out, packed, group=group)
    else:
        parts = [torch.empty_like(packed) for _ in range(world)]
        dist.all_gather(parts, packed, group=group)
        out = torch.cat(parts, 0)
    rows = []
    for r in range(world):
        rb, re_ = shard_range(n, r, world)
        rows.append(out[r * cap: r * cap + (re_ - rb)])
    full = torch.cat(rows, 0) if rows else out[:0]
    return full[:, 0].contiguous(), full[:, 1:].contiguous()
