"""Rank-side plumbing for multi-GPU runs (one process per GPU, torch.distributed).

The cone-beam operators shard with no data-path collective: channels (and
whole volumes) are independent (DESIGN.md s.10).  This module holds the small
host-side pieces bench.py needs -- which channels a rank owns, the max over
ranks of device timings, rank-0 reporting -- so they can be tested on CPU with
the gloo backend (tests/test_dist_cpu.py).
"""
from __future__ import annotations

import os
from typing import Sequence, Tuple


def env_world() -> Tuple[int, int, int]:
    """(rank, local_rank, world_size) from the torchrun environment (1 process if unset)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def channel_shard(channels: int, rank: int, world: int) -> Tuple[int, int]:
    """Contiguous balanced split of `channels` over `world` ranks: (first, count).
    The first `channels % world` ranks get one extra channel; counts may be 0."""
    if channels < 0 or world < 1 or not (0 <= rank < world):
        raise ValueError("bad shard request")
    base, extra = divmod(channels, world)
    first = rank * base + min(rank, extra)
    return first, base + (1 if rank < extra else 0)


def max_over_ranks(values: Sequence[float], device="cpu"):
    """Element-wise MAX over all ranks of a list of floats (identity if not distributed)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t.cpu()]


def sum_over_ranks(values: Sequence[float], device="cpu"):
    """Element-wise SUM over all ranks (work counters for the whole-job aggregate)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return [float(x) for x in t.cpu()]


def barrier(cuda: bool = False):
    """synchronize + barrier + synchronize (the bracket bench.py puts around the timed region)."""
    import torch
    import torch.distributed as dist
    if cuda:
        torch.cuda.synchronize()
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.barrier()
    if cuda:
        torch.cuda.synchronize()
