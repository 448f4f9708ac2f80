"""Frequency-channel sharding across ranks (host logic only, no arithmetic of the method).

Channels are independent ("each frequency band can be processed independently",
PAPER.md:39), so the path shards over F with disjoint inputs and outputs and NO data-path
collective.  The only cross-rank operations are the ones bench.py needs for timing: a barrier and
a max over ranks of the device-timed duration.
"""
from __future__ import annotations


def channel_range(F_total: int, rank: int, world: int) -> tuple[int, int]:
    """Channels [f0, f1) owned by `rank`: contiguous blocks, sizes differ by at most one, the
    first F_total % world ranks get the larger blocks.  Blocks are disjoint and cover [0, F_total)."""
    if F_total < 0 or world < 1 or not (0 <= rank < world):
        raise ValueError("need F_total >= 0, world >= 1, 0 <= rank < world")
    q, r = divmod(F_total, world)
    f0 = rank * q + min(rank, r)
    return f0, f0 + q + (1 if rank < r else 0)


def shard_packed(packed, rank: int, world: int):
    """This rank's channels of a [T][F][N] stream as a contiguous [T][F_local][N] array (numpy
    array or torch tensor; a copy, because corr_execute needs the local stream contiguous)."""
    f0, f1 = channel_range(packed.shape[1], rank, world)
    part = packed[:, f0:f1, :]
    return part.contiguous() if hasattr(part, "contiguous") else part.copy()


def max_over_ranks(seconds: float, device=None) -> float:
    """Max over ranks of a per-rank duration (the job's time is its slowest rank's).  A no-op
    without an initialised process group."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(seconds)
    t = torch.tensor([seconds], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
