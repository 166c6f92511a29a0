"""Host-side multi-GPU logic: snapshots are independent problems
(PAPER.md:81, 115 -- every time sample has its own V, grid and image), so N GPUs shard a run
by snapshot index with NO data-path collective.  The only cross-rank traffic is the timing
reduction of bench.py (max over ranks) and the final count of units processed.

No imaging arithmetic lives here.
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def snapshot_shard(n_snapshots: int, rank: int, world_size: int) -> range:
    """Snapshot indices of `rank`: round-robin (n = rank, rank + W, ...), so consecutive time
    samples land on different GPUs and every rank's share differs by at most one."""
    if world_size < 1 or not (0 <= rank < world_size) or n_snapshots < 0:
        raise ValueError("bad shard request: n=%d rank=%d world=%d" % (n_snapshots, rank, world_size))
    return range(rank, n_snapshots, world_size)


def reduce_timing(elapsed_ms: float, units: float, device="cpu"):
    """-> (max over ranks of elapsed_ms, sum over ranks of units).  With no process group
    (single process) it returns its inputs."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(elapsed_ms), float(units)
    t = torch.tensor([float(elapsed_ms)], dtype=torch.float64, device=device)
    u = torch.tensor([float(units)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def barrier():
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.barrier()
