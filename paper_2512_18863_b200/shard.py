"""Multi-GPU sharding of the dose path: argument bookkeeping only.

Control points are independent units and Eq. 9 is a sum over them, so rank r of N takes the
contiguous block [n_cp*r/N, n_cp*(r+1)/N); density, tables and dL/dDose are replicated.  The forward ends with ONE
sum all-reduce of the dose grid; the backward needs no reduction (gradient rows of different control points are
disjoint) — only a gather of the [n_cp][...] rows when one rank wants them all.
"""
from __future__ import annotations


def shard_range(n_cp: int, rank: int, world: int) -> tuple[int, int]:
    """Half-open range of control points of `rank`; the ranges tile [0, n_cp) and differ in size by at most 1."""
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    return (n_cp * rank) // world, (n_cp * (rank + 1)) // world


def reduce_dose(dose):
    """Sum all-reduce of a rank's partial dose grid (torch tensor, in place); a no-op without a process group."""
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(dose)
    return dose


def gather_rows(rows, n_cp: int):
    """All-gather of per-control-point gradient rows ([hi-lo][...] on each rank) into [n_cp][...] on every rank."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return rows
    world = dist.get_world_size()
    sizes = [shard_range(n_cp, r, world) for r in range(world)]
    width = max(hi - lo for lo, hi in sizes)
    pad = torch.zeros((width,) + tuple(rows.shape[1:]), dtype=rows.dtype, device=rows.device)
    pad[: rows.shape[0]] = rows
    parts = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(parts, pad)
    return torch.cat([p[: hi - lo] for p, (lo, hi) in zip(parts, sizes)], dim=0)
