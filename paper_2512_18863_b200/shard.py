"""Multi-GPU sharding of the dose path: argument bookkeeping only.

Control points are independent units and Eq. 9 is a sum over them, so rank r of N takes the
contiguous block [n_cp*r/N, n_cp*(r+1)/N); density, tables and dL/dDose are replicated.  The forward ends with ONE
sum all-reduce of the dose grid; the backward needs no reduction (gradient rows of different control points are
disjoint) — only a gather of the [n_cp][...] rows when one rank wants them all.

`ShardedDose` is the per-rank driver `bench.py --gpus N` runs: it owns the rank's slice of the parameters and calls an
engine (anything with `dose(leaves, jaws, gantry, mu, out=)` / `dose_backward(..., g, out=)`: the CUDA `Engine`, or a
stub in the CPU tests) on it.  A rank whose block is empty (n_cp < world) calls nothing and contributes zeros.
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
    width = max(max(hi - lo for lo, hi in sizes), 1)
    pad = torch.zeros((width,) + tuple(rows.shape[1:]), dtype=rows.dtype, device=rows.device)
    pad[: rows.shape[0]] = rows
    parts = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(parts, pad)
    return torch.cat([p[: hi - lo] for p, (lo, hi) in zip(parts, sizes)], dim=0)


class ShardedDose:
    """One rank's share of a full-arc forward / backward.

    engine      object with dose(leaves, jaws, gantry, mu, out=) and dose_backward(leaves, jaws, gantry, mu, g, out=)
    leaves, jaws, gantry, mu   the WHOLE arc (torch tensors on the rank's device); the rank keeps rows [lo, hi)
    dose_shape  shape of the dose grid
    """

    def __init__(self, engine, leaves, jaws, gantry, mu, dose_shape, rank: int, world: int):
        import torch
        self.engine, self.rank, self.world = engine, rank, world
        self.n_cp = int(gantry.shape[0])
        self.lo, self.hi = shard_range(self.n_cp, rank, world)
        self.leaves, self.jaws = leaves[self.lo:self.hi].contiguous(), jaws[self.lo:self.hi].contiguous()
        self.gantry, self.mu = gantry[self.lo:self.hi].contiguous(), mu[self.lo:self.hi].contiguous()
        self.dose = torch.zeros(tuple(dose_shape), dtype=torch.float32, device=gantry.device)
        self.grads = (torch.zeros_like(self.leaves), torch.zeros_like(self.jaws), torch.zeros_like(self.mu))

    @property
    def empty(self) -> bool:
        return self.hi <= self.lo

    def forward(self):
        """Partial dose of this rank's control points, then the one sum all-reduce: every rank ends with the arc dose."""
        if self.empty:
            self.dose.zero_()
        else:
            self.engine.dose(self.leaves, self.jaws, self.gantry, self.mu, out=self.dose)
        return reduce_dose(self.dose)

    def backward(self, g):
        """Gradient rows of this rank's control points (no collective: rows of different control points are disjoint)."""
        if not self.empty:
            self.engine.dose_backward(self.leaves, self.jaws, self.gantry, self.mu, g, out=self.grads)
        return self.grads

    def gather(self):
        """[n_cp][...] gradient arrays on every rank."""
        return tuple(gather_rows(t, self.n_cp) for t in self.grads)
