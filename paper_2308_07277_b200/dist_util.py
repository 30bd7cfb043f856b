"""Multi-GPU plumbing for the band-parallel mode (one process per GPU, torch.distributed).

Every (band, k) unit of H|psi> is independent (the paper's band / k-point parallelism,
PAPER.md:1007-1008), so ranks only ever exchange *timings*: there is no data-path collective.
V_loc, beta and D are replicated; bands (or whole band sets) are partitioned.
"""
from __future__ import annotations


def shard_range(n_units: int, rank: int, world: int):
    """Contiguous, balanced partition of range(n_units): sizes differ by at most one."""
    if world < 1 or not (0 <= rank < world):
        raise ValueError("bad rank/world")
    base, rem = divmod(n_units, world)
    start = rank * base + min(rank, rem)
    return start, start + base + (1 if rank < rem else 0)


def units_per_step(n_units: int, world: int, scaling: str) -> int:
    """Whole-job units per step: weak = every rank processes its own full set; strong = one set split."""
    if scaling == "weak":
        return n_units * world
    if scaling == "strong":
        return n_units
    raise ValueError(scaling)


def max_over_ranks(values, device=None):
    """Element-wise MAX of a list of floats over all ranks (identity when not distributed)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return [float(v) for v in values]
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t.cpu()]
