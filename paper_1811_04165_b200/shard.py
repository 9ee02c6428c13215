"""Multi-GPU plumbing of the bench: how independent beams are spread over ranks and how per-rank
device times are combined.  No data-path collective exists (the paper's cluster runs one beam per
GPU): ranks only agree on a time (max over ranks) and
on a unit count (sum over ranks), through `torch.distributed` (NCCL on the GPU box, gloo in the CPU
tests).  Nothing here computes any part of the search.
"""
from __future__ import annotations

from typing import List, Tuple


def beams_of_rank(n_beams: int, rank: int, world: int) -> List[int]:
    """Beam indices rank `rank` of `world` processes: contiguous blocks, sizes differing by at most
    one, every beam owned by exactly one rank."""
    if world <= 0 or not (0 <= rank < world) or n_beams < 0:
        raise ValueError("bad (n_beams, rank, world) = (%d, %d, %d)" % (n_beams, rank, world))
    base, extra = divmod(n_beams, world)
    lo = rank * base + min(rank, extra)
    return list(range(lo, lo + base + (1 if rank < extra else 0)))


from synth.filterbank import beam_seed  # noqa: E402,F401  (data recipe: lives with the generator)


def combine(local_ms: float, local_units: float, device=None) -> Tuple[float, float]:
    """(max over ranks of local_ms, sum over ranks of local_units).  A no-op without an initialised
    process group (single process)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(local_ms), float(local_units)
    t = torch.tensor([float(local_ms)], dtype=torch.float64, device=device)
    u = torch.tensor([float(local_units)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())
