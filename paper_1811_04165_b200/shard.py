"""Multi-GPU plumbing: how independent beams (the bench) or one beam's DM rows (dm_rows_of_rank / gather_rows) are
spread over ranks and how per-rank device times are combined.  No data-path collective exists (the paper's cluster runs one beam per
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


def dm_rows_of_rank(ndm: int, rank: int, world: int, multiple: int = 1) -> Tuple[int, int]:
    """[lo, hi) of the DM rows rank `rank` searches when ONE beam's trial list is split over the ranks (SURVEY 8(e):
    contiguous ranges, so that a rank's delay apron only grows with its own largest DM; 8(f) f3).  `multiple` keeps
    range boundaries on multiples of a block of rows (e.g. the fine DMs of one coarse DM of a subband plan).  Every
    row belongs to exactly one rank; sizes differ by at most one block."""
    if world <= 0 or not (0 <= rank < world) or ndm < 0 or multiple < 1 or ndm % multiple:
        raise ValueError("bad (ndm, rank, world, multiple) = (%d, %d, %d, %d)" % (ndm, rank, world, multiple))
    blocks = ndm // multiple
    base, extra = divmod(blocks, world)
    lo = rank * base + min(rank, extra)
    return lo * multiple, (lo + base + (1 if rank < extra else 0)) * multiple


def plan_for_rank(cfg, rank: int, world: int, **plan_kw):
    """(plan, lo, hi): the plan of rank `rank` when ONE beam's DM trials are split over `world` GPUs (SURVEY 8(e),
    8(f) f3).  A direct plan gets the slice dm_list[lo:hi]; a subband plan gets whole coarse trials (a slice of the
    coarse grid with all its fine trials), so lo and hi are multiples of n_fine.  Delays are relative to the highest
    channel frequency whatever the slice (DD.3), so the rows a rank computes are bit for bit the rows lo..hi-1 of the
    one-GPU search; every rank reads the same input (its plan needs only its own largest delay of it) and the S/N
    tables meet in gather_rows.  The coarse DMs of a slice are coarse_first + lo/n_fine * step + a * step: identical to
    the one-GPU grid when first and step are dyadic (as in BASELINE.json), else equal up to the last bit of a DM."""
    import numpy as np
    from .binding import plan_create
    sb = getattr(cfg, "subband", None)
    if sb is not None:
        lo, hi = dm_rows_of_rank(sb.n_coarse * sb.n_fine, rank, world, sb.n_fine)
        a0, na = lo // sb.n_fine, (hi - lo) // sb.n_fine
        if na == 0:
            return None, lo, hi
        plan = plan_create(cfg.chan_freq_mhz(), cfg.t_samp_s, None, cfg.widths, cfg.nsamp_out, n_subbands=sb.n_subbands,
                           n_coarse=na, coarse_dm_first=sb.coarse_first + a0 * sb.coarse_step,
                           coarse_dm_step=sb.coarse_step, n_fine=sb.n_fine, fine_dm_step=sb.fine_step, **plan_kw)
        return plan, lo, hi
    lo, hi = dm_rows_of_rank(cfg.ndm, rank, world)
    if hi == lo:
        return None, lo, hi
    plan = plan_create(cfg.chan_freq_mhz(), cfg.t_samp_s, np.ascontiguousarray(cfg.dm_list()[lo:hi]), cfg.widths,
                       cfg.nsamp_out, **plan_kw)
    return plan, lo, hi


def gather_rows(local, ndm: int, device=None):
    """The [ndm][nW] table of a search whose DM rows were split with dm_rows_of_rank: every rank passes its own rows
    (a float32 or int32 tensor [hi - lo][nW]); all ranks get the whole table.  This gather of at most a few hundred
    kilobytes is the only exchange of a DM-sharded search: every rank reads the whole input itself."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return local
    world = dist.get_world_size()
    sizes = [dm_rows_of_rank(ndm, r, world)[1] - dm_rows_of_rank(ndm, r, world)[0] for r in range(world)]
    most = max(sizes)  # all_gather wants equal shapes: pad every rank's rows to the largest share, trim afterwards
    mine = torch.zeros((most,) + tuple(local.shape[1:]), dtype=local.dtype, device=local.device)
    mine[: local.shape[0]] = local
    parts = [torch.empty_like(mine) for _ in range(world)]
    dist.all_gather(parts, mine)
    return torch.cat([p[:n] for p, n in zip(parts, sizes)], dim=0)


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
