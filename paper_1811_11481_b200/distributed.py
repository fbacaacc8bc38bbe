"""Multi-GPU plumbing: one process per GPU, no data-path collective.

Sectors and time frames are independent units (PAPER.md:49 sector-local tracking; PAPER.md:185 one time frame per GPU
on the farm).  Two ways to use N GPUs, both running the unchanged single-GPU library on every rank:
  * frames  -- every rank tracks its own time frame (weak scaling; the farm's mode);
  * sectors -- ONE frame is split into contiguous sector ranges: rank r tracks sectors
    shard_sectors(36, N, r); track ids become global by adding the exclusive scan of the per-rank track counts.
The only communication is the timing / throughput reduction and, for the sector split, one all-gather of the
per-rank track counts (4 bytes per rank).  This module holds index arithmetic only -- no tracking step.

Limit of the sector split: tpcca_merge / tpcca_find_legs / tpcca_fit_legs run per rank on the rank's own sectors, and no
boundary records are exchanged.  A track crossing from the last sector of one rank into the first sector of the next
therefore stays two segments (and the ring closure 17 -> 0 is lost whenever a z side is spread over several ranks).  Only
splits whose cuts all fall between the two z sides -- world == 2 for the 36-sector TPC -- give the whole-frame merged
tracks; `cuts_inside_a_side` tells which case applies and bench.py reports it.  tpcca_track itself (assignment, sector
tracks) is exact for every split.
"""
from __future__ import annotations

import os

import numpy as np


def init(world: int, rank: int, backend: str = "nccl"):
    import torch.distributed as dist
    if not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29511")
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return dist


def _dev(dist):
    return "cuda" if dist.get_backend() == "nccl" else "cpu"


def aggregate(dist, ms_local: float, units_local: int):
    """(max over ranks of the elapsed ms, sum over ranks of the units processed)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(ms_local), int(units_local)
    import torch
    t = torch.tensor([ms_local], dtype=torch.float64, device=_dev(dist))
    u = torch.tensor([units_local], dtype=torch.int64, device=_dev(dist))
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), int(u.item())


def shard_sectors(n_sectors: int, world: int, rank: int) -> tuple[int, int]:
    """Contiguous sector range [b, e) of `rank` when ONE frame is split over ranks."""
    b = (n_sectors * rank) // world
    e = (n_sectors * (rank + 1)) // world
    return b, e


def cuts_inside_a_side(n_sectors: int, world: int, ring: int) -> int:
    """How many rank boundaries of `shard_sectors` cut through a z side (a ring of `ring` sectors) instead of falling
    between two sides.  0: the per-rank merger sees every pair of neighbouring sectors, so merged tracks equal the
    whole-frame ones; > 0: segments meeting at those cuts (and at the ring closure of a divided side) stay unmerged."""
    if ring <= 0 or world <= 1:
        return 0
    return sum(1 for r in range(1, world) if 0 < shard_sectors(n_sectors, world, r)[0] < n_sectors
               and shard_sectors(n_sectors, world, r)[0] % ring != 0)


def shard_frame(clusters: np.ndarray, sector_offsets: np.ndarray, world: int, rank: int):
    """The rank's piece of one frame: (clusters[lo:hi], re-based CSR offsets over ALL sectors, lo).

    The offsets keep n_sectors + 1 entries (sectors outside the rank's range are empty), so the library handle is the
    same on every rank and the sector numbers in the track records stay global."""
    so = np.asarray(sector_offsets, dtype=np.int64)
    ns = len(so) - 1
    b, e = shard_sectors(ns, world, rank)
    lo, hi = int(so[b]), int(so[e])
    local = (np.clip(so, lo, hi) - lo).astype(np.int32)
    return clusters[lo:hi], local, lo


def track_id_offsets(counts) -> np.ndarray:
    """Exclusive scan of the per-rank track counts: the global id of rank r's track i is offsets[r] + i.  Track ids are
    in (sector, row, ...) order (A4), so the concatenation over ranks IS the whole-frame numbering."""
    c = np.asarray(counts, dtype=np.int64)
    return np.concatenate([[0], np.cumsum(c)[:-1]]).astype(np.int64)


def gather_counts(dist, n_local: int) -> np.ndarray:
    """all-gather of one int per rank (the track count); [n_local] without a process group."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return np.array([n_local], dtype=np.int64)
    import torch
    mine = torch.tensor([n_local], dtype=torch.int64, device=_dev(dist))
    out = [torch.zeros_like(mine) for _ in range(dist.get_world_size())]
    dist.all_gather(out, mine)
    return np.array([int(t.item()) for t in out], dtype=np.int64)


def globalise_assignment(local_assign: np.ndarray, id_offset: int) -> np.ndarray:
    """Local track ids -> global ones (-1 stays -1)."""
    a = np.asarray(local_assign).astype(np.int64)
    return np.where(a >= 0, a + int(id_offset), -1).astype(np.int32)
