"""Multi-GPU plumbing: one process per GPU, one time frame per rank, no data-path collective.

Sectors and time frames are independent units (PAPER.md:49 sector-local tracking; PAPER.md:185 one
time frame per GPU on the farm), so the only communication is the timing/throughput reduction below.
"""
from __future__ import annotations

import os


def init(world: int, rank: int, backend: str = "nccl"):
    import torch.distributed as dist
    if not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29511")
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return dist


def aggregate(dist, ms_local: float, units_local: int):
    """(max over ranks of the elapsed ms, sum over ranks of the units processed)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(ms_local), int(units_local)
    import torch
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([ms_local], dtype=torch.float64, device=dev)
    u = torch.tensor([units_local], dtype=torch.int64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), int(u.item())


def shard_sectors(n_sectors: int, world: int, rank: int) -> tuple[int, int]:
    """Contiguous sector range [b, e) of `rank` when ONE frame is split over ranks (strong-scaling option)."""
    b = (n_sectors * rank) // world
    e = (n_sectors * (rank + 1)) // world
    return b, e
