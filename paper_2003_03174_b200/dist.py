"""Multi-GPU plumbing.  The tracking step shards by independent problems: tracks never read each
other's state ("Parallelization can easily be achieved over the tracks") and time frames
are independent, so every rank runs the whole path on its own time frame (or its own
contiguous slice of the tracks, with the tracklet index replicated) and there is NO data-path
collective.  torch.distributed is used only for the barrier and the max-over-ranks of the timings.
"""
from __future__ import annotations

import os
from typing import Tuple


def env_rank() -> Tuple[int, int, int]:
    """(rank, world_size, local_rank) from the torchrun environment; (0, 1, 0) outside it."""
    return (int(os.environ.get("RANK", 0)), int(os.environ.get("WORLD_SIZE", 1)), int(os.environ.get("LOCAL_RANK", 0)))


def init(backend: str, device=None):
    """Initialise torch.distributed from the torchrun environment (also for a single rank, so that the same
    barrier / all-reduce code runs at every N).  Returns (rank, world)."""
    rank, world, _ = env_rank()
    if world > 1 or "TORCHELASTIC_RUN_ID" in os.environ:
        import torch.distributed as dist
        if not dist.is_initialized():
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            os.environ.setdefault("MASTER_PORT", "29500")
            kw = dict(device_id=device) if (device is not None and backend == "nccl") else {}
            dist.init_process_group(backend=backend, rank=rank, world_size=world, **kw)
    return rank, world


def shutdown():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.destroy_process_group()


def track_slice(n_tracks: int, rank: int, world: int) -> Tuple[int, int]:
    """Contiguous slice [lo, hi) of the tracks owned by `rank` when ONE time frame is split over the
    ranks (strong scaling): sizes differ by at most one, the slices tile [0, n_tracks) in rank order."""
    base, rem = divmod(n_tracks, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def _reduce(value: float, op_name: str, device) -> float:
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=getattr(dist.ReduceOp, op_name))
    return float(t.item())


def max_over_ranks(value: float, device="cpu") -> float:
    return _reduce(value, "MAX", device)


def sum_over_ranks(value: float, device="cpu") -> float:
    return _reduce(value, "SUM", device)


def gather_sharded(shard: dict, n_tracks: int) -> dict:
    """Strong scaling leaves the outputs sharded by `track_slice`; this puts the shards of all ranks back together
    (last axis = tracks, rank order = track order) on every rank.  Not part of any timed path."""
    import numpy as np
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return shard
    parts = [None] * dist.get_world_size()
    dist.all_gather_object(parts, {k: np.ascontiguousarray(v) for k, v in shard.items()})
    full = {k: np.concatenate([p[k] for p in parts], axis=-1) for k in shard}
    assert all(v.shape[-1] == n_tracks for v in full.values())
    return full
