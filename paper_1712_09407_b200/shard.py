"""Host-side sharding of the sector tracker over ranks (one process per GPU).

The path needs no exchange step: sectors are tracked "individually", the paper's CPU
tracker used "trivial parallelization over the sectors" (L112), and events are independent.  So
the two ways to use N GPUs are

* event-level data parallelism (what ``bench.py --gpus N`` times): rank r tracks events
  r, r + N, r + 2N, ... of the stream; no collective on the data path; and
* a sector partition of ONE event: rank r tracks a contiguous range of sectors; the only
  communication is one gather of the (small) track lists at the end.

This module holds only index arithmetic and the gather — no tracker arithmetic.  The ``track``
callable that turns a sub-event into tracks is supplied by the caller (``SectorTracker.track_event``
on a GPU box; the CPU tests pass the oracle), so the logic is testable with the ``gloo`` backend.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np


def event_shard(n_events: int, rank: int, world: int) -> range:
    """Events of a stream that rank `rank` of `world` tracks: rank, rank + world, ..."""
    if world < 1 or not 0 <= rank < world:
        raise ValueError("need 0 <= rank < world")
    return range(rank, n_events, world)


def sector_shard(n_sectors: int, rank: int, world: int) -> range:
    """Contiguous sector range of rank `rank`; sizes differ by at most one, low ranks get the extra."""
    if world < 1 or not 0 <= rank < world:
        raise ValueError("need 0 <= rank < world")
    q, r = divmod(n_sectors, world)
    lo = rank * q + min(rank, r)
    return range(lo, lo + q + (1 if rank < r else 0))


@dataclass
class SubEvent:
    xyz: np.ndarray         # float32 [n, 3] view of the caller's array (clusters of the shard's sectors)
    row_start: np.ndarray   # uint32 [n_local_sectors * n_rows + 1], rebased to start at 0
    first_cluster: int      # global index of the shard's first cluster
    first_sector: int
    n_sectors: int


def check_partition(n_sectors: int, world: int, cross_sector: bool = False) -> None:
    """Raise if the sector partition over `world` ranks is not usable: a rank without sectors (world > n_sectors) would
    hand the tracker an event of zero sectors; with cross-sector steps on (global tracking, track merging) every
    rank's range must be a whole number of 18-sector rings starting on a ring boundary."""
    if world < 1:
        raise ValueError("world must be >= 1")
    if world > n_sectors:
        raise ValueError(f"sector partition: {world} ranks for {n_sectors} sectors leaves ranks without work; "
                         "use event-level data parallelism (event_shard) instead")
    if cross_sector:
        for r in range(world):
            sh = sector_shard(n_sectors, r, world)
            if sh.start % 18 or len(sh) % 18:
                raise ValueError("global_tracking / merge_tracks look into the neighbouring sector: with them on, every "
                                 f"rank needs whole rings of 18 sectors, but rank {r} of {world} would get sectors "
                                 f"{sh.start}..{sh.stop - 1}; shard by events, or use at most n_sectors / 18 ranks")


def slice_event(xyz: np.ndarray, row_start: np.ndarray, n_rows: int, sectors: range) -> SubEvent:
    """The clusters of a contiguous sector range as an event of its own (input marshalling only)."""
    if sectors.step != 1:
        raise ValueError("sector range must be contiguous")
    if len(sectors) == 0:
        raise ValueError("empty sector range: this rank has no sectors to track")
    rs = np.asarray(row_start)
    lo, hi = sectors.start * n_rows, sectors.stop * n_rows
    c0, c1 = int(rs[lo]), int(rs[hi])
    sub_rs = (rs[lo:hi + 1].astype(np.int64) - c0).astype(np.uint32)
    return SubEvent(np.asarray(xyz).reshape(-1, 3)[c0:c1], sub_rs, c0, sectors.start, len(sectors))


def globalize(tracks: np.ndarray, cluster_ids: np.ndarray, sub: SubEvent):
    """Shard-local track records and cluster ids -> the event's sector numbers and cluster indices."""
    t = tracks.copy()
    t["sector"] += np.uint32(sub.first_sector)
    t["seed_cluster"] += np.uint32(sub.first_cluster)
    return t, (cluster_ids.astype(np.uint32) + np.uint32(sub.first_cluster))


def merge_shards(parts):
    """[(tracks, cluster_ids)] in rank order -> one track array + one id list, `first_cluster` rebased.

    Rank order is sector order, and inside a shard the tracker already emits tracks in (sector,
    start row, start index) order (G28), so concatenation keeps the output order.
    """
    tracks, ids, off = [], [], 0
    for t, c in parts:
        t = t.copy()
        t["first_cluster"] += np.uint32(off)
        off += len(c)
        tracks.append(t)
        ids.append(c)
    if not tracks:
        raise ValueError("no shards")
    return np.concatenate(tracks), np.concatenate(ids)


def track_event_sharded(track, xyz, row_start, n_sectors: int, n_rows: int, group=None, *, cross_sector: bool):
    """Track one event with its sectors partitioned over the ranks of `group` (torch.distributed).

    `track(sub: SubEvent) -> (tracks, cluster_ids)` runs the sector tracker on this rank's device.
    Every rank returns the merged (tracks, cluster_ids) of the whole event.  One all_gather of the
    track lists is the only communication; with the NCCL backend the objects travel via NVLink.

    The partition is exact for the plain sector tracker only (sectors are tracked "individually").
    `cross_sector` has no default on purpose: `track` is an opaque callback, so only the caller knows which cuts it
    runs with, and a forgotten flag would lose prolongations and links without any error.
    Pass cross_sector=True when `track` runs with global_tracking = 1 or merge_tracks = 1 (PAPER.md L116-L136, L28:
    the steps that look into the neighbouring sector): every rank must then hold whole rings of 18 sectors, which
    check_partition enforces — any other split would silently drop prolongations and links, because the kernels
    (and the oracle) skip those steps unless their sector count is a multiple of 18.
    """
    import torch.distributed as dist
    world = dist.get_world_size(group) if dist.is_initialized() else 1
    rank = dist.get_rank(group) if dist.is_initialized() else 0
    check_partition(n_sectors, world, cross_sector=cross_sector)
    sub = slice_event(xyz, row_start, n_rows, sector_shard(n_sectors, rank, world))
    t, c = track(sub)
    mine = globalize(t, c, sub)
    if world == 1:
        return merge_shards([mine])
    parts = [None] * world
    dist.all_gather_object(parts, mine, group=group)
    return merge_shards(parts)


def max_over_ranks(ms: float, group=None, device=None) -> float:
    """Device time of a multi-GPU step = the slowest rank's (never wall clock)."""
    import torch
    import torch.distributed as dist
    if not dist.is_initialized() or dist.get_world_size(group) == 1:
        return float(ms)
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return float(t.item())
