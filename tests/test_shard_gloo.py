"""The N > 1 path on CPU: world_size-2 gloo processes run the host-side sharding logic of
paper_1712_09407_b200/shard.py.  The tracker inside each rank is the CPU
oracle here (there is no GPU on this box); what is tested is the slicing, index rebasing, gather and
merge, and the max-over-ranks timing reduction that bench.py uses.

PAPER.md L28 ("reconstructs the tracks in each TPC sector individually") and L112 ("trivial
parallelization over the sectors") are what make the partition exact: the merged result of the
sector shards must be IDENTICAL to tracking the whole event at once.
"""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out_dir: str):
    if ROOT not in sys.path:
        sys.path.insert(0, ROOT)
    import torch.distributed as dist
    from oracle import Oracle
    from paper_1712_09407_b200 import shard
    from tpcsynth import generate_event
    from dataclasses import replace

    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ev = generate_event(3)                      # 36 sectors, pp-like
        R = ev.geometry.n_rows

        def track(sub):
            geo = replace(ev.geometry, n_sectors=sub.n_sectors)
            o = Oracle.for_geometry(geo).run(np.ascontiguousarray(sub.xyz), sub.row_start)
            # oracle track records -> the fields the shard module touches (same names as TRACK_DTYPE)
            return o.tracks, o.track_cluster_ids

        tracks, ids = shard.track_event_sharded(track, ev.xyz, ev.row_start, ev.geometry.n_sectors, R, cross_sector=False)
        ms = shard.max_over_ranks(10.0 + rank)      # slowest rank decides
        mine = list(shard.event_shard(7, rank, world))
        np.savez(os.path.join(out_dir, f"r{rank}.npz"), tracks=tracks, ids=ids, ms=ms, mine=np.array(mine))
    finally:
        dist.destroy_process_group()


def test_sector_partition_matches_whole_event_world2(tmp_path, oracle_run):
    import torch.multiprocessing as mp
    world, port = 2, _free_port()
    mp.start_processes(_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True, start_method="spawn")
    ev, o = oracle_run(3)
    for rank in range(world):
        z = np.load(tmp_path / f"r{rank}.npz")
        assert np.array_equal(z["ids"], o.track_cluster_ids)
        t = z["tracks"]
        assert len(t) == len(o.tracks)
        for f in o.tracks.dtype.names:
            assert np.array_equal(t[f], o.tracks[f]), f
        assert float(z["ms"]) == 11.0
        assert list(z["mine"]) == list(range(rank, 7, world))


def test_shard_index_arithmetic():
    from paper_1712_09407_b200 import shard
    for n, w in [(36, 1), (36, 2), (36, 8), (36, 5), (1, 1), (3, 4)]:
        got = [s for r in range(w) for s in shard.sector_shard(n, r, w)]
        assert got == list(range(n))
        sizes = [len(shard.sector_shard(n, r, w)) for r in range(w)]
        assert max(sizes) - min(sizes) <= 1
        ev = sorted(e for r in range(w) for e in shard.event_shard(n, r, w))
        assert ev == list(range(n))
    with pytest.raises(ValueError):
        shard.sector_shard(36, 2, 2)


def test_slice_event_rebases(event):
    from paper_1712_09407_b200 import shard
    ev = event(3)
    R = ev.geometry.n_rows
    sub = shard.slice_event(ev.xyz, ev.row_start, R, range(5, 9))
    assert sub.row_start[0] == 0 and sub.row_start[-1] == len(sub.xyz)
    assert sub.first_cluster == ev.row_start[5 * R]
    assert np.array_equal(sub.xyz, ev.xyz.reshape(-1, 3)[ev.row_start[5 * R]:ev.row_start[9 * R]])
    assert np.array_equal(np.diff(sub.row_start.astype(np.int64)),
                          np.diff(ev.row_start[5 * R:9 * R + 1].astype(np.int64)))


def test_partition_is_refused_where_it_would_change_results():
    """the sector partition is exact for the plain sector tracker only.  With the steps that look
    into the neighbouring sector on (global tracking, track merging: PAPER.md L116-L136, L28) a rank must hold whole
    rings of 18 sectors — the kernels and the oracle skip those steps otherwise — and a rank without sectors cannot
    create a tracker: both are refused instead of returning a different result silently."""
    from paper_1712_09407_b200 import shard
    shard.check_partition(36, 8)                                    # plain tracker: any split of whole sectors
    shard.check_partition(36, 2, cross_sector=True)                 # two rings of 18
    shard.check_partition(36, 1, cross_sector=True)
    shard.check_partition(18, 1, cross_sector=True)
    for world in (3, 4, 8, 36):
        with pytest.raises(ValueError, match="whole rings of 18"):
            shard.check_partition(36, world, cross_sector=True)
    with pytest.raises(ValueError, match="whole rings of 18"):
        shard.check_partition(18, 2, cross_sector=True)
    with pytest.raises(ValueError, match="without work"):
        shard.check_partition(36, 37)
    with pytest.raises(ValueError, match="without work"):
        shard.check_partition(1, 2)
    with pytest.raises(ValueError, match="empty sector range"):
        shard.slice_event(np.zeros((0, 3), np.float32), np.zeros(160, np.uint32), 159, range(0, 0))
    # track_event_sharded applies the check before anything is tracked (world = 1 here: no process group)
    called = []
    with pytest.raises(ValueError, match="whole rings of 18"):
        shard.track_event_sharded(lambda sub: called.append(sub), np.zeros((0, 3), np.float32), np.zeros(5 * 159 + 1, np.uint32),
                                  5, 159, cross_sector=True)
    assert not called
    # the flag has no default: forgetting it is a TypeError, not a silent loss of prolongations and links
    with pytest.raises(TypeError, match="cross_sector"):
        shard.track_event_sharded(lambda sub: called.append(sub), np.zeros((0, 3), np.float32), np.zeros(5 * 159 + 1, np.uint32),
                                  5, 159)
    assert not called


def _worker_rings(rank: int, world: int, port: int, out_dir: str):
    if ROOT not in sys.path:
        sys.path.insert(0, ROOT)
    import torch.distributed as dist
    from dataclasses import replace
    from oracle import Oracle
    from paper_1712_09407_b200 import shard
    from tpcsynth import generate_event
    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ev = generate_event(3)
        n_ext = []

        def track(sub):
            geo = replace(ev.geometry, n_sectors=sub.n_sectors)
            o = Oracle.for_geometry(geo, global_tracking=1).run(np.ascontiguousarray(sub.xyz), sub.row_start)
            n_ext.append(len(o.global_ext))
            return o.tracks, o.track_cluster_ids

        tracks, ids = shard.track_event_sharded(track, ev.xyz, ev.row_start, 36, ev.geometry.n_rows, cross_sector=True)
        np.savez(os.path.join(out_dir, f"g{rank}.npz"), ids=ids, n_ext=np.array(n_ext))
    finally:
        dist.destroy_process_group()


def test_ring_partition_keeps_global_tracking_world2(tmp_path, oracle_run):
    """Two ranks, one ring of 18 sectors each, global tracking on: the tracks equal the whole event's, and the
    prolongations found by the two rings add up to the whole event's (the two z halves never exchange anything)."""
    import torch.multiprocessing as mp
    world, port = 2, _free_port()
    mp.start_processes(_worker_rings, args=(world, port, str(tmp_path)), nprocs=world, join=True, start_method="spawn")
    ev, o = oracle_run(3, global_tracking=1)
    n = 0
    for rank in range(world):
        z = np.load(tmp_path / f"g{rank}.npz")
        assert np.array_equal(z["ids"], o.track_cluster_ids)
        n += int(z["n_ext"][0])
    assert n == len(o.global_ext) > 100
