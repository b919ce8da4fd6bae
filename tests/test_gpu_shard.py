"""Multi-GPU readiness that one GPU can prove (sectors are tracked "individually",
L112: the CPU tracker is parallelised the same trivial way).

No multi-GPU node has been available, so `shard.track_event_sharded` has never run with the CUDA tracker across devices.
What one device can show is that its semantics hold for the product path: the event is cut into the two rings of 18
sectors (the finest split the cross-sector steps allow), each ring is tracked by a SectorTracker of its own as a rank
would, the shards are merged with the same `globalize` / `merge_shards` the collective path uses, and the result must be
the whole-event result of the GPU, byte for byte, and the oracle's.  Also with global tracking and track merging on,
whose prolongations and links stay inside a ring.
"""
from dataclasses import replace

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _t():
    import paper_1712_09407_b200 as t
    return t


def _track_rings(ev, **cuts):
    """The event as two 18-sector shards, each through its own SectorTracker -> merged (tracks, ids), per-ring results."""
    t = _t()
    from paper_1712_09407_b200 import shard
    shard.check_partition(ev.geometry.n_sectors, 2, cross_sector=True)
    parts, rings = [], []
    for rank in range(2):
        sub = shard.slice_event(ev.xyz, ev.row_start, ev.geometry.n_rows, shard.sector_shard(ev.geometry.n_sectors, rank, 2))
        geo = replace(ev.geometry, n_sectors=sub.n_sectors)
        n = max(len(sub.xyz), 1)
        with t.SectorTracker(geo, n, max(n // 8, 1024), **cuts) as trk:
            r = trk.track_event(np.ascontiguousarray(sub.xyz), sub.row_start)
        parts.append(shard.globalize(r.tracks, r.cluster_ids, sub))
        rings.append((sub, r))
    return shard.merge_shards(parts), rings


def _track_whole(ev, **cuts):
    t = _t()
    n = max(ev.n_clusters, 1)
    with t.SectorTracker(ev.geometry, n, max(n // 8, 1024), **cuts) as trk:
        return trk.track_event(ev.xyz, ev.row_start)


@pytest.mark.parametrize("cfg", [3, 4])
def test_two_rings_equal_the_whole_event(cfg, event, oracle_run):
    ev, o = oracle_run(cfg, n_threads=8)
    whole = _track_whole(ev)
    (tracks, ids), _ = _track_rings(ev)
    assert tracks.tobytes() == whole.tracks.tobytes()          # every field of every record, parameters included
    assert np.array_equal(ids, whole.cluster_ids)
    assert np.array_equal(ids, o.track_cluster_ids)
    for f in ("sector", "first_row", "last_row", "n_clusters", "first_cluster", "seed_cluster"):
        assert np.array_equal(tracks[f], o.tracks[f]), f


@pytest.mark.parametrize("cfg", [3, 4])
def test_two_rings_keep_the_cross_sector_steps(cfg, event, oracle_run):
    """global_tracking = 1 and merge_tracks = 1 look into the neighbouring sector of the same ring only: the rings'
    prolongations and links, moved back to the event's numbering, are the whole event's."""
    cuts = dict(global_tracking=1, merge_tracks=1)
    ev, o = oracle_run(cfg, n_threads=8, **cuts)
    whole = _track_whole(ev, **cuts)
    (tracks, ids), rings = _track_rings(ev, **cuts)
    assert tracks.tobytes() == whole.tracks.tobytes() and np.array_equal(ids, whole.cluster_ids)
    assert np.array_equal(ids, o.track_cluster_ids)
    # prolongations: per-ring records -> event numbering (track index, sector, picked-up cluster indices)
    gext, gids, merge, track0 = [], [], [], 0
    for sub, r in rings:
        g = r.global_ext.copy()
        g["track"] += np.uint32(track0)
        g["sector"] += np.uint32(sub.first_sector)
        g["first_cluster"] += np.uint32(sum(len(x) for x in gids))
        gext.append(g)
        gids.append(r.global_cluster_ids.astype(np.uint32) + np.uint32(sub.first_cluster))
        m = r.merge.copy()
        m["rank"] += np.uint32(track0)
        for f in ("next", "prev"):
            m[f] = np.where(m[f] >= 0, m[f] + track0, m[f])
        merge.append(m)
        track0 += len(r.tracks)
    gext, gids, merge = np.concatenate(gext), np.concatenate(gids), np.concatenate(merge)
    assert len(gext) == len(whole.global_ext) == len(o.global_ext) > 100
    assert gext.tobytes() == whole.global_ext.tobytes()
    assert np.array_equal(gids, whole.global_cluster_ids)
    assert len(merge) == len(whole.merge)
    assert merge.tobytes() == whole.merge.tobytes()
    assert (whole.merge["next"] >= 0).sum() > 50                 # the links are there to be kept
