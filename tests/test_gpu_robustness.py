"""GPU edge cases and the boundary's error behaviour (include/tpcst.h), through the C ABI.

PAPER.md L142: the one production bug of the paper's tracker was a noisy sector exhausting GPU
memory; here a capacity overflow must come back as TPCST_ERR_CAPACITY with the context still usable.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _t():
    import paper_1712_09407_b200 as t
    return t


def _same(a, b):
    assert np.array_equal(a.tracks, b.tracks)
    assert np.array_equal(a.cluster_ids, b.cluster_ids)
    assert a.n_tracklets == b.n_tracklets


def _oracle_tracks(ev, **cuts):
    from oracle import Oracle
    return Oracle.for_geometry(ev.geometry, **cuts).run(ev.xyz, ev.row_start)


def _subset(ev, keep):
    """Event restricted to the clusters where keep is True (rows stay grouped)."""
    sr = np.repeat(np.arange(len(ev.row_start) - 1), np.diff(ev.row_start.astype(np.int64)))
    cnt = np.bincount(sr[keep], minlength=len(ev.row_start) - 1)
    rs = np.zeros(len(ev.row_start), np.uint32)
    rs[1:] = np.cumsum(cnt)
    return np.ascontiguousarray(ev.xyz[keep]), rs


def test_empty_event(event):
    t = _t()
    ev = event(1)
    with t.SectorTracker(ev.geometry, 1024, 1024) as trk:
        r = trk.track_event(np.zeros((0, 3), np.float32), np.zeros(ev.geometry.n_rows + 1, np.uint32))
        assert len(r.tracks) == 0 and len(r.cluster_ids) == 0 and r.n_tracklets == 0
        r = trk.track_event(ev.xyz[:1].copy(), np.r_[0, np.ones(ev.geometry.n_rows, np.uint32)].astype(np.uint32))
        assert len(r.tracks) == 0 and r.n_tracklets == 0


def test_empty_and_trackless_events_with_every_option(event):
    """No clusters, and clusters without a single track, through the optional stages (second selection round, global
    tracking, sort / refit / merge): empty results, no error, and the context tracks a real event afterwards."""
    t = _t()
    ev = event(3)
    R, S = ev.geometry.n_rows, ev.geometry.n_sectors
    opts = dict(select_rounds=2, global_tracking=1, merge_tracks=1)
    o = _oracle_tracks(ev, **opts)
    with t.SectorTracker(ev.geometry, ev.n_clusters, 8192, **opts) as trk:
        r = trk.track_event(np.zeros((0, 3), np.float32), np.zeros(S * R + 1, np.uint32))
        assert len(r.tracks) == 0 and len(r.merge) == 0 and len(r.global_ext) == 0
        keep = np.zeros(ev.n_clusters, bool)
        keep[::40] = True                                                 # far too sparse for a chain of three
        xyz, rs = _subset(ev, keep)
        r = trk.track_event(xyz, rs)
        assert len(r.tracks) == 0 and len(r.merge) == 0 and len(r.global_ext) == 0
        r = trk.track_event(ev.xyz, ev.row_start)
        assert np.array_equal(r.cluster_ids, o.track_cluster_ids) and len(r.merge) == len(o.tracks) > 1000
        assert np.array_equal(r.merge["next"], o.merge["next"]) and np.array_equal(r.global_cluster_ids, o.global_cluster_ids)


def test_ragged_rows_and_empty_sectors(event):
    """Rows emptied at random, whole sectors emptied: still identical to the oracle."""
    t = _t()
    ev = event(3)
    R = ev.geometry.n_rows
    rng = np.random.default_rng(7)
    sr = np.repeat(np.arange(len(ev.row_start) - 1), np.diff(ev.row_start.astype(np.int64)))
    dead_rows = rng.random(len(ev.row_start) - 1) < 0.03
    dead_sec = np.isin(sr // R, [0, 17, 35])
    keep = ~dead_rows[sr] & ~dead_sec
    xyz, rs = _subset(ev, keep)
    from oracle import Oracle
    o = Oracle.for_geometry(ev.geometry).run(xyz, rs)
    with t.SectorTracker(ev.geometry, len(xyz), 8192) as trk:
        r = trk.track_event(xyz, rs)
        assert np.array_equal(trk.debug_fetch(t.TPCST_DBG_LINKS).reshape(2, -1), np.stack([o.up, o.dn]))
    assert len(o.tracks) > 100
    assert np.array_equal(r.cluster_ids, o.track_cluster_ids)
    assert np.array_equal(r.tracks["seed_cluster"], o.tracks["seed_cluster"])


def test_range_check_free_sqrt_and_div_are_ieee():
    """construct_tracklets' sqrt / quotient sequences equal __fsqrt_rn / __fdiv_rn bit for bit: every fp32
    in [2^-8, 2^8) for the square root, 2^28 operand pairs for the quotient (include/tpcst.h)."""
    n, bad = _t().selftest_math(1 << 28)
    assert n == (0x43800000 - 0x3b800000) + (1 << 28) and bad == 0


def test_exact_ties_are_broken_by_original_index(event):
    """G8 / G20: every cluster stored twice (bit-identical coordinates, shuffled inside its row) makes
    every neighbour pair and every chi2 minimum an exact tie; the smaller original index must win
    on both sides, so links, tracklets and tracks still equal the oracle's."""
    t = _t()
    ev = event(1)
    rng = np.random.default_rng(11)
    rs0 = ev.row_start.astype(np.int64)
    parts, rs = [], np.zeros(len(rs0), np.uint32)
    for i in range(len(rs0) - 1):
        row = np.repeat(ev.xyz[rs0[i]:rs0[i + 1]], 2, axis=0)
        parts.append(row[rng.permutation(len(row))])
        rs[i + 1] = rs[i] + len(row)
    xyz = np.ascontiguousarray(np.concatenate(parts), dtype=np.float32)
    from oracle import Oracle
    o = Oracle.for_geometry(ev.geometry).run(xyz, rs)
    with t.SectorTracker(ev.geometry, len(xyz), 8192) as trk:
        r = trk.track_event(xyz, rs)
        assert np.array_equal(trk.debug_fetch(t.TPCST_DBG_LINKS_RAW).reshape(2, -1), np.stack([o.up_raw, o.dn_raw]))
        assert np.array_equal(trk.debug_fetch(t.TPCST_DBG_ROW_HITS).reshape(-1, ev.geometry.n_rows), o.hits)
    assert len(o.tracks) > 50
    assert np.array_equal(r.cluster_ids, o.track_cluster_ids)
    assert np.array_equal(r.tracks["seed_cluster"], o.tracks["seed_cluster"])


def test_out_of_range_and_nan_coordinates(event):
    """G4: coordinates outside the sector / z range are clamped into edge bins, NaN goes to bin 0 and
    never satisfies a predicate; the result still equals the oracle's."""
    t = _t()
    ev = event(1)
    xyz = ev.xyz.copy()
    rng = np.random.default_rng(3)
    i = rng.choice(len(xyz), 60, replace=False)
    xyz[i[:15], 1] = 1e4
    xyz[i[15:30], 1] = -1e4
    xyz[i[30:40], 2] = -5.0
    xyz[i[40:50], 2] = 1e6
    xyz[i[50:55], 1] = np.nan
    xyz[i[55:], 2] = np.nan
    from oracle import Oracle
    o = Oracle.for_geometry(ev.geometry).run(xyz, ev.row_start)
    with t.SectorTracker(ev.geometry, len(xyz), 4096) as trk:
        r = trk.track_event(xyz, ev.row_start)
        assert np.array_equal(trk.debug_fetch(t.TPCST_DBG_BIN_OF), o.bin_of)
        assert np.array_equal(trk.debug_fetch(t.TPCST_DBG_LINKS_RAW).reshape(2, -1), np.stack([o.up_raw, o.dn_raw]))
    assert np.array_equal(r.cluster_ids, o.track_cluster_ids)


def test_input_locations_and_determinism(event):
    """Pageable numpy, pinned torch and device torch inputs give byte-identical results, run after run."""
    import torch
    t = _t()
    ev = event(3)
    with t.SectorTracker(ev.geometry, ev.n_clusters, 8192) as trk:
        a = trk.track_event(ev.xyz, ev.row_start)
        px = torch.from_numpy(ev.xyz).pin_memory()
        pr = torch.from_numpy(ev.row_start.astype(np.int32)).pin_memory()
        b = trk.track_event(px, pr)
        dx, dr = px.cuda(), pr.cuda()
        torch.cuda.synchronize()
        c = trk.track_event(dx, dr)
        _same(a, b)
        _same(a, c)
        for _ in range(5):
            _same(a, trk.track_event(dx, dr))


def test_four_slot_stream(event):
    """BASELINE.json configs[4]: submit / wait with TPCST_N_SLOTS = 4 events in flight equals the synchronous calls AND the
    oracle, for nine distinct events from pinned host memory (every slot reused twice); slot state errors on every slot."""
    import torch
    t = _t()
    assert t.TPCST_N_SLOTS == 4
    evs = [event(3, seed) for seed in range(11, 20)]
    nmax = max(e.n_clusters for e in evs)
    with t.SectorTracker(evs[0].geometry, nmax, 8192) as trk:
        ref = [trk.track_event(e.xyz, e.row_start) for e in evs]
        for e, r in zip(evs, ref):
            o = _oracle_tracks(e)
            assert np.array_equal(r.cluster_ids, o.track_cluster_ids) and np.array_equal(r.tracks["seed_cluster"], o.tracks["seed_cluster"])
        pinned = [(torch.from_numpy(e.xyz).pin_memory(), torch.from_numpy(e.row_start.astype(np.int32)).pin_memory())
                  for e in evs]
        got = [None] * len(evs)
        D = t.TPCST_N_SLOTS
        for i in range(len(evs) + D - 1):
            if i < len(evs):
                trk.submit_event(*pinned[i], i % D)
            if i >= D - 1:
                got[i - (D - 1)] = trk.wait_event((i - (D - 1)) % D)
        for a, b in zip(ref, got):
            _same(a, b)
        # slot state errors, on every slot
        for s in range(D):
            with pytest.raises(t.TpcstError) as e:
                trk.wait_event(s)
            assert e.value.status == t.TPCST_ERR_STATE
        for s in range(D):
            trk.submit_event(*pinned[s], s)
        for s in range(D):
            with pytest.raises(t.TpcstError) as e:
                trk.submit_event(*pinned[(s + 1) % D], s)
            assert e.value.status == t.TPCST_ERR_STATE
        for s in reversed(range(D)):
            _same(ref[s], trk.wait_event(s))
        for bad in (-1, D):
            with pytest.raises(t.TpcstError) as e:
                trk.submit_event(*pinned[0], bad)
            assert e.value.status == t.TPCST_ERR_ARG


def test_device_row_start_is_validated_on_the_device(event):
    """TPCST_DEVICE input: the host cannot look at row_start, so bin_rows checks what tpcst_submit_event checks for host
    input (row_start[0] == 0, non-decreasing, row_start[last] == n_clusters) and the wait reports TPCST_ERR_ARG; nothing
    is read beyond the caller's n_clusters, and the context stays usable."""
    import torch
    t = _t()
    ev = event(3)
    good = _oracle_tracks(ev)
    xyz = torch.from_numpy(ev.xyz).cuda()
    rs_good = torch.from_numpy(ev.row_start.astype(np.int32)).cuda()
    torch.cuda.synchronize()
    with t.SectorTracker(ev.geometry, 2 * ev.n_clusters, 8192) as trk:
        for kind in ("last_too_large", "last_too_small", "first_not_zero", "not_monotone", "middle_beyond_n"):
            rs = ev.row_start.astype(np.int64).copy()
            if kind == "last_too_large":
                rs[-1] += 7                                   # within max_clusters, beyond the caller's xyz
            elif kind == "last_too_small":
                rs[-1] -= 1
            elif kind == "first_not_zero":
                rs[0] = 1
            elif kind == "not_monotone":
                rs[100] = rs[102] + 1
            else:
                rs[2000:2010] = ev.n_clusters + 5
            bad = torch.from_numpy(rs.astype(np.int32)).cuda()
            torch.cuda.synchronize()                              # inputs made on torch's default stream: the library orders
            with pytest.raises(t.TpcstError) as e:                # its kernels after cuda_stream_compute only (include/tpcst.h)
                trk.track_event(xyz, bad)
            assert e.value.status == t.TPCST_ERR_ARG, kind
            # after a failed event the debug accessors refuse to index with the caller's invalid row_start; the counters
            # (with the error bits) stay readable
            for what in (t.TPCST_DBG_LINKS, t.TPCST_DBG_STARTS, t.TPCST_DBG_ROW_HITS, t.TPCST_DBG_BIN_OF, t.TPCST_DBG_OWNERS):
                with pytest.raises(t.TpcstError) as e:
                    trk.debug_fetch(what)
                assert e.value.status == t.TPCST_ERR_STATE, (kind, what)
            assert trk.debug_fetch(t.TPCST_DBG_COUNTERS)[4] != 0, kind
            r = trk.track_event(xyz, rs_good)
            assert np.array_equal(r.cluster_ids, good.track_cluster_ids), kind
            assert trk.debug_fetch(t.TPCST_DBG_COUNTERS)[4] == 0 and len(trk.debug_fetch(t.TPCST_DBG_BIN_OF)) == ev.n_clusters


def test_calls_select_and_restore_the_device(event):
    """Every call selects the device that owns the workspace and restores the caller's current device (include/tpcst.h).
    With one GPU: the current device is unchanged by create / submit / wait / debug_fetch / destroy.  With two: a tracker
    on cuda:1 is created and driven while cuda:0 is current."""
    import torch
    t = _t()
    ev = event(1)
    ref = _oracle_tracks(ev)
    ndev = torch.cuda.device_count()
    target = ndev - 1
    torch.cuda.set_device(0)
    trk = t.SectorTracker(ev.geometry, ev.n_clusters, 1024, device=f"cuda:{target}")
    assert torch.cuda.current_device() == 0
    for s in range(t.TPCST_N_SLOTS):
        trk.submit_event(ev.xyz, ev.row_start, s)
        assert torch.cuda.current_device() == 0
    for s in range(t.TPCST_N_SLOTS):
        r = trk.wait_event(s)
        assert np.array_equal(r.cluster_ids, ref.track_cluster_ids)
    links = trk.debug_fetch(t.TPCST_DBG_LINKS).reshape(2, -1)
    assert np.array_equal(links[0], ref.up) and torch.cuda.current_device() == 0
    trk.close()
    assert torch.cuda.current_device() == 0


def test_capacity_overflow_is_an_error_not_a_hang(event):
    t = _t()
    ev = event(2)
    with t.SectorTracker(ev.geometry, ev.n_clusters, 200) as trk:       # 5820 tracklets do not fit in 200
        with pytest.raises(t.TpcstError) as e:
            trk.track_event(ev.xyz, ev.row_start)
        assert e.value.status == t.TPCST_ERR_CAPACITY
        small = event(1)                                                  # the context stays usable
        r = trk.track_event(small.xyz, small.row_start)
        assert len(r.tracks) == len(_oracle_tracks(small).tracks)
    with t.SectorTracker(ev.geometry, 1000, 100) as trk:                 # more clusters than the workspace holds
        with pytest.raises(t.TpcstError) as e:
            trk.track_event(ev.xyz, ev.row_start)
        assert e.value.status == t.TPCST_ERR_CAPACITY


def test_all_noise_sector(event):
    """A sector filled with uniform noise (the L142 scenario): bounded work, same answer as the oracle."""
    t = _t()
    ev = event(1)
    R = ev.geometry.n_rows
    rng = np.random.default_rng(5)
    per_row = 3000
    ymax = ev.geometry.row_x * ev.geometry.tan_half_angle
    xyz = np.empty((R * per_row, 3), np.float32)
    xyz[:, 0] = np.repeat(ev.geometry.row_x, per_row)
    xyz[:, 1] = rng.uniform(-1, 1, R * per_row) * np.repeat(ymax, per_row)
    xyz[:, 2] = rng.uniform(0, 250, R * per_row)
    rs = (np.arange(R + 1) * per_row).astype(np.uint32)
    o = _oracle_tracks(type("E", (), dict(geometry=ev.geometry, xyz=xyz, row_start=rs)))
    with t.SectorTracker(ev.geometry, len(xyz), len(xyz) // 4) as trk:
        r = trk.track_event(xyz, rs)
        assert np.array_equal(trk.debug_fetch(t.TPCST_DBG_LINKS).reshape(2, -1), np.stack([o.up, o.dn]))
        assert r.n_tracklets == len(o.nhits)
        assert np.array_equal(trk.debug_fetch(t.TPCST_DBG_ROW_HITS).reshape(-1, R), o.hits)
    assert np.array_equal(r.cluster_ids, o.track_cluster_ids)


def test_bad_arguments(event):
    t = _t()
    ev = event(1)
    R = ev.geometry.n_rows
    with t.SectorTracker(ev.geometry, ev.n_clusters, 1024) as trk:
        rs = ev.row_start.copy()
        rs[5] = rs[7] + 1                                                 # not monotone
        with pytest.raises(t.TpcstError) as e:
            trk.track_event(ev.xyz, rs)
        assert e.value.status == t.TPCST_ERR_ARG
        rs = ev.row_start.copy()
        rs[-1] -= 1                                                       # last offset != n_clusters
        with pytest.raises(t.TpcstError) as e:
            trk.track_event(ev.xyz, rs)
        assert e.value.status == t.TPCST_ERR_ARG
    with pytest.raises(t.TpcstError):
        t.SectorTracker(ev.geometry, ev.n_clusters, 1024, bin_y=0.0)
    with pytest.raises(t.TpcstError) as e:
        t.SectorTracker(ev.geometry, ev.n_clusters, 1024, bin_y=0.01, bin_z=0.01)   # grid too fine for a row table
    assert e.value.status in (t.TPCST_ERR_RANGE, t.TPCST_ERR_ARG)


def _noise_rows(geom, counts, seed):
    """Uniform-noise clusters, counts[k] on row k of one sector."""
    rng = np.random.default_rng(seed)
    counts = np.asarray(counts, np.int64)
    n = int(counts.sum())
    ymax = geom.row_x * geom.tan_half_angle
    xyz = np.empty((n, 3), np.float32)
    xyz[:, 0] = np.repeat(geom.row_x, counts)
    xyz[:, 1] = rng.uniform(-1, 1, n) * np.repeat(ymax, counts)
    xyz[:, 2] = rng.uniform(0, 250, n)
    rs = np.zeros(len(counts) + 1, np.uint32)
    rs[1:] = np.cumsum(counts)
    return xyz, rs


def test_maximum_sizes(event):
    """include/tpcst.h limits: 65535 clusters on a row is tracked like any other row, 65536 is
    TPCST_ERR_RANGE; so is a sector whose rows span 2^20 positions.  The context stays usable."""
    t = _t()
    geom = event(1).geometry
    R = geom.n_rows
    counts = np.zeros(R, np.int64)
    counts[40] = 65535
    counts[39] = counts[41] = 300
    xyz, rs = _noise_rows(geom, counts, 11)
    o = _oracle_tracks(type("E", (), dict(geometry=geom, xyz=xyz, row_start=rs)))
    with t.SectorTracker(geom, 70000, 4096) as trk:
        r = trk.track_event(xyz, rs)
        assert np.array_equal(trk.debug_fetch(t.TPCST_DBG_BIN_OF), o.bin_of)
        assert np.array_equal(trk.debug_fetch(t.TPCST_DBG_LINKS).reshape(2, -1), np.stack([o.up, o.dn]))
        assert r.n_tracklets == len(o.nhits)
        counts[40] = 65536
        xyz2, rs2 = _noise_rows(geom, counts, 12)
        with pytest.raises(t.TpcstError) as e:
            trk.track_event(xyz2, rs2)
        assert e.value.status == t.TPCST_ERR_RANGE
        assert r.n_tracklets == trk.track_event(xyz, rs).n_tracklets
    counts = np.zeros(R, np.int64)
    counts[:17] = 62000                                                   # 1.054 M clusters in one sector
    xyz, rs = _noise_rows(geom, counts, 13)
    with t.SectorTracker(geom, len(xyz), 4096) as trk:
        with pytest.raises(t.TpcstError) as e:
            trk.track_event(xyz, rs)
        assert e.value.status == t.TPCST_ERR_RANGE


def test_two_contexts_and_all_slots_interleaved(event):
    """Two trackers on one GPU (different geometries, different cuts), events submitted alternately on all four slots of
    both: every result equals the one the same tracker gives alone.  Nothing is shared between contexts, and the
    slots' streams do not disturb each other."""
    t = _t()
    a_ev, b_ev = event(2), event(3)
    with t.SectorTracker(a_ev.geometry, a_ev.n_clusters, a_ev.n_clusters // 8) as ta, \
            t.SectorTracker(b_ev.geometry, b_ev.n_clusters, 8192, select_mode=1, global_tracking=1, merge_tracks=1) as tb:
        ra, rb = ta.track_event(a_ev.xyz, a_ev.row_start), tb.track_event(b_ev.xyz, b_ev.row_start)
        for rnd in range(3):
            for s in (0, 1, 2, 3):
                ta.submit_event(a_ev.xyz, a_ev.row_start, s)
                tb.submit_event(b_ev.xyz, b_ev.row_start, s)
            for s in (3, 1, 0, 2):
                xa, xb = ta.wait_event(s), tb.wait_event(s)
                _same(xa, ra)
                _same(xb, rb)
                assert xb.merge.tobytes() == rb.merge.tobytes() and xb.global_ext.tobytes() == rb.global_ext.tobytes()
    assert len(ra.tracks) > 500 and len(rb.tracks) > 1000 and (rb.merge["next"] >= 0).sum() > 300


def test_graph_replay_equals_plain_launches(event):
    """include/tpcst.h, tpcst_set_graphs: the launch set of a slot is captured into a CUDA graph the second time the
    same input buffers come and replayed afterwards; a different buffer falls back to plain launches and is captured
    in turn.  Every result equals the one of a tracker with graphs off, byte for byte, for device and for host input."""
    import torch
    t = _t()
    a, b = event(3), event(3, 12)
    nmax = max(a.n_clusters, b.n_clusters)
    dev = {k: (torch.from_numpy(e.xyz).cuda(), torch.from_numpy(e.row_start.astype(np.int32)).cuda()) for k, e in (("a", a), ("b", b))}
    torch.cuda.synchronize()
    with t.SectorTracker(a.geometry, nmax, 8192) as plain:
        plain.set_graphs(False)
        ref = {k: plain.track_event(*dev[k]) for k in dev}
    with t.SectorTracker(a.geometry, nmax, 8192) as trk:
        for k in "aaabbbababbaa":                                     # plain, capture, replay, miss, capture, replay, ...
            _same(ref[k], trk.track_event(*dev[k]))
        for k, e in (("a", a), ("b", b), ("b", b), ("a", a), ("a", a)):   # host input: one graph whatever the event
            _same(ref[k], trk.track_event(e.xyz, e.row_start))
        for s in range(t.TPCST_N_SLOTS):                              # every slot has a graph of its own
            for _ in range(3):
                trk.submit_event(*dev["b"], s)
                _same(ref["b"], trk.wait_event(s))
        trk.set_profiling(1)                                          # no graph while profiling: per-kernel events are recorded
        _same(ref["a"], trk.track_event(*dev["a"]))
        assert trk.kernel_ms(0).sum() > 0
        trk.set_profiling(0)
        _same(ref["a"], trk.track_event(*dev["a"]))


def test_graph_cache_captures_each_input_once(event):
    """include/tpcst.h, tpcst_set_graphs: a slot remembers its last four input triples, captures a triple the second time
    it comes and replays it afterwards.  Alternating inputs (A,A,B,B,... and A,B,A,B,...) are captured once each and then
    only replayed; more distinct inputs than the table holds, taken in turn, are never captured.  TPCST_DBG_COUNTERS[5]
    and [6] count the slot's captures and replays.  Results are those of plain launches throughout."""
    import torch
    t = _t()
    evs = [event(1, seed) for seed in (None, 21, 22, 23, 24)]
    nmax = max(e.n_clusters for e in evs)
    dev = [(torch.from_numpy(e.xyz).cuda(), torch.from_numpy(e.row_start.astype(np.int32)).cuda()) for e in evs]
    torch.cuda.synchronize()
    with t.SectorTracker(evs[0].geometry, nmax, 4096) as plain:
        plain.set_graphs(False)
        ref = [plain.track_event(*d) for d in dev]
        assert list(plain.debug_fetch(t.TPCST_DBG_COUNTERS)[5:7]) == [0, 0]

    def counts(trk):
        c = trk.debug_fetch(t.TPCST_DBG_COUNTERS)
        return int(c[5]), int(c[6])

    for pattern, want in (("0011001100", (2, 6)),      # A A* B B* then replays only        (* = capture)
                          ("0101010101", (2, 6)),      # A B A* B* then replays only
                          ("0123012301", (4, 2)),      # four inputs fit the table: captured on their second visit
                          ("0123401234" * 2, (0, 0))): # five in turn never find themselves remembered: plain launches
        with t.SectorTracker(evs[0].geometry, nmax, 4096) as trk:
            for ch in pattern:
                _same(ref[int(ch)], trk.track_event(*dev[int(ch)]))
            assert counts(trk) == want, pattern


def test_max_passes_zero_means_the_default(event):
    """include/tpcst.h: a hand-filled tpcst_cuts that leaves the newest field, max_passes, at 0 gets the default (2)."""
    t = _t()
    ev = event(1)
    with t.SectorTracker(ev.geometry, ev.n_clusters, 4096) as trk:
        want = trk.track_event(ev.xyz, ev.row_start)
    with t.SectorTracker(ev.geometry, ev.n_clusters, 4096, max_passes=0) as trk:
        _same(want, trk.track_event(ev.xyz, ev.row_start))
    with pytest.raises(t.TpcstError) as e:
        t.SectorTracker(ev.geometry, ev.n_clusters, 4096, max_passes=1)
    assert e.value.status == t.TPCST_ERR_ARG


def test_selftest_random_access_runs_and_is_plausible():
    """include/tpcst.h, tpcst_selftest_random_access: the device's rate for random 4-byte gathers / atomic maxima over an L2-resident
    array.  A smoke test of the yardstick bench.py --l2-random prints: both times are positive, and 16 M accesses to a
    15 MB array take between 10 us (no GPU is that fast) and 10 ms (a rate below 1.6 G/s would mean it ran serially)."""
    t = _t()
    g, r = t.selftest_random_access(3_750_000, 16_000_000, reps=5)
    assert 0.01 < g < 10.0 and 0.01 < r < 10.0, (g, r)
    with pytest.raises(t.TpcstError) as e:
        t.selftest_random_access(0, 10)
    assert e.value.status == t.TPCST_ERR_ARG
