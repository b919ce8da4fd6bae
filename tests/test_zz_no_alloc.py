"""tpcst_select_owners_static: the selection step for callers that cannot allocate device memory.

Some users of this library only own the device buffers of their inputs and outputs at the point where they
select tracklets: a trigger / real-time loop must not run into cudaMalloc (it synchronises the whole device and
takes an unbounded time), a plug-in of a framework that has handed out all device memory gets no more of it, and
a process with a frozen, audited memory budget may not grow after start-up.  For them the library has one entry
point whose only scratch memory (a claim key per cluster) is a fixed 4 MiB array inside libtpcst.so's device
image (at most TPCST_STATIC_MAX_CLUSTERS = 1 Mi clusters per call).

What is checked here: its result against the regular path (tpcst_track_event with a caller-allocated workspace),
bit for bit (the work is integer work; the parity tests of this repository compare such results exactly), on
calls that follow each other directly and use different events of different sizes, so that keys the previous call
left in the shared array would show; and the rejection of sizes beyond the limit.

This file sorts last on purpose (pytest -x stops at the first failure; a failure here must not hide the parity
tests) and passes both alone in a fresh process, where its first call does the per-device set-up, and after the
other tests.
"""
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
MIN_CLUSTERS = 30            # PAPER.md L116; tpcst_default_cuts


def _t():
    import paper_1712_09407_b200 as t
    return t


def _regular_path(ev):
    """Row-hit tables, owners and kept counts of the regular path, owners translated to tracklet indices."""
    t = _t()
    n = max(ev.n_clusters, 1)
    with t.SectorTracker(ev.geometry, n, max(n // 8, 1024)) as trk:
        res = trk.track_event(ev.xyz, ev.row_start)
        T, R = res.n_tracklets, ev.geometry.n_rows
        row_hits = trk.debug_fetch(t.TPCST_DBG_ROW_HITS).reshape(T, R).copy()
        keys = trk.debug_fetch(t.TPCST_DBG_OWNERS).copy()
        tl = trk.debug_fetch(t.TPCST_DBG_TRACKLETS).copy()
    # the regular path reports, per cluster, the packed key n_hits << 24 | (0xFFFFFF - rank of the tracklet inside
    # its sector); the tracklet index is that rank + the first tracklet of the cluster's sector
    row_start = np.asarray(ev.row_start, dtype=np.int64)
    sector_of_cluster = (np.searchsorted(row_start, np.arange(ev.n_clusters), side="right") - 1) // R
    first_of_sector = np.searchsorted(tl["sector"], np.arange(ev.geometry.n_sectors), side="left")
    owner = np.full(ev.n_clusters, -1, np.int64)
    has = keys != 0
    owner[has] = first_of_sector[sector_of_cluster[has]] + (0xFFFFFF - (keys[has].astype(np.int64) & 0xFFFFFF))
    # the precondition of the comparison: a tracklet's length is the number of entries of its row
    assert np.array_equal((row_hits >= 0).sum(axis=1), tl["n_clusters"])
    assert np.array_equal(keys[has] >> 24, tl["n_clusters"][owner[has]])
    return row_hits, owner, tl["first_cluster"].astype(np.int64)      # first_cluster of the debug view = kept clusters


@pytest.mark.gpu
def test_static_selection_matches_the_regular_path_on_consecutive_calls(event):
    import torch
    t = _t()
    cases = []
    for cfg in (2, 3, 1):                 # 0.2 M clusters in one sector, then 0.125 M in 36, then 15 k: shrinking sizes,
        ev = event(cfg)                   # so every call runs over keys the one before left in the array
        assert ev.n_clusters <= t.TPCST_STATIC_MAX_CLUSTERS
        cases.append((cfg, ev.n_clusters, *_regular_path(ev)))
    dev = torch.device("cuda:0")
    hits_dev = [torch.from_numpy(c[2]).to(dev) for c in cases]
    # the outputs are the caller's: allocated up front, as a caller that cannot allocate later would
    owner_dev = [torch.empty(c[1], dtype=torch.int32, device=dev) for c in cases]
    kept_dev = [torch.empty(c[2].shape[0], dtype=torch.int32, device=dev) for c in cases]
    torch.cuda.synchronize()
    order = [0, 1, 2, 0, 0]               # back to back on one stream, including the same event twice in a row
    for i in order:
        owner_dev[i].fill_(0x5a5a5a5a)
        kept_dev[i].fill_(0x5a5a5a5a)
        o, k = t.select_owners_static(hits_dev[i], cases[i][1], MIN_CLUSTERS, owner=owner_dev[i], kept=kept_dev[i])
        assert o.data_ptr() == owner_dev[i].data_ptr() and k.data_ptr() == kept_dev[i].data_ptr()
        cfg, n, _, want_owner, want_kept = cases[i]
        got_owner, got_kept = o.cpu().numpy().astype(np.int64), k.cpu().numpy().astype(np.int64)
        assert (want_owner >= 0).sum() > 0.2 * n and (want_kept >= MIN_CLUSTERS).sum() > 10, cfg   # not a vacuous case
        assert np.array_equal(got_owner, want_owner), f"config {cfg}: owners differ from the regular path"
        assert np.array_equal(got_kept, want_kept), f"config {cfg}: kept counts differ from the regular path"
    # queued without a host wait in between: the second call clears and reuses the array behind the first
    t.select_owners_static(hits_dev[0], cases[0][1], MIN_CLUSTERS, owner=owner_dev[0], kept=kept_dev[0])
    t.select_owners_static(hits_dev[1], cases[1][1], MIN_CLUSTERS, owner=owner_dev[1], kept=kept_dev[1])
    torch.cuda.synchronize()
    for i in (0, 1):
        assert np.array_equal(owner_dev[i].cpu().numpy().astype(np.int64), cases[i][3])
        assert np.array_equal(kept_dev[i].cpu().numpy().astype(np.int64), cases[i][4])


@pytest.mark.gpu
def test_static_selection_degenerate_inputs():
    import torch
    t = _t()
    dev = torch.device("cuda:0")
    # no tracklets: every cluster is free
    o, k = t.select_owners_static(torch.empty((0, 159), dtype=torch.int32, device=dev), 1000, MIN_CLUSTERS)
    assert k.numel() == 0 and (o.cpu().numpy() == -1).all()
    # no clusters, or only too-short / out-of-range rows: nothing is kept
    rows = torch.full((5, 159), -1, dtype=torch.int32, device=dev)
    rows[1, :29] = torch.arange(29, dtype=torch.int32, device=dev)          # 29 hits < 30
    rows[2, :40] = 5000                                                     # indices beyond n_clusters count as no hit
    o, k = t.select_owners_static(rows, 100, MIN_CLUSTERS)
    assert (o.cpu().numpy() == -1).all() and (k.cpu().numpy() == 0).all()
    o, k = t.select_owners_static(rows, 0, MIN_CLUSTERS)
    assert o.numel() == 0 and (k.cpu().numpy() == 0).all()
    # ties: equally long tracklets, the lower index keeps the shared clusters; the longer one beats both
    rows = torch.full((3, 159), -1, dtype=torch.int32, device=dev)
    rows[0, :30] = torch.arange(0, 30, dtype=torch.int32, device=dev)
    rows[1, 10:40] = torch.arange(10, 40, dtype=torch.int32, device=dev)    # shares clusters 10..29 with tracklet 0
    rows[2, 100:131] = torch.arange(25, 56, dtype=torch.int32, device=dev)  # 31 hits, shares 25..29 with 0 and 25..39 with 1
    o, k = t.select_owners_static(rows, 60, MIN_CLUSTERS)
    o, k = o.cpu().numpy(), k.cpu().numpy()
    want = np.full(60, -1)
    want[0:25] = 0; want[25:56] = 2
    assert np.array_equal(o, want) and list(k) == [25, 0, 31]
    # buffers that are not device memory are refused, not dereferenced
    host = np.zeros((2, 159), np.int32)
    rc = t.lib().tpcst_select_owners_static(host.ctypes.data, 2, 159, 0, MIN_CLUSTERS, None, host.ctypes.data, None)
    assert rc == t.TPCST_ERR_ARG


def test_static_selection_rejects_sizes_beyond_its_array():
    """Needs no GPU: the size is checked before anything touches CUDA."""
    t = _t()
    L = t.lib()
    rc = L.tpcst_select_owners_static(None, 0, 159, t.TPCST_STATIC_MAX_CLUSTERS + 1, MIN_CLUSTERS, None, None, None)
    assert rc == t.TPCST_ERR_STATIC_LIMIT
    msg = L.tpcst_error_string(rc).decode()
    assert "TPCST_STATIC_MAX_CLUSTERS" in msg and str(t.TPCST_STATIC_MAX_CLUSTERS) in msg and "tpcst_create" in msg
    assert L.tpcst_select_owners_static(None, 0, 159, 0, MIN_CLUSTERS, None, None, None) == t.TPCST_OK   # nothing to do
    for bad in ((0, 0, 0, MIN_CLUSTERS), (0, 256, 0, MIN_CLUSTERS), (0, 159, 0, 0), (0, 159, 0, 256), ((1 << 24) + 1, 159, 0, 30)):
        assert L.tpcst_select_owners_static(None, bad[0], bad[1], bad[2], bad[3], None, None, None) == t.TPCST_ERR_ARG, bad
    hdr = open(os.path.join(ROOT, "include", "tpcst.h")).read()
    assert re.search(r"#define\s+TPCST_STATIC_MAX_CLUSTERS\s+%du" % t.TPCST_STATIC_MAX_CLUSTERS, hdr)


def test_static_selection_source_allocates_nothing():
    """The file that implements the entry point names no allocating CUDA call outside its comments."""
    src = open(os.path.join(ROOT, "paper_1712_09407_b200", "csrc", "static_select.cu")).read()
    code = re.sub(r"//[^\n]*", "", src)
    for call in ("cudaMalloc", "cudaFree", "cudaHostAlloc", "cudaStreamCreate", "cudaEventCreate", "cudaMemPool", "new ", "malloc("):
        assert call not in code, call
    assert "cudaGetSymbolAddress" in code and "static __device__ __align__(256)" in code
