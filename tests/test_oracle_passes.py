"""Pins of the oracle's iterated construction passes (NEXT-4; G22d; cut `max_passes`, default 2).

PAPER.md L45: "These parameters are then used to extrapolate the trajectory to adjacent rows and search for more
clusters belonging to the tracklet.  When meeting a chi2-condition the clusters are collected to the tracklet and the
track parameters are refitted.  This is repeated until no more clusters are found."  G22 reads the repetition as the
per-row cycle of ONE upward and ONE downward pass; G22d is the literal reading: pass 3 goes up again from the refitted
state, pass 4 down, ... until a pass picks up nothing new (or `max_passes`).

Pins: a hand-worked event in which the third pass MUST pick up a cluster the first two cannot (both chi2 values are
recomputed here in float64 from the textbook formulas); clean tracks on which further passes change nothing; on the
dense and the pp-like configuration: a tracklet never loses a cluster, untouched tracklets are byte-identical to the
two-pass result, the passes reach a fixed point, the clusters of pass 3 are exactly those a whole-row scan of the
refitted two-pass tracklets finds (the plain definition), and they belong to the tracklet's particle.
"""
import numpy as np
import pytest

from oracle import Oracle
from tpcsynth import Geometry

GEO = Geometry(n_sectors=1)
R = GEO.n_rows
X = GEO.row_x.astype(np.float64)


def _line_event(rows, m=0.05, c=0.4, dy=None):
    xyz = np.zeros((len(rows), 3), np.float32)
    for i, k in enumerate(rows):
        xyz[i] = (X[k], m * X[k] + (dy or {}).get(k, 0.0), c * X[k])
    cnt = np.zeros(R, np.int64)
    cnt[list(rows)] = 1
    rs = np.zeros(R + 1, np.uint32)
    rs[1:] = np.cumsum(cnt)
    return xyz, rs


def test_third_pass_picks_up_what_the_first_two_cannot():
    """Straight track on rows 20..100, the cluster of row 21 displaced by +0.55 cm in y.
    Seeds: the triplet (20, 21, 22) has deviation^2 = 0.55^2 = 0.30 > nf_max_dev2 = 0.25, so cluster 21 gets no links;
    22 is the start (its down link to 21 is not reciprocal), chain 22..99.
    Pass 1 (up): 22 -> 100.  Pass 2 (down): refit 100 -> 22 with ~80 clusters, sigma_y of the prediction ~0.02 cm:
    on row 21 chi2 = 0.55^2 / (0.0144 + ~0.0003) ~ 20 > 10: a miss (below the seed, counted once); row 20 lies on the
    line and is picked up; rows 19..15 are empty: the pass ends.  Two passes: rows 20 and 22..100, 80 clusters.
    Pass 3 (up) starts on row 20 with the covariance reset (C_yy = err_y2, C_ss = 0.25): after the update with the hit
    of row 20 C_yy = err_y2 / 2, and one row (0.75 cm) higher the predicted variance is err_y2/2 + 0.75^2 * 0.25 (1 + m^2)^3
    + ... ~ 0.149, so chi2 = 0.55^2 / (0.149 + 0.0144) ~ 1.85 <= 10: the cluster of row 21 is picked up, and the
    refit goes on over rows 22..100 ungated.  Three passes: 81 clusters, state at the top row (x_ref = x[100]).
    Pass 4 (down) finds nothing new and is discarded."""
    rows = list(range(20, 101))
    xyz, rs = _line_event(rows, dy={21: 0.55})
    m, err2, c0s, c0k = 0.05, 0.0144, 0.25, 2.5e-3
    # the two chi2 values, float64, textbook: variance of the predicted y one row above a freshly reset state
    dx = X[21] - X[20]
    cos2 = 1.0 / (1.0 + m * m)
    h2 = dx / cos2 ** 1.5                                   # dy'/d(sin phi) at kappa = 0
    h4 = 0.5 * dx * dx / cos2 ** 1.5                        # dy'/d(kappa)
    var3 = err2 / 2 + h2 * h2 * c0s + h4 * h4 * c0k
    chi2_pass3 = 0.55 ** 2 / (var3 + err2)
    chi2_pass2_min = 0.55 ** 2 / (2 * err2)                 # even with sigma_pred^2 as large as err_y2 it would fail
    assert 1.5 < chi2_pass3 < 2.2 and chi2_pass2_min > 10.0
    r2 = Oracle.for_geometry(GEO).run(xyz, rs)
    assert len(r2.nhits) == 1 and (r2.first_row[0], r2.last_row[0], r2.nhits[0]) == (20, 100, 80)
    assert r2.hits[0, 21] == -1 and r2.n_passes[0] == 2 and r2.ref_row[0] == 20
    r3 = Oracle.for_geometry(GEO, max_passes=3).run(xyz, rs)
    assert (r3.first_row[0], r3.last_row[0], r3.nhits[0]) == (20, 100, 81)
    assert r3.hits[0, 21] == 1 and r3.n_passes[0] == 3 and r3.ref_row[0] == 100
    assert np.array_equal(np.delete(r3.hits[0], 21), np.delete(r2.hits[0], 21))
    assert r3.tracks[0]["x_ref"] == GEO.row_x[100] and r3.tracks[0]["n_clusters"] == 81
    # the state is the line at the top row (the displaced cluster, at the far end, tilts the fit by ~0.55 * 4 / 81 cm there)
    assert r3.tracks[0]["y"] == pytest.approx(m * X[100], abs=0.04)
    assert r3.tracks[0]["sinphi"] == pytest.approx(m / np.sqrt(1 + m * m), abs=5e-3)
    for mp in (4, 8):
        r = Oracle.for_geometry(GEO, max_passes=mp).run(xyz, rs)
        assert np.array_equal(r.hits, r3.hits) and r.n_passes[0] == 3
        assert np.array_equal(r.params, r3.params) and np.array_equal(r.chi2, r3.chi2)


@pytest.mark.parametrize("rows", [list(range(20, 101)), [k for k in range(20, 101) if not 60 <= k <= 63],
                                  [k for k in range(20, 101) if not 60 <= k <= 64]])
def test_further_passes_change_nothing_on_clean_tracks(rows):
    xyz, rs = _line_event(rows)
    ref = Oracle.for_geometry(GEO).run(xyz, rs)
    for mp in (3, 4, 8):
        r = Oracle.for_geometry(GEO, max_passes=mp).run(xyz, rs)
        for f in ("hits", "first_row", "last_row", "nhits", "params", "cov", "chi2", "ref_row"):
            assert np.array_equal(getattr(r, f), getattr(ref, f)), (mp, f)
        assert np.all(r.n_passes == 2)


@pytest.mark.parametrize("cfg", [2, 3])
def test_passes_only_add_clusters_and_reach_a_fixed_point(oracle_run, cfg):
    ev, r2 = oracle_run(cfg)
    prev, n_changed = r2, []
    for mp in range(3, 16):
        _, r = oracle_run(cfg, max_passes=mp)
        assert np.array_equal(r.start_cluster, r2.start_cluster)
        had = prev.hits >= 0
        assert np.array_equal(r.hits[had], prev.hits[had])                  # no cluster is lost or exchanged
        assert np.all(r.first_row <= prev.first_row) and np.all(r.last_row >= prev.last_row)
        assert np.array_equal((r.hits >= 0).sum(1)[r.nhits > 0], r.nhits[r.nhits > 0])
        same = r.n_passes == prev.n_passes
        for f in ("params", "cov", "chi2", "hits", "ref_row"):              # untouched tracklets: identical bytes
            assert np.array_equal(getattr(r, f)[same], getattr(prev, f)[same]), (mp, f)
        assert np.all(r.n_passes[~same] == mp) and np.all(r.n_passes <= mp)
        up = (r.n_passes & 1) == 1                                          # the state sits where the last kept pass ended
        assert np.array_equal(r.ref_row, np.where(up, r.last_row, r.first_row))
        n_changed.append(int((~same).sum()))
        prev = r
    # pass 3 does find clusters, and the passes die out — a fixed point (every pass starts from a reset covariance, so
    # the rows next to its starting end are searched with a wide gate and a row left empty there can be filled by a
    # noise cluster; each empty row can be filled once).  Seeds 2 / 3: 774, 127, 61, 27, 11, 7, 4, 2, 2, 1, 0 / 12, 1, 0.
    assert n_changed[0] > (100 if cfg == 2 else 2)
    assert n_changed[-1] == n_changed[-2] == 0 and sum(n_changed[1:]) < n_changed[0]
    if cfg == 3:
        assert n_changed[2:] == [0] * 11
    # invariants of the output still hold at the fixed point
    _, r = oracle_run(cfg, max_passes=15)
    assert len(np.unique(r.track_cluster_ids)) == len(r.track_cluster_ids) and np.all(r.tracks["n_clusters"] >= 30)


@pytest.mark.parametrize("cfg", [2, 3])
def test_third_pass_equals_whole_row_scan_of_the_two_pass_tracklets(oracle_run, cfg):
    """The plain definition of pass 3: starting from the two-pass result, every row without a hit is scanned WHOLE
    (no grid) for the best cluster within the chi2 cut (oracle diagnostic orc_third_pass_gain, which modifies nothing).
    The clusters max_passes = 3 adds are exactly those, tracklet by tracklet; passes the scan ends on a failure are
    discarded (G22d)."""
    ev, r2 = oracle_run(cfg)
    _, r3 = oracle_run(cfg, max_passes=3)
    o = Oracle.for_geometry(ev.geometry)
    o.run(ev.xyz, ev.row_start, fetch=False)
    g = o.third_pass_gain(ev.xyz, len(r2.nhits))
    failed, gain = (g >> 31) != 0, (g & np.uint32(0x7fffffff)).astype(np.int64)
    added = (r3.hits >= 0).sum(1) - (r2.hits >= 0).sum(1)
    assert np.array_equal(added, np.where(failed, 0, gain))
    assert added.sum() > (500 if cfg == 2 else 3) and failed.sum() < 0.01 * len(g)
    # the added clusters belong to the particle the tracklet follows (synthetic truth; sanity of the reading)
    good = tot = 0
    for t in np.nonzero(added)[0]:
        old = r2.hits[t][r2.hits[t] >= 0]
        new = r3.hits[t][(r3.hits[t] >= 0) & (r2.hits[t] < 0)]
        ids, cnt = np.unique(ev.truth_id[old], return_counts=True)
        if cnt.max() < 0.8 * len(old):
            continue
        tot += len(new)
        good += int((ev.truth_id[new] == ids[cnt.argmax()]).sum())
    if cfg == 2:
        print(f"pass 3, config 2: {tot} clusters added to truth-pure tracklets, {good} of the tracklet's particle")
        assert tot > 300 and good >= 0.5 * tot
