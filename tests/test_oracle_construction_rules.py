"""Hand-worked pins of the control flow of the oracle's tracklet construction (oracle/tpc_oracle.cpp,
construct_sector): the stop rules G21 / G23, the miss counter of the two passes (G22) and the truncation
rule G22c, on events small enough to work out on paper.

PAPER.md L45: "These parameters are then used to extrapolate the trajectory to adjacent rows and search for
more clusters belonging to the tracklet.  When meeting a chi2-condition the clusters are collected to the
tracklet and the track parameters are refitted.  This is repeated until no more clusters are found."
The paper gives no stop rule; DESIGN.md section 3 (step 5) reads it as: stop after more than `max_row_gap`
(4) consecutive rows without a cluster (G21), a prediction outside the sector counts as such a row (G23), in
the down pass only rows below the chain's first row are counted (G22.2), and the tracklet ends where the down
pass ended (G22c).

Every event here is ONE noise-free straight track (infinite momentum) in one sector: y = y0 + m x,
z = c x, one cluster per row on a chosen set of rows, so that the residuals are fp32 rounding (chi2 ~ 1e-8)
and every pickup decision is decided by the presence or absence of a cluster, never by the chi2 cut.  The
expected row ranges follow from the rules by counting rows; each case names the one-line mutation of the
oracle it is there to catch (each was applied by hand once and the case failed).

How the seeds come about (L40-L43, G9/G32): a cluster gets links only if it has a neighbour on BOTH adjacent
rows, so the first and the last cluster of a run of consecutive rows have none, the second cluster of a run
is a tracklet start, and a run of three rows forms no chain.
"""
import numpy as np
import pytest

from oracle import Oracle
from tpcsynth import Geometry

GEO = Geometry(n_sectors=1)
R = GEO.n_rows
X = GEO.row_x.astype(np.float64)


def line_event(rows, y0=0.0, m=0.05, c=0.4, dy=None):
    """One cluster on each row of `rows` at (x_k, y0 + m x_k (+ dy[k]), c x_k)."""
    rows = sorted(rows)
    xyz = np.zeros((len(rows), 3), np.float32)
    for i, k in enumerate(rows):
        xyz[i] = (X[k], y0 + m * X[k] + (dy or {}).get(k, 0.0), c * X[k])
    cnt = np.zeros(R, np.int64)
    cnt[rows] = 1
    rs = np.zeros(R + 1, np.uint32)
    rs[1:] = np.cumsum(cnt)
    return xyz, rs


def run(rows, **kw):
    cuts = kw.pop("cuts", {})
    xyz, rs = line_event(rows, **kw)
    r = Oracle.for_geometry(GEO, **cuts).run(xyz, rs)
    row_of = np.searchsorted(rs, np.arange(len(xyz)), side="right") - 1
    return r, row_of


def tracklet(r, row_of, start_row):
    """Index of the tracklet whose start cluster sits on `start_row`."""
    t = [i for i, c in enumerate(r.start_cluster) if row_of[c] == start_row]
    assert len(t) == 1, (start_row, [int(row_of[c]) for c in r.start_cluster])
    return t[0]


def hit_rows(r, t):
    return np.nonzero(r.hits[t] >= 0)[0].tolist()


def span(r, t):
    return int(r.first_row[t]), int(r.last_row[t]), int(r.nhits[t])


ALL = list(range(20, 101))                       # 81 rows


def without(rows, *gaps):
    drop = {k for a, b in gaps for k in range(a, b + 1)}
    return [k for k in rows if k not in drop]


def test_full_track_is_one_tracklet_over_all_rows():
    # run 20..100: start = row 21 (second cluster of the run), chain 21..99; the up pass picks up row 100,
    # finds rows 101..105 empty (5 > max_row_gap) and stops; the down pass refits 100..21 and picks up row 20,
    # then rows 19..15 are empty and it stops.
    r, row_of = run(ALL)
    assert len(r.nhits) == 1
    assert int(r.chain_len[0]) == 79
    assert span(r, 0) == (20, 100, 81)
    assert hit_rows(r, 0) == ALL


def test_gap_of_max_row_gap_rows_is_crossed_in_both_passes():
    # rows 60..63 empty (4 = max_row_gap).  Seeds: row 21 (run 20..59) and row 65 (run 64..100).
    # A (seed 21): chain to 58, picks up 59; misses 60, 61, 62, 63 -> miss = 4, NOT > 4; picks up 64 and goes on to 100.
    # B (seed 65): up pass to 100; down pass: 64 is below the seed row and is picked up; 63..60 -> 4 misses below,
    #   NOT > 4; 59 is picked up and it goes on down to 20.
    # Catches `++miss >= max_row_gap` (either pass) and an off-by-one in the gap cut.
    r, row_of = run(without(ALL, (60, 63)))
    assert len(r.nhits) == 2
    expect = without(ALL, (60, 63))
    for seed_row in (21, 65):
        t = tracklet(r, row_of, seed_row)
        assert span(r, t) == (20, 100, 77), seed_row
        assert hit_rows(r, t) == expect


def test_gap_of_more_than_max_row_gap_rows_ends_the_tracklet():
    # rows 60..64 empty (5).  A (seed 21): the fifth miss, on row 64, makes miss = 5 > 4: the up pass ends, the top
    #   hit row stays 59; the down pass refits 59..21, picks up 20, then 19..15 are empty.
    # B (seed 66, run 65..100): down pass picks up 65 below the seed, then 64..60 -> miss = 5 > 4 below: it ends,
    #   the last update was on row 65.
    # Catches a missing stop in either pass (the `below` misses DO stop the down pass).
    r, row_of = run(without(ALL, (60, 64)))
    assert len(r.nhits) == 2
    a, b = tracklet(r, row_of, 21), tracklet(r, row_of, 66)
    assert span(r, a) == (20, 59, 40) and hit_rows(r, a) == list(range(20, 60))
    assert span(r, b) == (65, 100, 36) and hit_rows(r, b) == list(range(65, 101))


def test_miss_counter_is_reset_by_a_pickup_and_counts_only_below_the_seed_in_the_down_pass():
    # rows 50..52 and 56..58 empty (3 + 3).  The run 53..55 has three rows and forms no chain.
    # Seeds: 21 (run 20..49) and 60 (run 59..100).
    # A (seed 21), up pass: picks 49; misses 50..52 (3); picks 53, 54, 55 (counter back to 0); misses 56..58 (3);
    #   picks 59 ... 100.  Without the reset the count would reach 6 > 4 on row 58 and the tracklet would end at 55.
    #   Down pass: rows 58..56 and 52..50 lie INSIDE the range (>= seed row 21): searched, empty, NOT counted.
    #   If in-range misses were counted (they are never reset inside the range) the pass would stop on row 50
    #   with 6 > 4 and the tracklet would start at row 53.
    # B (seed 60), down pass below the seed: picks 59; misses 58..56 (3); picks 55, 54, 53 (reset); misses 52..50 (3);
    #   picks 49 ... 20.  Without the reset below it would end on row 50 (first row 53).
    r, row_of = run(without(ALL, (50, 52), (56, 58)))
    assert len(r.nhits) == 2
    expect = without(ALL, (50, 52), (56, 58))
    for seed_row in (21, 60):
        t = tracklet(r, row_of, seed_row)
        assert span(r, t) == (20, 100, 75), seed_row
        assert hit_rows(r, t) == expect


def test_rows_beyond_the_last_or_first_row_end_the_pass():
    # a track reaching the outermost / innermost row: the loops end at R - 1 and at 0 (G21 "row index leaves [0, R-1]")
    rows = list(range(0, 31))
    r, row_of = run(rows)
    assert span(r, tracklet(r, row_of, 1)) == (0, 30, 31)
    rows = list(range(130, R))
    r, row_of = run(rows)
    assert span(r, tracklet(r, row_of, 131)) == (130, R - 1, R - 130)


def _edge_case():
    """A straight track leaving the sector through its side (y0 = -85.2, m = 0.85): clusters on the line on rows
    0..80 (far beyond the edge: out-of-sector coordinates are legal input, G4), except row 30, which ends the
    seed chain well inside the sector."""
    y0, m = -85.2, 0.85
    rows = without(list(range(0, 81)), (30, 30))
    ymax = X * float(GEO.tan_half_angle)
    y_line = y0 + m * X
    inside = np.abs(y_line) <= ymax + 1.0                      # G23 with edge_margin = 1 cm
    return y0, m, rows, y_line, ymax, inside


def test_prediction_outside_the_sector_is_a_miss_G23():
    # G23: a row whose predicted |y| exceeds ymax[k] + edge_margin is not searched — a miss, although a cluster
    # sits exactly on the prediction.  The seed chain is 1..28 (run 0..29); past it the up pass picks up row 29,
    # misses row 30 (empty), picks up 31, 32, ... while the line is inside the sector + 1 cm, and never again
    # after it: the top row follows from the geometry alone.
    y0, m, rows, y_line, ymax, inside = _edge_case()
    k_last = int(np.nonzero(inside)[0].max())
    assert inside[:k_last + 1].all() and not inside[k_last + 1:].any()          # one crossing, upwards
    margin = np.abs(np.abs(y_line) - (ymax + 1.0))
    assert margin.min() > 0.05 and 35 < k_last < 75                               # no row sits on the boundary
    r, row_of = run(rows, y0=y0, m=m)
    t = tracklet(r, row_of, 1)
    assert int(r.chain_len[t]) == 28
    first, last, n = span(r, t)
    assert (first, last) == (0, k_last)
    assert hit_rows(r, t) == without(list(range(0, k_last + 1)), (30, 30))
    # with a wider margin the next rows are picked up too: the margin is what decided
    wide = y_line[k_last + 3] - ymax[k_last + 3] + 0.01
    r2, row_of2 = run(rows, y0=y0, m=m, cuts=dict(edge_margin=float(wide)))
    assert span(r2, tracklet(r2, row_of2, 1))[1] == k_last + 3


def test_prediction_outside_the_sector_is_a_miss_in_the_down_pass_too():
    # the mirror image: y = 108.6 - 0.85 x enters the sector through its side around row 27 and is followed
    # DOWNWARDS.  Clusters on rows 0..80 except row 50; seeds: row 1 (run 0..49) and row 52 (run 51..80).
    # Seed 52: the up pass ends at row 80 (nothing above).  Down pass below the seed: picks up 51, misses 50
    # (empty), picks up 49, 48, ... as long as the prediction lies inside the sector + 1 cm; every row below is a
    # miss although a cluster sits on the line, and after five of them the pass ends.
    y0, m = 108.6, -0.85
    rows = without(list(range(0, 81)), (50, 50))
    ymax = X * float(GEO.tan_half_angle)
    y_line = y0 + m * X
    inside = np.abs(y_line) <= ymax + 1.0
    k_first = int(np.nonzero(inside[:81])[0].min())
    assert inside[k_first:81].all() and not inside[:k_first].any() and 10 < k_first < 45
    assert np.abs(np.abs(y_line[:81]) - (ymax[:81] + 1.0)).min() > 0.05
    r, row_of = run(rows, y0=y0, m=m)
    t = tracklet(r, row_of, 52)
    first, last, n = span(r, t)
    assert (first, last) == (k_first, 80)
    assert hit_rows(r, t) == without(list(range(k_first, 81)), (50, 50))


def _kf_two_steps_in_double(s, dx, r_top, err2=0.0144, c0s=0.25):
    """The first two updates of the down pass on a straight track, textbook Kalman filter in float64 restricted
    to (y, sin phi) (kappa plays no role in one step from a diagonal prior with C_y,kappa = 0 ... its gain on y
    enters only through h4 c0_kappa dx^2, kept below).  Returns sin phi after the second update.
    r_top = y(cluster on the top row) - y(state there)."""
    # update on the top row from the diagonal prior: K = 1/2 on y, nothing on sin phi
    y_off = 0.5 * r_top                                        # state is now y_line + y_off (if the state sat on the line: r_top/2)
    Cyy, Css = 0.5 * err2, c0s
    c = np.sqrt(1 - s * s)
    h2 = dx / c ** 3                                           # dy'/ds for kappa = 0 (G16: dx [2 cs + ss (r0 + r1)] / cs^2 at s' = s)
    Cyy1 = Cyy + h2 * h2 * Css + (0.5 * dx * dx / c ** 3) ** 2 * 2.5e-3
    Cys1 = h2 * Css + (0.5 * dx * dx / c ** 3) * dx * 2.5e-3
    return y_off, s + Cys1 / (Cyy1 + err2)                     # gain on sin phi, to be multiplied by the residual


def test_tracklet_ends_where_the_down_pass_ended_G22c():
    # G22c (truncation): if the down pass fails INSIDE the hit range, the tracklet is [row of the last down-pass
    # update, top hit row] and the hits of the up pass below it are dropped.
    # Track y = -85 + 0.85 x (sin phi = 0.6476) on rows 0..40, the top cluster (row 40) displaced by +0.34 cm:
    # the up pass accepts it (chi2 = 0.34^2 / ~0.0146 ~ 8 <= 10) as the last hit.  Down pass: the prior is reset
    # (C_ss = 0.25), the update with the displaced cluster moves y half way (+0.17); transported one row down the
    # residual of the (undisplaced) cluster on row 39 is -0.17 and the gain on sin phi is ~ -0.58: sin phi jumps
    # to ~0.745.  With max_sinphi = 0.70 that update fails (G17 "after the update, fail if |s| > max_sinphi"):
    # the pass ends with ONE update.  Expected: first_row = last_row = 40, nhits = 1, every other hit dropped.
    y0, m = -85.0, 0.85
    rows = list(range(0, 41))
    s = m / np.sqrt(1 + m * m)
    _, s_gain = _kf_two_steps_in_double(s, X[39] - X[40], 0.34)
    s_after = s + (s_gain - s) * (-0.17)
    assert 0.72 < s_after < 0.78 and s < 0.66                  # the hand calculation: 0.6476 -> ~0.745
    r, row_of = run(rows, y0=y0, m=m, dy={40: 0.34}, cuts=dict(max_sinphi=0.70))
    t = tracklet(r, row_of, 1)
    assert int(r.chain_len[t]) == 39                           # chain 1..39; row 40 is picked up by the up pass
    assert span(r, t) == (40, 40, 1)
    assert hit_rows(r, t) == [40]
    assert len(r.tracks) == 0
    # the same event with the default limit 0.95: nothing fails, the whole track is refitted
    r, row_of = run(rows, y0=y0, m=m, dy={40: 0.34})
    assert span(r, tracklet(r, row_of, 1)) == (0, 40, 41)
    # and without the displacement the tighter limit is harmless
    r, row_of = run(rows, y0=y0, m=m, cuts=dict(max_sinphi=0.70))
    assert span(r, tracklet(r, row_of, 1)) == (0, 40, 41)


def test_near_threshold_decisions_are_logged_G29():
    """G29 / L102: the oracle logs every pickup decision that hangs on less than 1e-4 (relative) — chi2 within 1e-4 of
    the cut, or two candidates whose chi2 differ by less than 1e-4 — so that a difference of a build with another
    rounding can be excused (or not).  Track on rows 20..100 plus a cluster on row 101 displaced by d: bisection on d
    finds the displacement at which the up pass stops picking it up; within 1e-6 of that point (both sides) the decision
    on row 101 is in the log, 2 % away from it (both sides) it is not.  A second cluster on row 101 at the mirrored
    position (equal chi2 to rounding) is logged as a near tie whatever d."""
    rows = list(range(20, 102))

    def run_d(d, twin=False):
        xyz, rs = line_event(rows, dy={101: d})
        if twin:                                   # a second cluster on row 101, mirrored about the track
            m, c = 0.05, 0.4
            extra = np.array([[X[101], m * X[101] - d, c * X[101]]], np.float32)
            xyz = np.concatenate([xyz, extra])
            rs = rs.copy(); rs[102:] += 1
        r = Oracle.for_geometry(GEO).run(xyz, rs)
        row_of = np.searchsorted(rs, np.arange(len(xyz)), side="right") - 1
        t = tracklet(r, row_of, 21)
        return r, t, bool(r.hits[t, 101] >= 0), any((a, b) == (t, 101) for a, b in r.near.tolist())

    lo, hi = 0.30, 0.50                            # picked up at 0.30 (chi2 ~ 6), not at 0.50 (chi2 ~ 17)
    assert run_d(lo)[2] and not run_d(hi)[2]
    for _ in range(40):
        mid = 0.5 * (lo + hi)
        if run_d(mid)[2]:
            lo = mid
        else:
            hi = mid
    assert hi - lo < 1e-9 and 0.36 < lo < 0.42
    for d, picked in ((lo * (1 - 1e-6), True), (hi * (1 + 1e-6), False)):
        _, _, got, near = run_d(d)
        assert got == picked and near, d
    for d, picked in ((lo * 0.98, True), (hi * 1.02, False)):
        _, _, got, near = run_d(d)
        assert got == picked and not near, d
    r, t, got, near = run_d(0.2, twin=True)
    assert got and near                            # a near tie of two clusters that both pass the cut
    r, t, got, near = run_d(0.2)
    assert got and not near                        # the same cluster alone: nothing hangs on 1e-4
