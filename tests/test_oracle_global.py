"""Pins of the oracle's global tracking (NEXT-2; section 5; G33-G36).

The paper gives two sentences and no formula, so the pins are: the rotation of a helix state into the
neighbouring sector's frame against the closed-form helix (and its Jacobian against finite
differences of the exact map, which also measures the two neglected couplings), the invariants the
readings promise, and what the step is for (L116: it recovers the short piece a track leaves in the
neighbouring sector) on synthetic truth.
"""
import numpy as np
import pytest

from oracle import Oracle
from tpcsynth import Geometry

DPHI = 2.0 * np.arctan(np.tan(np.deg2rad(10.0)).astype(np.float32).astype(np.float64))


@pytest.fixture(scope="module")
def orc():
    return Oracle.for_geometry(Geometry(n_sectors=36))


def _exact_rotation(x0, y, z, s, t, k, sg):
    """Exact map of a helix state on the plane x = x0 to the plane x' = const through the same point of the
    frame rotated by sg * DPHI (double precision, plain geometry)."""
    d = sg * DPHI
    xr = x0 * np.cos(d) + y * np.sin(d)
    yr = -x0 * np.sin(d) + y * np.cos(d)
    return xr, yr, z, np.sin(np.arcsin(s) - d), t, k


def _state_on_plane(x0, y, z, s, t, k, sg, xr_ref):
    """The rotated state moved along its helix to the plane x' = xr_ref (exact circle, double)."""
    xr, yr, zr, sr, tr, kr = _exact_rotation(x0, y, z, s, t, k, sg)
    dx = xr_ref - xr
    s1 = sr + kr * dx
    c0, c1 = np.sqrt(1 - sr * sr), np.sqrt(1 - s1 * s1)
    y1 = yr + dx * (sr + s1) / (c0 + c1)
    dl = (np.arcsin(s1) - np.arcsin(sr)) / kr if abs(kr) > 1e-12 else dx / c0
    return np.array([y1, zr + tr * dl, s1, tr, kr])


@pytest.mark.parametrize("sg", [1.0, -1.0])
def test_rotation_matches_exact_geometry(orc, sg):
    rng = np.random.default_rng(5)
    for _ in range(50):
        x0 = rng.uniform(85, 240)
        y, z = sg * x0 * np.tan(np.deg2rad(10)) * rng.uniform(0.8, 1.0), rng.uniform(0, 250)
        s, t, k = rng.uniform(-0.5, 0.5), rng.uniform(-1, 1), rng.uniform(-0.01, 0.01)
        st = np.zeros(20, np.float32)
        st[:5] = (y, z, s, t, k)
        out = orc.rotate(st, x0, sg)
        assert out is not None
        b, xr = out
        ex = _exact_rotation(x0, y, z, s, t, k, sg)
        assert abs(xr - ex[0]) < 1e-4 * abs(ex[0])
        assert np.allclose(b[:5], ex[1:], rtol=2e-6, atol=2e-5)
    # a point on the shared edge of the two sectors lies on the opposite edge of the neighbour
    st[:5] = (sg * 150.0 * np.tan(np.deg2rad(10)), 10.0, 0.1, 0.0, 0.001)
    b, xr = orc.rotate(st, 150.0, sg)
    assert abs(b[0] / xr + sg * np.tan(np.deg2rad(10))) < 1e-5


def test_rotation_jacobian_and_the_neglected_couplings(orc):
    """C' = J C J with J = diag(c/c', 1, c'/c, 1, 1) is the Jacobian of the exact map (state re-expressed on
    the plane x' = const through the nominal point) up to d s'/d y = -kappa sds and d z'/d y = -t sds / c'."""
    x0, y, z, s, t, k, sg = 100.0, 17.0, 50.0, 0.3, 0.7, 0.004, 1.0
    xr_ref = _exact_rotation(x0, y, z, s, t, k, sg)[0]
    p0 = np.array([y, z, s, t, k])
    F = np.zeros((5, 5))
    for j, h in enumerate([1e-4, 1e-4, 1e-6, 1e-6, 1e-8]):
        a, b = p0.copy(), p0.copy()
        a[j] += h
        b[j] -= h
        F[:, j] = (_state_on_plane(x0, *a, sg, xr_ref) - _state_on_plane(x0, *b, sg, xr_ref)) / (2 * h)
    c, sr = np.sqrt(1 - s * s), np.sin(np.arcsin(s) - DPHI)
    c1 = np.sqrt(1 - sr * sr)
    J = np.diag([c / c1, 1, c1 / c, 1, 1])
    extra = np.zeros((5, 5))
    extra[2, 0] = -k * np.sin(DPHI)
    extra[1, 0] = -t * np.sin(DPHI) / c1
    assert np.allclose(F, J + extra, atol=2e-5)
    # and the oracle applies exactly J C J
    rng = np.random.default_rng(1)
    A = rng.normal(size=(5, 5))
    Cm = (A @ A.T * 1e-3).astype(np.float32)
    st = np.zeros(20, np.float32)
    st[:5] = p0
    st[5:] = [Cm[i, j] for i in range(5) for j in range(i + 1)]
    b, _ = orc.rotate(st, x0, sg)
    want = J @ Cm.astype(np.float64) @ J
    got = np.zeros((5, 5))
    it = iter(b[5:])
    for i in range(5):
        for j in range(i + 1):
            got[i, j] = got[j, i] = next(it)
    assert np.allclose(got, want, rtol=1e-5, atol=1e-9)


def test_rotation_fails_beyond_max_sinphi(orc):
    st = np.zeros(20, np.float32)
    st[:5] = (17.0, 0.0, -0.93, 0.0, 0.0)          # phi - 20 deg leaves the band
    assert orc.rotate(st, 100.0, 1.0) is None


@pytest.mark.parametrize("cfg", [3])
def test_global_tracking_invariants_and_purpose(event, oracle_run, cfg):
    ev, r0 = oracle_run(cfg, n_threads=4)
    _, r = oracle_run(cfg, n_threads=4, global_tracking=1)
    R = ev.geometry.n_rows
    # the sector tracker's own results do not change
    assert np.array_equal(r.track_cluster_ids, r0.track_cluster_ids) and np.array_equal(r.tracks, r0.tracks)
    ge, ids = r.global_ext, r.global_cluster_ids
    assert len(ge) > 100 and ge["n_clusters"].sum() == len(ids)
    sr_of = np.repeat(np.arange(len(ev.row_start) - 1), np.diff(ev.row_start.astype(np.int64)))
    assert (np.diff(ge["track"].astype(np.int64) * 2 + ge["end"]) > 0).all()          # ordered by (track, end)
    pure = tot = 0
    for g in ge:
        tk = r.tracks[g["track"]]
        lst = ids[g["first_cluster"]: g["first_cluster"] + g["n_clusters"]]
        rows, secs = sr_of[lst] % R, sr_of[lst] // R
        assert (r.owner[lst] == 0).all()                                              # only free clusters (G35)
        half, j = tk["sector"] // 18, tk["sector"] % 18
        assert g["sector"] in (half * 18 + (j + 1) % 18, half * 18 + (j + 17) % 18) and (secs == g["sector"]).all()
        if g["end"] == 0:                                                             # inner end: rows descend
            assert tk["first_row"] <= 30 and (np.diff(rows) < 0).all() and rows[0] < tk["first_row"]
        else:
            assert tk["last_row"] >= R - 31 and (np.diff(rows) > 0).all() and rows[0] > tk["last_row"]
        assert g["row"] == rows[-1] and 1 <= g["n_clusters"] <= 30
        own = r.track_cluster_ids[tk["first_cluster"]: tk["first_cluster"] + tk["n_clusters"]]
        truth = np.bincount(ev.truth_id[own][ev.truth_id[own] != 0xFFFFFFFF]).argmax()
        pure += int((ev.truth_id[lst] == truth).sum())
        tot += len(lst)
    assert pure / tot > 0.98                                                          # picks up its own track
    # L116: what it is for — clusters of found tracks that sit in a neighbouring sector in a piece
    # too short for the sector tracker are now attached to a track
    assert len(np.unique(ids)) > 0.9 * len(ids)


# ------------------------------------------------------------------ hand-worked prolongations (G33, G35, G36)
def _crossing_track(n_rows_beyond, drop=(), sg=1, x_cross=None, drop_own=()):
    """One noise-free straight track in an 18-sector ring that runs through sector 4 and leaves it through the
    side towards sector 4 + sg, where it is followed up to the outer wall.  In the frame of sector 4 the line is
    y = sg * (ymax(x_c) + 0.7 (x - x_c)), z = 0.3 x: inclined by 35 deg, so it crosses the sector edge (inclined
    by 10 deg) at x = x_c, chosen just below the row from which `n_rows_beyond` rows are left.  Clusters: rows
    70..R-1 wherever the line is inside a sector (|y_local| <= ymax there), minus the rows in `drop`.
    Returns (geometry, xyz, row_start, rows of sector 4, rows of the neighbour)."""
    geo = Geometry(n_sectors=18)
    R, X, th = geo.n_rows, geo.row_x.astype(np.float64), float(geo.tan_half_angle)
    k_first_nb = R - n_rows_beyond
    xc = x_cross if x_cross is not None else X[k_first_nb] - 0.4
    own, nb = {}, {}
    for k in range(70, R):
        yl = sg * (xc * th + 0.7 * (X[k] - xc))
        if abs(yl) <= X[k] * th and k not in drop_own:
            own[k] = (X[k], yl, 0.3 * X[k])
    # the same line seen from the neighbour: a point (x, y) of sector 4's frame is (x cos d + y sin d, -x sin d + y cos d)
    # there, d = sg * DPHI; solve x' = X[k] along the line
    d = sg * DPHI
    y_at = lambda x: sg * (xc * th + 0.7 * (x - xc))
    for k in range(70, R):
        lo, hi = 50.0, 400.0
        for _ in range(80):                                        # bisection on x: x cos d + y(x) sin d is increasing
            mid = 0.5 * (lo + hi)
            if mid * np.cos(d) + y_at(mid) * np.sin(d) < X[k]:
                lo = mid
            else:
                hi = mid
        x = 0.5 * (lo + hi)
        yl = -x * np.sin(d) + y_at(x) * np.cos(d)
        if abs(yl) <= X[k] * th and k not in drop and k not in own and k not in drop_own:
            nb[k] = (X[k], yl, 0.3 * x)
    s_own, s_nb = 4, 4 + sg
    cnt = np.zeros(18 * R, np.int64)
    pts = []
    for s, d_ in sorted([(s_own, own), (s_nb, nb)]):
        for k in sorted(d_):
            cnt[s * R + k] = 1
            pts.append(d_[k])
    rs = np.zeros(18 * R + 1, np.uint32)
    rs[1:] = np.cumsum(cnt)
    return geo, np.array(pts, np.float32), rs, sorted(own), sorted(nb)


@pytest.mark.parametrize("sg", [1, -1])
def test_short_piece_in_the_neighbouring_sector_is_picked_up(sg):
    """L116: "segments shorter than 30 clusters in the neighbouring sector are lost" by the sector tracker; L130: the
    track "is extrapolated to the neighbouring sector" and the construction is continued there.  18 rows beyond the
    crossing: the sector track ends on the last row inside sector 4, the prolongation of its OUTER end collects
    exactly the 18 clusters of the neighbour, in row order, and ends on the outermost row."""
    geo, xyz, rs, own, nb = _crossing_track(18, sg=sg)
    R = geo.n_rows
    assert nb == list(range(R - 18, R)) and own == list(range(70, R - 18))
    r = Oracle.for_geometry(geo, global_tracking=1).run(xyz, rs)
    assert len(r.tracks) == 1 and r.tracks[0]["sector"] == 4 and r.tracks[0]["last_row"] == R - 19
    assert len(r.global_ext) == 1
    g = r.global_ext[0]
    assert (g["track"], g["end"], g["sector"], g["n_clusters"], g["row"]) == (0, 1, 4 + sg, 18, R - 1)
    ids = r.global_cluster_ids[g["first_cluster"]: g["first_cluster"] + 18]
    assert ids.tolist() == [int(rs[(4 + sg) * R + k]) for k in nb]
    # the state after the last pickup sits on the last cluster, with the line's direction in the neighbour's frame
    assert g["y"] == pytest.approx(xyz[ids[-1], 1], abs=2e-3) and g["z"] == pytest.approx(xyz[ids[-1], 2], abs=2e-3)
    assert g["sinphi"] == pytest.approx(sg * np.sin(np.arctan(0.7) - DPHI), abs=2e-3)
    assert g["chi2"] < 1e-2


def test_prolongation_gap_rule_and_free_clusters_only():
    # G35: the miss counter of the prolongation — a gap of max_row_gap (4) rows is crossed, one of 5 ends it
    geo, xyz, rs, own, nb = _crossing_track(18, drop=range(145, 149))
    R = geo.n_rows
    r = Oracle.for_geometry(geo, global_tracking=1).run(xyz, rs)
    g = r.global_ext[0]
    assert len(r.global_ext) == 1 and (g["n_clusters"], g["row"]) == (14, R - 1)
    geo, xyz, rs, own, nb = _crossing_track(18, drop=range(145, 150))
    r = Oracle.for_geometry(geo, global_tracking=1).run(xyz, rs)
    g = r.global_ext[0]
    assert len(r.global_ext) == 1 and (g["n_clusters"], g["row"]) == (4, 144)
    # two gaps of 3 rows with a pickup in between: the counter is reset by a pickup
    geo, xyz, rs, own, nb = _crossing_track(18, drop=list(range(144, 147)) + list(range(150, 153)))
    r = Oracle.for_geometry(geo, global_tracking=1).run(xyz, rs)
    g = r.global_ext[0]
    assert len(r.global_ext) == 1 and (g["n_clusters"], g["row"]) == (12, R - 1)
    # G33 "at the edge of a sector": the line is 0.58 / 1.36 / 2.15 / 2.93 / 3.72 cm inside the edge on the last
    # five rows before the crossing.  Without the last three rows the end is 2.93 cm from the edge (< gt_edge = 3):
    # it qualifies, three empty rows are crossed and the 18 clusters are picked up; without the last four it is
    # 3.72 cm away: no prolongation, although four empty rows would have been crossed (max_row_gap = 4)
    geo, xyz, rs, own, nb = _crossing_track(18, drop_own=range(R - 21, R - 18))
    r = Oracle.for_geometry(geo, global_tracking=1).run(xyz, rs)
    assert r.tracks[0]["last_row"] == R - 22 and len(r.global_ext) == 1 and r.global_ext[0]["n_clusters"] == 18
    geo, xyz, rs, own, nb = _crossing_track(18, drop_own=range(R - 22, R - 18))
    r = Oracle.for_geometry(geo, global_tracking=1).run(xyz, rs)
    assert r.tracks[0]["last_row"] == R - 23 and len(r.global_ext) == 0
    r = Oracle.for_geometry(geo, global_tracking=1, gt_edge=4.0).run(xyz, rs)
    assert len(r.global_ext) == 1 and r.global_ext[0]["n_clusters"] == 18
    # G33: more than gt_max_rows rows beyond the end -> no prolongation (here the piece is a sector track of its own)
    geo, xyz, rs, own, nb = _crossing_track(31)
    r = Oracle.for_geometry(geo, global_tracking=1).run(xyz, rs)
    assert len(r.tracks) == 2 and len(r.global_ext) == 0
    # ... and with the limit raised the ends do qualify, but the clusters are owned by the two sector tracks:
    # only FREE clusters are picked up (G35), so there is still nothing
    r = Oracle.for_geometry(geo, global_tracking=1, gt_max_rows=32).run(xyz, rs)
    assert len(r.tracks) == 2 and len(r.global_ext) == 0
    # an end far from the sector edge does not qualify (G33: within gt_edge = 3 cm): a radial track in mid-sector
    # that simply stops 18 rows below the outer wall
    geo = Geometry(n_sectors=18)
    X = geo.row_x.astype(np.float64)
    rows = np.arange(70, R - 18)
    xyz = np.stack([X[rows], 0.02 * X[rows], 0.3 * X[rows]], 1).astype(np.float32)
    cnt = np.zeros(18 * R, np.int64)
    cnt[4 * R + rows] = 1
    rs = np.zeros(18 * R + 1, np.uint32)
    rs[1:] = np.cumsum(cnt)
    r = Oracle.for_geometry(geo, global_tracking=1).run(xyz, rs)
    assert len(r.tracks) == 1 and r.tracks[0]["last_row"] == R - 19 and len(r.global_ext) == 0
