"""Pins of the oracle's steps 1-4 (binning, neighbours finder, evolution, chains).

The paper prints no worked example (PAPER.md has no numbers for L36-L46), so the pins are what the
method's definition and the mathematics fix: closed forms, invariants, brute-force enumeration
(the plain definition, MODE_TRIPLET) against the grid-accelerated search, grid independence, a
hand-worked 3-row example, and noise-free tracks whose links must follow truth.
"""
import numpy as np
import pytest

from oracle import MODE_GRID, MODE_ROWSCAN, MODE_TRIPLET, Oracle
from tpcsynth import NOISE_ID, Geometry

f32 = np.float32


def _rows_of(ev):
    R = ev.geometry.n_rows
    sr = np.searchsorted(ev.row_start.astype(np.int64), np.arange(ev.n_clusters), side="right") - 1
    return sr // R, sr % R


# ------------------------------------------------------------------ geometry tables / binning
def test_derived_tables_closed_form(event):
    ev = event(1)
    o = Oracle.for_geometry(ev.geometry)
    x = ev.geometry.row_x.astype(np.float64)
    ymax = o.array("tab_ymax")
    assert np.allclose(ymax, x * np.tan(np.deg2rad(10.0)), rtol=1e-6)
    # interpolation weights of the chord d-u at x[k]: w_up + w_dn = 1, and they reproduce x[k]
    wu, wd = o.array("tab_w_up").astype(np.float64), o.array("tab_w_dn").astype(np.float64)
    k = np.arange(1, 158)
    assert np.allclose(wu[k] + wd[k], 1.0, atol=2e-7)
    assert np.allclose(x[k + 1] * wu[k] + x[k - 1] * wd[k], x[k], rtol=1e-6)
    # uniform pitch -> 1/2; pitch change 0.75 -> 1.0 at row 62: w_up = 0.75/1.75
    assert wu[10] == pytest.approx(0.5, abs=1e-6) and wu[62] == pytest.approx(0.75 / 1.75, abs=1e-6)
    assert np.allclose(o.array("tab_ratio_up")[:-1], x[1:] / x[:-1], rtol=1e-6)
    assert np.allclose(o.array("tab_ratio_dn")[1:], x[:-1] / x[1:], rtol=1e-6)
    # windows: slope * pitch + const with the defaults 1.0/0.5 (y) and 0.5/0.5 (z)
    assert o.array("tab_wy_up")[0] == pytest.approx(1.25, abs=1e-5) and o.array("tab_wy_up")[150] == pytest.approx(2.0, abs=1e-5)
    assert o.array("tab_wz_dn")[100] == pytest.approx(1.0, abs=1e-5)
    ny = o.array("tab_ny")
    assert np.array_equal(ny, np.ceil(2 * ymax.astype(np.float64) / 1.0).astype(np.uint32) + 1)   # default bin_y = 1 cm
    assert o.nz == int(np.ceil(250.0 / 4.0)) + 1


def _tables_from_definition(geo, bin_y=1.0, wy=(1.0, 0.5), wz=(0.5, 0.5)):
    """DESIGN.md section 3 "Derived tables", written out: each entry is float32(float64 expression of the fp32 inputs).
    Independent of the oracle (numpy only); entries the definition leaves out (first / last row) are 0."""
    x = geo.row_x.astype(np.float32).astype(np.float64)
    R = len(x)
    tan = float(np.float32(geo.tan_half_angle))
    z = np.zeros(R, np.float64)
    t = {"tab_ymax": x * tan}
    up, dn, mid = np.arange(R - 1), np.arange(1, R), np.arange(1, R - 1)
    for name, (slope, const) in (("wy", wy), ("wz", wz)):
        a, b = z.copy(), z.copy()
        a[up] = float(np.float32(slope)) * (x[up + 1] - x[up]) + float(np.float32(const))
        b[dn] = float(np.float32(slope)) * (x[dn] - x[dn - 1]) + float(np.float32(const))
        t[f"tab_{name}_up"], t[f"tab_{name}_dn"] = a, b
    ru, rd, wu, wd = z.copy(), z.copy(), z.copy(), z.copy()
    ru[up] = x[up + 1] / x[up]
    rd[dn] = x[dn - 1] / x[dn]
    wu[mid] = (x[mid] - x[mid - 1]) / (x[mid + 1] - x[mid - 1])
    wd[mid] = (x[mid + 1] - x[mid]) / (x[mid + 1] - x[mid - 1])
    t.update(tab_ratio_up=ru, tab_ratio_dn=rd, tab_w_up=wu, tab_w_dn=wd)
    t = {k: v.astype(np.float32) for k, v in t.items()}
    t["tab_ny"] = (np.ceil(2.0 * t["tab_ymax"].astype(np.float64) / float(np.float32(bin_y))) + 1.0).astype(np.uint32)
    return t


def test_derived_tables_bit_for_bit(event):
    """Both sides depend on the derived tables bit for bit (they decide window membership and bins), so the oracle's are
    pinned at bit level to the definition, not to 1e-6: np.float32(float64 expression), DESIGN.md section 3."""
    for cfg in (1, 3):
        ev = event(cfg)
        o = Oracle.for_geometry(ev.geometry)
        want = _tables_from_definition(ev.geometry)
        for name, w in want.items():
            got = o.array(name)
            assert got.dtype == w.dtype and got.shape == w.shape, name
            assert np.array_equal(got.view(np.uint32), w.view(np.uint32)), name


@pytest.mark.parametrize("cfg", [1, 2, 3])
def test_binning_invariants(oracle_run, cfg):
    ev, r = oracle_run(cfg)
    S, R = ev.geometry.n_sectors, ev.geometry.n_rows
    sec, row = _rows_of(ev)
    o = Oracle.for_geometry(ev.geometry)
    ny = o.array("tab_ny").astype(np.int64)
    ymax = o.array("tab_ymax").astype(np.float64)
    off = r.bin_row_offset.astype(np.int64)
    n_row = np.diff(ev.row_start.astype(np.int64))
    for sr in range(S * R):
        cnt = r.bin_count[off[sr]:off[sr + 1]].astype(np.int64)
        st = r.bin_start[off[sr]:off[sr + 1]].astype(np.int64)
        assert cnt.sum() == n_row[sr]
        assert np.array_equal(st, np.concatenate([[0], np.cumsum(cnt)[:-1]]))
        g0, g1 = ev.row_start[sr], ev.row_start[sr + 1]
        assert np.array_equal(np.bincount(r.bin_of[g0:g1], minlength=cnt.size), cnt)
    # every cluster lies inside its bin's bounds (edge bins open-ended), recomputed in double
    b = r.bin_of.astype(np.int64)
    iy, iz = b % ny[row], b // ny[row]
    y, z = ev.xyz[:, 1].astype(np.float64), ev.xyz[:, 2].astype(np.float64)
    fy, fz = (y + ymax[row]) / 1.0, z / 4.0             # default bins: 1 cm x 4 cm
    tol = 1e-5
    lo_ok = (fy >= iy - tol) | (iy == 0)
    hi_ok = (fy < iy + 1 + tol) | (iy == ny[row] - 1)
    assert lo_ok.all() and hi_ok.all()
    assert (((fz >= iz - tol) | (iz == 0)) & ((fz < iz + 1 + tol) | (iz == o.nz - 1))).all()


def test_binning_clamps_outliers():
    geo = Geometry(n_sectors=1)
    R = geo.n_rows
    xyz = np.zeros((4, 3), f32)
    xyz[:, 0] = geo.row_x[0]
    xyz[:, 1] = [-1000.0, 1000.0, 0.0, np.nan]
    xyz[:, 2] = [-5.0, 1e9, 125.0, 10.0]
    rs = np.zeros(R + 1, np.uint32); rs[1:] = 4
    o = Oracle.for_geometry(geo)
    r = o.run(xyz, rs, stop_after=1)
    ny, nz = int(o.array("tab_ny")[0]), o.nz
    assert r.bin_of[0] == 0 and r.bin_of[1] == nz * ny - 1
    assert r.bin_of[3] % ny == 0                       # NaN y -> column 0


# ------------------------------------------------------------------ neighbours finder
def _links_equal(a, b):
    return np.array_equal(a.up_raw, b.up_raw) and np.array_equal(a.dn_raw, b.dn_raw)


def test_hand_worked_three_rows():
    # Three rows at x = 100, 101, 102 (uniform pitch -> w_up = w_dn = 1/2, ratios ~ 1).
    # Centre c = (0, 10).  Down: d0 = (-0.1, 9.9).  Up: u0 = (0.3, 10.1), u1 = (0.1, 10.1).
    # Pair (u1, d0): ey = 0.05 - 0.05 - 0 = 0, ez = 5.05 + 4.95 - 10 = 0  -> D = 0
    # Pair (u0, d0): ey = 0.15 - 0.05 = 0.1                                  -> D = 0.01
    geo = Geometry(n_sectors=1, n_rows=3, row_x=np.array([100, 101, 102], f32))
    xyz = np.array([[100, -0.1, 9.9], [101, 0.0, 10.0], [102, 0.3, 10.1], [102, 0.1, 10.1]], f32)
    rs = np.array([0, 1, 2, 4], np.uint32)
    r = Oracle.for_geometry(geo).run(xyz, rs)
    assert r.up_raw.tolist() == [-1, 3, -1, -1] and r.dn_raw.tolist() == [-1, 0, -1, -1]
    # one-sided match gives no link (G9 "best pair"): remove the down cluster
    r2 = Oracle.for_geometry(geo).run(xyz[1:], np.array([0, 0, 1, 3], np.uint32))
    assert (r2.up_raw == -1).all() and (r2.dn_raw == -1).all()
    # tie on D: duplicate u1 -> the smaller original index wins (G8)
    xyz3 = np.vstack([xyz, xyz[3:4]])
    r3 = Oracle.for_geometry(geo).run(xyz3, np.array([0, 1, 2, 5], np.uint32))
    assert r3.up_raw[1] == 3


def _numpy_bruteforce_links(xyz, row_start, tab, R):
    """Independent statement of G6-G8: every (u, d) pair, fp32 arithmetic, lexicographic argmin.  `tab`: the derived
    tables from _tables_from_definition (not the oracle's own)."""
    y, z = xyz[:, 1], xyz[:, 2]
    ru, rd = tab["tab_ratio_up"], tab["tab_ratio_dn"]
    wu, wd = tab["tab_w_up"], tab["tab_w_dn"]
    wyu, wyd, wzu, wzd = tab["tab_wy_up"], tab["tab_wy_dn"], tab["tab_wz_up"], tab["tab_wz_dn"]
    up = np.full(len(y), -1, np.int32); dn = np.full(len(y), -1, np.int32)
    for k in range(1, R - 1):
        U = np.arange(row_start[k + 1], row_start[k + 2]); Dn = np.arange(row_start[k - 1], row_start[k])
        if U.size == 0 or Dn.size == 0:
            continue
        for c in range(row_start[k], row_start[k + 1]):
            mu = (np.abs(y[U] - y[c] * ru[k]) <= wyu[k]) & (np.abs(z[U] - z[c] * ru[k]) <= wzu[k])
            md = (np.abs(y[Dn] - y[c] * rd[k]) <= wyd[k]) & (np.abs(z[Dn] - z[c] * rd[k]) <= wzd[k])
            uu, dd = U[mu], Dn[md]
            if uu.size == 0 or dd.size == 0:
                continue
            ey = (f32(y[uu] * wu[k])[:, None] + f32(y[dd] * wd[k])[None, :]) - y[c]
            ez = (f32(z[uu] * wu[k])[:, None] + f32(z[dd] * wd[k])[None, :]) - z[c]
            D = f32(ey * ey) + f32(ez * ez)
            assert D.dtype == np.float32
            ok = D <= f32(0.25)
            if not ok.any():
                continue
            Dm = np.where(ok, D, np.inf)
            iu, idn = np.nonzero(Dm == Dm.min())
            j = np.lexsort((dd[idn], uu[iu]))[0]
            up[c], dn[c] = uu[iu[j]], dd[idn[j]]
    return up, dn


def test_neighbours_equal_bruteforce_config1(event):
    ev = event(1)
    o = Oracle.for_geometry(ev.geometry)
    grid = o.run(ev.xyz, ev.row_start, mode=MODE_GRID, stop_after=3)
    scan = o.run(ev.xyz, ev.row_start, mode=MODE_ROWSCAN, stop_after=3)
    trip = o.run(ev.xyz, ev.row_start, mode=MODE_TRIPLET, stop_after=3)
    assert _links_equal(grid, trip) and _links_equal(scan, trip)
    up, dn = _numpy_bruteforce_links(ev.xyz, ev.row_start.astype(np.int64), _tables_from_definition(ev.geometry), ev.geometry.n_rows)
    assert np.array_equal(up, trip.up_raw) and np.array_equal(dn, trip.dn_raw)
    assert (trip.up_raw >= 0).sum() > 0.95 * ev.n_clusters


def test_neighbours_dense_random_with_ties():
    # 5 rows, dense uniform noise on a 0.25 cm lattice (many exactly-equal D and duplicated points)
    rng = np.random.default_rng(7)
    geo = Geometry(n_sectors=1, n_rows=5, row_x=np.array([100, 101, 102, 103, 104], f32))
    n = 220
    rows = np.repeat(np.arange(5), n)
    xyz = np.zeros((5 * n, 3), f32)
    xyz[:, 0] = geo.row_x[rows]
    xyz[:, 1] = np.round(rng.uniform(-6, 6, 5 * n) * 4) / 4
    xyz[:, 2] = np.round(rng.uniform(100, 108, 5 * n) * 4) / 4
    rs = (np.arange(6) * n).astype(np.uint32)
    o = Oracle.for_geometry(geo)
    trip = o.run(xyz, rs, mode=MODE_TRIPLET, stop_after=3)
    grid = o.run(xyz, rs, mode=MODE_GRID, stop_after=3)
    assert _links_equal(grid, trip)
    up, dn = _numpy_bruteforce_links(xyz, rs.astype(np.int64), _tables_from_definition(geo), 5)
    assert np.array_equal(up, trip.up_raw) and np.array_equal(dn, trip.dn_raw)
    assert (trip.up_raw >= 0).sum() > 300


@pytest.mark.parametrize("cfg", [2, 3])
def test_neighbours_grid_equals_rowscan(event, oracle_run, cfg):
    ev, grid = oracle_run(cfg)
    scan = Oracle.for_geometry(ev.geometry).run(ev.xyz, ev.row_start, mode=MODE_ROWSCAN, stop_after=3)
    assert _links_equal(grid, scan)


@pytest.mark.parametrize("by,bz", [(1.0, 1.0), (2.0, 4.0), (4.0, 2.0), (8.0, 8.0), (0.7, 13.0)])
def test_grid_independence(event, oracle_run, by, bz):
    ev, ref = oracle_run(2)
    r = Oracle.for_geometry(ev.geometry, bin_y=by, bin_z=bz).run(ev.xyz, ev.row_start)
    assert _links_equal(r, ref)
    assert np.array_equal(r.hits, ref.hits)                   # pickup is grid independent too (G20)
    assert np.array_equal(r.track_cluster_ids, ref.track_cluster_ids)


def test_straight_tracks_link_along_truth():
    # Noise-free straight lines y = a + b x, z = c + d x on the real (non-uniform pitch) rows: the
    # chord interpolation is exact, so D ~ 0 and every interior cluster links to its own track.
    rng = np.random.default_rng(3)
    geo = Geometry(n_sectors=1)
    R = geo.n_rows
    x = geo.row_x.astype(np.float64)
    nt = 12
    a = np.linspace(-10, 10, nt); b = rng.uniform(-0.05, 0.05, nt)
    c = np.linspace(20, 200, nt); d = rng.uniform(0.0, 0.2, nt)
    xyz = np.zeros((R * nt, 3), f32)
    xyz[:, 0] = np.repeat(geo.row_x, nt)
    xyz[:, 1] = (a[None, :] * x[:, None] / x[0] + b[None, :] * (x[:, None] - x[0])).ravel()
    xyz[:, 2] = (c[None, :] * x[:, None] / x[0] + d[None, :] * (x[:, None] - x[0])).ravel()
    rs = (np.arange(R + 1) * nt).astype(np.uint32)
    r = Oracle.for_geometry(geo).run(xyz, rs, stop_after=3)
    idx = np.arange(R * nt)
    interior = (idx >= nt) & (idx < (R - 1) * nt)
    assert np.array_equal(r.up_raw[interior], idx[interior] + nt)
    assert np.array_equal(r.dn_raw[interior], idx[interior] - nt)
    assert (r.up_raw[~interior] == -1).all()


def test_links_follow_truth_on_config1(oracle_run):
    ev, r = oracle_run(1)
    has = r.up >= 0
    same = ev.truth_id[has] == ev.truth_id[r.up[has]]
    assert same.mean() >= 0.99
    assert has.mean() > 0.9


# ------------------------------------------------------------------ evolution, starts, chains
@pytest.mark.parametrize("cfg", [1, 2, 3])
def test_evolution_reciprocal_and_recomputed(oracle_run, cfg):
    ev, r = oracle_run(cfg)
    idx = np.arange(ev.n_clusters, dtype=np.int32)
    up_e = np.where((r.up_raw >= 0) & (r.dn_raw[np.maximum(r.up_raw, 0)] == idx), r.up_raw, -1)
    dn_e = np.where((r.dn_raw >= 0) & (r.up_raw[np.maximum(r.dn_raw, 0)] == idx), r.dn_raw, -1)
    assert np.array_equal(up_e, r.up) and np.array_equal(dn_e, r.dn)
    has = r.up >= 0                                           # every stored link is reciprocal
    assert np.array_equal(r.dn[r.up[has]], idx[has])
    hasd = r.dn >= 0
    assert np.array_equal(r.up[r.dn[hasd]], idx[hasd])
    sec, row = _rows_of(ev)
    assert np.array_equal(row[r.up[has]], row[has] + 1) and np.array_equal(sec[r.up[has]], sec[has])


@pytest.mark.parametrize("cfg", [1, 2, 3])
def test_chain_invariants(oracle_run, cfg):
    ev, r = oracle_run(cfg)
    sec, row = _rows_of(ev)
    starts = r.start_cluster.astype(np.int64)
    assert np.all(np.diff(starts) > 0)                        # ids in (sector, row, index) order (G12)
    assert np.all((r.up[starts] >= 0) & (r.dn[starts] < 0))
    seen = np.zeros(ev.n_clusters, np.int32)
    for s, ln in zip(starts, r.chain_len):
        c, n = s, 0
        while c >= 0:
            seen[c] += 1; n += 1
            nxt = r.up[c]
            if nxt >= 0:
                assert row[nxt] == row[c] + 1
            c = nxt
        assert n == ln and ln >= 3
    assert seen.max() <= 1
    # every start with a long enough chain is listed
    cand = np.nonzero((r.up >= 0) & (r.dn < 0))[0]
    def clen(c):
        n = 0
        while c >= 0:
            n += 1; c = r.up[c]
        return n
    expect = [c for c in cand if clen(c) >= 3]
    assert np.array_equal(np.array(expect, np.int64), starts)


def test_no_links_touch_noise_much(oracle_run):
    ev, r = oracle_run(3)
    has = r.up >= 0
    noise_linked = (ev.truth_id[has] == NOISE_ID).mean()
    assert noise_linked < 0.01
