"""Pins of the oracle's steps 5-7 (Kalman construction, selection, output).

Closed forms (analytic helix transport, finite-difference Jacobian in double), the textbook
Kalman update on random SPD covariances, noise-free helices whose parameters must be recovered,
pull / chi2 statistics on smeared tracks, the sequential greedy selection reference, and the
invariants north_star names (no cluster in two tracks, length >= min_clusters).
"""
from dataclasses import replace

import numpy as np
import pytest

from oracle import MODE_GRID, MODE_ROWSCAN, Oracle
from tpcsynth import CONFIGS, KB, Geometry, generate_event

f32 = np.float32
IDX = [(i, j) for i in range(5) for j in range(i + 1)]        # lower-triangle packing order


def pack(p, Cm):
    return np.concatenate([np.asarray(p, f32), np.array([Cm[i, j] for i, j in IDX], f32)])


def unpack(v):
    Cm = np.zeros((5, 5))
    for n, (i, j) in enumerate(IDX):
        Cm[i, j] = Cm[j, i] = v[5 + n]
    return v[:5].astype(np.float64), Cm


def helix_transport(p, dx):
    """Exact circle/helix transport of (y, z, sin phi, dz/ds, kappa) by dx, float64."""
    y, z, s, t, k = p
    s1 = s + k * dx
    ph0, ph1 = np.arcsin(s), np.arcsin(s1)
    if abs(k) > 1e-12:
        y1 = y + (np.cos(ph0) - np.cos(ph1)) / k
        path = (ph1 - ph0) / k
    else:
        y1 = y + dx * np.tan(ph0)
        path = dx / np.cos(ph0)
    return np.array([y1, z + t * path, s1, t, k])


@pytest.fixture(scope="module")
def orc():
    return Oracle.for_geometry(Geometry(n_sectors=1))


# ------------------------------------------------------------------ transport (G16)
@pytest.mark.parametrize("dx", [0.75, 1.5, -1.0, 7.5, -12.0])
def test_transport_matches_analytic_helix(orc, dx):
    rng = np.random.default_rng(11)
    for _ in range(50):
        pt = rng.uniform(0.15, 5.0)
        k = rng.choice([-1, 1]) * KB * 0.5 / pt
        p = np.array([rng.uniform(-20, 20), rng.uniform(0, 250), rng.uniform(-0.6, 0.6), rng.uniform(-1, 1), k])
        out = orc.transport(pack(p, np.eye(5) * 1e-3), dx)
        ref = helix_transport(p, dx)
        assert out is not None
        assert np.allclose(out[:5], ref, rtol=2e-6, atol=2e-5)


def test_transport_straight_line_limit(orc):
    p = np.array([1.0, 50.0, 0.3, 0.5, 0.0])
    out = orc.transport(pack(p, np.eye(5) * 1e-3), 2.0)
    tanphi = 0.3 / np.sqrt(1 - 0.09)
    assert out[0] == pytest.approx(1.0 + 2.0 * tanphi, rel=1e-6)
    assert out[1] == pytest.approx(50.0 + 0.5 * 2.0 / np.sqrt(1 - 0.09), rel=1e-6)
    assert out[2] == pytest.approx(0.3) and out[4] == 0.0


def test_transport_fails_beyond_max_sinphi(orc):
    p = np.array([0.0, 10.0, 0.9, 0.1, 0.01])
    assert orc.transport(pack(p, np.eye(5)), 10.0) is None          # s' = 1.0 > 0.95
    assert orc.transport(pack(p, np.eye(5)), 4.0) is not None       # s' = 0.94


def test_covariance_transport_equals_F_C_Ft(orc):
    rng = np.random.default_rng(5)
    for _ in range(20):
        k = rng.choice([-1, 1]) * KB * 0.5 / rng.uniform(0.2, 3.0)
        p = np.array([rng.uniform(-10, 10), rng.uniform(0, 200), rng.uniform(-0.5, 0.5), rng.uniform(-1, 1), k])
        A = rng.normal(size=(5, 5)) * np.array([0.1, 0.1, 0.02, 0.03, 1e-4])[:, None]
        Cm = A @ A.T + np.diag([1e-3, 1e-3, 1e-5, 1e-5, 1e-9])
        dx, nrows = rng.choice([0.75, 1.0, 1.5, -1.5, 4.5]), 3.0
        F = np.zeros((5, 5))
        for j in range(5):                                          # central differences in double
            h = 1e-6 * max(1.0, abs(p[j])) if j < 4 else 1e-9
            pp, pm = p.copy(), p.copy()
            pp[j] += h; pm[j] -= h
            F[:, j] = (helix_transport(pp, dx) - helix_transport(pm, dx)) / (2 * h)
        F[1, 2] = 0.0; F[1, 4] = 0.0                                # G16: dz'/ds and dz'/dk are neglected
        Q = np.diag([0, 0, 1e-6 * nrows, 1e-6 * nrows, 0])
        ref = F @ Cm @ F.T + Q
        out = orc.transport(pack(p, Cm), float(dx), nrows)
        _, Co = unpack(out)
        scale = np.sqrt(np.outer(np.diag(ref), np.diag(ref)))
        assert np.abs(Co - ref).max() / scale.max() < 1e-4
        assert np.all(np.abs(Co - ref) <= 2e-4 * scale + 1e-12)


# ------------------------------------------------------------------ update (G17, G19)
def test_update_equals_textbook_kalman(orc):
    rng = np.random.default_rng(9)
    H = np.zeros((2, 5)); H[0, 0] = H[1, 1] = 1.0
    V = np.diag([0.0144, 0.0144])
    for _ in range(30):
        A = rng.normal(size=(5, 5)) * np.array([0.2, 0.2, 0.03, 0.05, 2e-4])[:, None]
        Cm = A @ A.T + np.diag([1e-3, 1e-3, 1e-5, 1e-5, 1e-9])
        p = np.array([rng.uniform(-10, 10), rng.uniform(0, 200), rng.uniform(-0.5, 0.5), rng.uniform(-1, 1), 1e-3])
        pin = pack(p, Cm)
        p32, C32 = unpack(pin)                                      # what the oracle really got (fp32 inputs)
        m = np.array([p32[0] + rng.normal(0, 0.3), p32[1] + rng.normal(0, 0.3)])
        m = m.astype(f32).astype(np.float64)
        S = H @ C32 @ H.T + V
        K = C32 @ H.T @ np.linalg.inv(S)
        r = m - H @ p32
        p_ref = p32 + K @ r
        C_ref = (np.eye(5) - K @ H) @ C32
        chi2_ref = r @ np.linalg.inv(S) @ r
        out, chi2 = orc.update(pin, float(m[0]), float(m[1]))
        po, Co = unpack(out)
        assert chi2 == pytest.approx(chi2_ref, rel=2e-4)
        assert np.allclose(po, p_ref, rtol=1e-4, atol=1e-6)
        scale = np.sqrt(np.outer(np.diag(C32), np.diag(C32)))
        assert np.all(np.abs(Co - C_ref) <= 1e-4 * scale)


def test_structural_zeros_of_decoupled_filter(oracle_run):
    # With dz'/ds, dz'/dk neglected (G16) and a diagonal prior (G15) the (y, s, k) and (z, t)
    # sub-filters never couple: six covariance elements are exactly zero on every tracklet.
    _, r = oracle_run(2)
    zero = [IDX.index(ij) for ij in [(1, 0), (2, 1), (3, 0), (3, 2), (4, 1), (4, 3)]]
    assert np.all(r.cov[:, zero] == 0.0)
    assert np.all(r.cov[:, [IDX.index((i, i)) for i in range(5)]] > 0.0)


# ------------------------------------------------------------------ whole construction
def _single_sector_event(n, sigma, seed, pt_lo=0.5, pt_hi=5.0):
    cfg = replace(CONFIGS[1], n_primaries=n, sigma_yz=sigma, pt_lo=pt_lo, pt_hi=pt_hi)
    return generate_event(cfg, seed)


def _truth_at_first_row(ev, trk, ids):
    """Analytic (y, z, sinphi, dzds, qpt) of the track's truth helix at its x_ref row."""
    cl = ids[trk["first_cluster"]: trk["first_cluster"] + trk["n_clusters"]]
    tid = np.bincount(ev.truth_id[cl]).argmax()
    c0 = cl[0]
    if ev.truth_id[c0] != tid:          # first cluster taken from a crossing track: no truth at x_ref
        return tid, None
    tr = ev.tracks
    return tid, np.array([ev.true_y[c0], ev.true_z[c0], ev.true_sinphi[c0], tr["tanl"][tid], tr["q"][tid] / tr["pt"][tid]])


def test_noise_free_helices_recovered():
    ev = _single_sector_event(25, 0.0, 21)
    o = Oracle.for_geometry(ev.geometry)
    r = o.run(ev.xyz, ev.row_start)
    R = ev.geometry.n_rows
    n_true = np.bincount(ev.truth_id, minlength=25)
    assert len(r.tracks) == (n_true >= 30).sum() >= 18   # every findable helix, once
    seen = set()
    for trk in r.tracks:
        tid, ref = _truth_at_first_row(ev, trk, r.track_cluster_ids)
        seen.add(tid)
        cl = r.track_cluster_ids[trk["first_cluster"]: trk["first_cluster"] + trk["n_clusters"]]
        assert np.all(ev.truth_id[cl] == tid)
        assert trk["n_clusters"] == n_true[tid]                     # all crossed rows collected
        got = np.array([trk["y"], trk["z"], trk["sinphi"], trk["dzds"], trk["qpt"]], np.float64)
        assert trk["x_ref"] == ev.xyz[cl[0], 0]
        assert np.allclose(got[:2], ref[:2], atol=2e-3)
        assert np.allclose(got[2:4], ref[2:4], rtol=2e-3, atol=2e-4)
        assert got[4] == pytest.approx(ref[4], rel=2e-2, abs=2e-3)
    assert len(seen) == len(r.tracks)


def test_pulls_and_chi2_on_smeared_tracks():
    # Smearing sigma equal to the assumed error, Q = 0: chi2/ndf ~ 1 and unit pulls.  30 tracks per
    # sector keep crossings (wrong-cluster outliers) rare; widths are the central-68% half width.
    pulls, chi2ndf = [], []
    for seed in range(40, 56):
        ev = _single_sector_event(30, 0.12, seed)
        o = Oracle.for_geometry(ev.geometry, q_sinphi=0.0, q_dzds=0.0)
        r = o.run(ev.xyz, ev.row_start)
        for trk in r.tracks:
            if trk["n_clusters"] < 100:
                continue
            _, ref = _truth_at_first_row(ev, trk, r.track_cluster_ids)
            if ref is None:
                continue
            cov = trk["cov"]
            kbz = KB * 0.5
            got = np.array([trk["y"], trk["z"], trk["sinphi"], trk["dzds"], trk["qpt"]], np.float64)
            sig = np.sqrt([cov[0], cov[2], cov[5], cov[9], cov[14] / kbz ** 2])
            pulls.append((got - ref) / sig)
            chi2ndf.append(trk["chi2"] / (2 * trk["n_clusters"] - 5))
    pulls = np.array(pulls)
    assert len(pulls) > 350
    q = np.percentile(pulls, [16, 50, 84], axis=0)
    w = (q[2] - q[0]) / 2
    # y, sinphi, qpt: unit pulls; z, dzds only approximately (neglected Jacobian terms, G16)
    assert np.all(np.abs(w[[0, 2, 4]] - 1.0) < 0.12), w
    assert np.all(np.abs(w[[1, 3]] - 1.0) < 0.2), w
    assert np.all(np.abs(q[1]) < 0.15), q[1]
    assert np.mean(chi2ndf) == pytest.approx(1.0, abs=0.05)


# ------------------------------------------------------------------ the filter as a straight-line fit (closed form)
def _wls(A, b, w):
    N = A.T @ (w[:, None] * A)
    return np.linalg.solve(N, A.T @ (w * b)), np.linalg.inv(N)


@pytest.mark.parametrize("y0,m,c", [(-20.0, 0.25, 0.0), (3.0, 0.0, 0.6)])
def test_kappa_frozen_filter_is_the_weighted_least_squares_line_fit(y0, m, c):
    """Textbook special case: with kappa frozen at 0 (c0_kappa = 0) and no process noise the
    model is a straight line, and a Kalman filter over a set of points IS the weighted least-squares fit of that
    set with its prior as pseudo-measurements.  One straight track, one cluster on each of rows 10..120, smeared
    by 30 um so that the filter's linearisation point (it fits sin phi, the line is linear in tan phi) is exact
    to ~1e-6; the assumed errors stay 0.12 cm.  What the construction must then reproduce, written as two
    numpy least-squares problems in float64:
      up pass (G15, G22.1): the seed chain starts on row 11 (row 10 has no links), the first chain cluster is the
        prior of (y, z), so the state at the top row is the line fit of the clusters of rows 11..120;
      down pass (G22.2): prior = that state with the variances reset to (err_y2, err_z2, c0_sinphi, c0_dzds),
        then ALL clusters of rows 120..10 (row 10 is picked up below the seed) -> the track parameters at
        x_ref = x[10] = fit of 111 points + 2 pseudo-measurements at the top row, covariance = (A^T W A)^-1,
        chi2 = the minimum of the weighted sum of squares (prior terms included).
    The two cases separate what the y fit and the z fit depend on: (m = 0.25, dz/ds = 0) has an inclined
    track and a flat z, (m = 0, dz/ds = 0.6) the reverse (z' = z + t ds uses the CURRENT sin phi in ds — G16
    neglects dz'/ds — so with both inclined the filter differs from the joint fit at the 1e-4 cm level)."""
    geo = Geometry(n_sectors=1)
    R, X = geo.n_rows, geo.row_x.astype(np.float64)
    rows = np.arange(10, 121)
    rng = np.random.default_rng(3)
    xs = X[rows]
    path = (xs - xs[0]) * np.sqrt(1 + m * m)
    y = (y0 + m * xs + rng.normal(0, 0.003, len(rows))).astype(f32)
    z = (30.0 + c * path + rng.normal(0, 0.003, len(rows))).astype(f32)
    xyz = np.stack([xs.astype(f32), y, z], 1)
    cnt = np.zeros(R, np.int64); cnt[rows] = 1
    rs = np.zeros(R + 1, np.uint32); rs[1:] = np.cumsum(cnt)
    r = Oracle.for_geometry(geo, c0_kappa=0.0, q_sinphi=0.0, q_dzds=0.0).run(xyz, rs)
    assert len(r.tracks) == 1
    tk = r.tracks[0]
    assert (tk["first_row"], tk["last_row"], tk["n_clusters"]) == (10, 120, 111) and tk["qpt"] == 0.0
    y, z = y.astype(np.float64), z.astype(np.float64)
    err2, c0s, c0t = 0.0144, 0.25, 1.0
    w_meas = np.full(len(xs), 1.0 / err2)
    # up pass: line through the clusters of rows 11..120, at the top row
    A = np.stack([np.ones(len(xs) - 1), xs[1:] - xs[-1]], 1)
    (y_top, T_up), _ = _wls(A, y[1:], w_meas[1:])
    A = np.stack([np.ones(len(xs) - 1), (xs[1:] - xs[-1]) * np.sqrt(1 + T_up ** 2)], 1)
    (z_top, t_up), _ = _wls(A, z[1:], w_meas[1:])
    # down pass: all 111 clusters + the reset prior at the top row; sigma(tan phi) = sigma(sin phi) / cos^3
    cos_up = 1.0 / np.sqrt(1 + T_up ** 2)
    A = np.vstack([np.stack([np.ones(len(xs)), xs - xs[0]], 1), [1.0, xs[-1] - xs[0]], [0.0, 1.0]])
    (y_ref, T), Cy = _wls(A, np.r_[y, y_top, T_up], np.r_[w_meas, 1 / err2, cos_up ** 6 / c0s])
    chi2 = np.sum(np.r_[w_meas, 1 / err2, cos_up ** 6 / c0s] * (A @ [y_ref, T] - np.r_[y, y_top, T_up]) ** 2)
    S = (xs - xs[0]) * np.sqrt(1 + T * T)
    A = np.vstack([np.stack([np.ones(len(xs)), S], 1), [1.0, S[-1]], [0.0, 1.0]])
    (z_ref, t), Cz = _wls(A, np.r_[z, z_top, t_up], np.r_[w_meas, 1 / err2, 1 / c0t])
    chi2 += np.sum(np.r_[w_meas, 1 / err2, 1 / c0t] * (A @ [z_ref, t] - np.r_[z, z_top, t_up]) ** 2)
    cos = 1.0 / np.sqrt(1 + T * T)
    assert tk["y"] == pytest.approx(y_ref, abs=2e-5) and tk["z"] == pytest.approx(z_ref, abs=2e-5)
    assert tk["sinphi"] == pytest.approx(T * cos, abs=2e-6) and tk["dzds"] == pytest.approx(t, abs=2e-6)
    cov = tk["cov"]
    assert cov[0] == pytest.approx(Cy[0, 0], rel=5e-4) and cov[2] == pytest.approx(Cz[0, 0], rel=5e-4)
    assert cov[5] == pytest.approx(Cy[1, 1] * cos ** 6, rel=5e-4) and cov[3] == pytest.approx(Cy[0, 1] * cos ** 3, rel=5e-4)
    assert cov[9] == pytest.approx(Cz[1, 1], rel=5e-4) and cov[7] == pytest.approx(Cz[0, 1], rel=5e-4)
    assert tk["chi2"] == pytest.approx(chi2, rel=1e-3)


@pytest.mark.parametrize("cfg", [1, 2, 3])
def test_pickup_grid_equals_rowscan(event, oracle_run, cfg):
    ev, grid = oracle_run(cfg)
    scan = Oracle.for_geometry(ev.geometry).run(ev.xyz, ev.row_start, mode=MODE_ROWSCAN)
    assert np.array_equal(grid.hits, scan.hits)
    assert np.array_equal(grid.params, scan.params) and np.array_equal(grid.chi2, scan.chi2)
    assert np.array_equal(grid.track_cluster_ids, scan.track_cluster_ids)
    assert np.array_equal(grid.near, scan.near)                     # the G29 audit log does not depend on the grid either


@pytest.mark.parametrize("cfg", [1, 2, 3])
def test_tracklet_invariants(oracle_run, cfg):
    ev, r = oracle_run(cfg)
    R = ev.geometry.n_rows
    rs = ev.row_start.astype(np.int64)
    T = len(r.nhits)
    assert r.hits.shape == (T, R)
    full = 0
    for t in range(T):
        h = r.hits[t]
        rows = np.nonzero(h >= 0)[0]
        assert len(rows) == r.nhits[t]
        assert rows[0] == r.first_row[t] and rows[-1] == r.last_row[t]
        sr = r.tracklet_sector[t] * R + rows                        # one hit per row, on that row
        assert np.all((h[rows] >= rs[sr]) & (h[rows] < rs[sr + 1]))
        c = int(r.start_cluster[t])                                 # chain clusters inside the fitted range are hits
        k = int(np.searchsorted(rs, c, side="right") - 1) % R
        n_in = 0
        while c >= 0:
            if r.first_row[t] <= k <= r.last_row[t]:
                assert h[k] == c
                n_in += 1
            c, k = r.up[c], k + 1
        full += n_in == r.chain_len[t]
    assert full >= 0.97 * T                                         # truncation (transport failure) is rare
    assert np.all(np.isfinite(r.params)) and np.all(np.abs(r.params[:, 2]) <= 0.95)


# ------------------------------------------------------------------ selection and output (G26-G28)
def _greedy_reference(r, R, min_clusters=30):
    """L46/L78 read sequentially: tracklets by (longest, then first); a cluster goes to the first taker."""
    owner = {}
    kept = np.zeros(len(r.nhits), np.int64)
    lists = {}
    for s in np.unique(r.tracklet_sector):
        ts = np.nonzero(r.tracklet_sector == s)[0]
        order = sorted(ts, key=lambda t: (-int(r.nhits[t]), t))
        for t in order:
            if r.nhits[t] < min_clusters:
                continue
            mine = []
            for k in range(R):
                h = r.hits[t, k]
                if h >= 0 and h not in owner:
                    owner[h] = t
                    mine.append(h)
            kept[t] = len(mine)
            lists[t] = mine
    return kept, lists


@pytest.mark.parametrize("cfg", [1, 2, 3])
def test_selection_equals_sequential_greedy(oracle_run, cfg):
    ev, r = oracle_run(cfg)
    R = ev.geometry.n_rows
    kept, lists = _greedy_reference(r, R)
    assert np.array_equal(kept, r.kept)
    kbz = f32(KB * 0.5)
    qpt = np.abs(r.params[:, 4] / kbz)
    acc = (kept >= 30) & (qpt <= 1.0 / 0.05)
    assert np.array_equal(acc, r.accepted.astype(bool))
    tk = r.tracks
    assert len(tk) == acc.sum()
    for trk, t in zip(tk, np.nonzero(acc)[0]):                      # output in tracklet-id order (G28)
        cl = r.track_cluster_ids[trk["first_cluster"]: trk["first_cluster"] + trk["n_clusters"]]
        assert cl.tolist() == lists[t]
        assert trk["seed_cluster"] == r.start_cluster[t]
        assert trk["sector"] == r.tracklet_sector[t]


@pytest.mark.parametrize("cfg", [1, 2, 3])
def test_output_invariants(oracle_run, cfg):
    ev, r = oracle_run(cfg)
    tk, ids = r.tracks, r.track_cluster_ids
    assert len(np.unique(ids)) == len(ids)                          # no cluster in two tracks
    assert np.all(tk["n_clusters"] >= 30)                           # L116
    assert np.all(np.abs(tk["qpt"]) <= 1.0 / 0.05)
    assert tk["n_clusters"].sum() == len(ids)
    assert np.array_equal(tk["first_cluster"], np.concatenate([[0], np.cumsum(tk["n_clusters"])[:-1]]))
    R = ev.geometry.n_rows
    sr = np.searchsorted(ev.row_start.astype(np.int64), ids, side="right") - 1
    for trk in tk:
        a = trk["first_cluster"]
        rows = sr[a:a + trk["n_clusters"]]
        assert np.all(np.diff(rows) > 0) and np.all(rows // R == trk["sector"])


def test_whole_chain_efficiency_config1(oracle_run):
    ev, r = oracle_run(1)
    tid = ev.truth_id
    n_true = np.bincount(tid, minlength=100)
    findable = set(np.nonzero(n_true >= 30)[0].tolist())
    found = set()
    for trk in r.tracks:
        cl = r.track_cluster_ids[trk["first_cluster"]: trk["first_cluster"] + trk["n_clusters"]]
        v, c = np.unique(tid[cl], return_counts=True)
        assert c.max() >= 0.8 * len(cl)                             # no fakes
        found.add(int(v[c.argmax()]))
    assert len(findable & found) >= 0.99 * len(findable)


def test_weighted_selection_alpha_infinity_is_length_rule(event, oracle_run):
    # L88-L94: alpha = infinity "results in the old behavior where only the tracklet length is decisive"
    ev, ref = oracle_run(2)
    r = Oracle.for_geometry(ev.geometry, select_mode=1, alpha=1e12).run(ev.xyz, ev.row_start)
    assert np.array_equal(r.kept, ref.kept)
    assert np.array_equal(r.track_cluster_ids, ref.track_cluster_ids)
    r6 = Oracle.for_geometry(ev.geometry, select_mode=1, alpha=6.0).run(ev.xyz, ev.row_start)
    assert len(np.unique(r6.track_cluster_ids)) == len(r6.track_cluster_ids)
    assert abs(len(r6.tracks) - len(ref.tracks)) < 0.05 * len(ref.tracks)


def _weighted_reference(r, R, alpha, min_clusters=30):
    """L80-L94 read sequentially (the mode-1 twin of _greedy_reference): per sector, tracklets in the order of
    decreasing weight w = n (alpha - chi2 / ndf), beta = ndf = 2 n - 5 (DESIGN.md step 6), ties -> lower id;
    a cluster goes to the first taker.  w is evaluated in fp32, one rounding per operation, as the specification
    writes it."""
    owner = {}
    kept = np.zeros(len(r.nhits), np.int64)
    lists = {}
    for s in np.unique(r.tracklet_sector):
        ts = np.nonzero(r.tracklet_sector == s)[0]
        n = r.nhits[ts].astype(f32)
        with np.errstate(divide="ignore", invalid="ignore"):
            w = n * (f32(alpha) - r.chi2[ts].astype(f32) / (f32(2.0) * n - f32(5.0)))
        for i in sorted(range(len(ts)), key=lambda i: (-float(w[i]), i)):
            t = ts[i]
            if r.nhits[t] < min_clusters:
                continue
            mine = [h for h in r.hits[t] if h >= 0 and h not in owner]
            for h in mine:
                owner[h] = i + 1                                   # what the oracle reports in mode 1: local id + 1
            kept[t] = len(mine)
            lists[t] = mine
    return kept, lists, owner


@pytest.mark.parametrize("cfg", [2, 3])
@pytest.mark.parametrize("alpha", [6.0, 2.0])
def test_weighted_selection_equals_sequential_reference(oracle_run, cfg, alpha):
    """NEXT-1 ("a cluster weight w is implemented as w = n (alpha - chi2 / beta) ... The clusters are
    then assigned to the tracks such that the cluster weights are maximum"), alpha = 6 (L94) and a stronger chi2
    influence, alpha = 2."""
    ev, r = oracle_run(cfg, select_mode=1, alpha=alpha)
    R = ev.geometry.n_rows
    kept, lists, owner = _weighted_reference(r, R, alpha)
    assert np.array_equal(kept, r.kept)
    own = np.zeros(ev.n_clusters, np.uint32)
    own[list(owner.keys())] = list(owner.values())
    assert np.array_equal(own, r.owner)
    acc = r.accepted.astype(bool)
    assert len(r.tracks) == acc.sum() > 100
    for trk, t in zip(r.tracks, np.nonzero(acc)[0]):
        cl = r.track_cluster_ids[trk["first_cluster"]: trk["first_cluster"] + trk["n_clusters"]]
        assert cl.tolist() == lists[t]
    if alpha == 2.0:                                               # the chi2 term does decide something
        _, ref = oracle_run(cfg)
        assert not np.array_equal(r.kept, ref.kept)


def test_weighted_selection_prefers_the_better_fit_at_equal_length(oracle_run):
    """What L86-L88 ask of the weight, checked without the formula: of two tracklets of the SAME length that
    share clusters ("two tracklets with almost identical clusters"), the one with the smaller chi2 gets them
    ("keep the better tracklet"), whichever was constructed first; under the length rule the first one does
    (L78).  A flipped sign of the chi2 term would hand them to the worse fit."""
    ev, r = oracle_run(2, select_mode=1, alpha=6.0)
    _, r0 = oracle_run(2)
    assert np.array_equal(r.hits, r0.hits) and np.array_equal(r.chi2, r0.chi2)     # construction does not depend on the mode
    R = ev.geometry.n_rows
    claim = r.nhits >= 30
    by_cluster = {}
    for t in np.nonzero(claim)[0]:
        for h in r.hits[t][r.hits[t] >= 0]:
            by_cluster.setdefault(int(h), []).append(int(t))
    first = np.searchsorted(r.tracklet_sector, r.tracklet_sector)   # first tracklet of the sector (ids are sector-major)
    n_pairs = n_later = 0
    for h, ts in by_cluster.items():
        if len(ts) != 2 or r.nhits[ts[0]] != r.nhits[ts[1]] or r.chi2[ts[0]] == r.chi2[ts[1]]:
            continue
        better = min(ts, key=lambda t: float(r.chi2[t]))
        n_pairs += 1
        n_later += better == ts[1]
        assert r.owner[h] == better - first[better] + 1
        assert r0.owner[h] == (int(r0.nhits[ts[0]]) << 24 | (0xFFFFFF - (ts[0] - first[ts[0]])))
    assert n_pairs > 200 and n_later > 50


# ------------------------------------------------------------------ second selection round (NEXT-4, G26b)
def _second_round_reference(r1, R, min_clusters=30):
    """G26b written out sequentially from the first round's arrays: only accepted tracklets take part,
    by (longest, then first) per sector; a cluster goes to the first taker."""
    owner = {}
    kept = np.zeros(len(r1.nhits), np.int64)
    lists = {}
    for s in np.unique(r1.tracklet_sector):
        ts = np.nonzero((r1.tracklet_sector == s) & (r1.accepted != 0))[0]
        for t in sorted(ts, key=lambda t: (-int(r1.nhits[t]), t)):
            mine = [h for h in r1.hits[t] if h >= 0 and h not in owner]
            for h in mine:
                owner[h] = t
            kept[t] = len(mine)
            lists[t] = mine
    return kept, lists, owner


@pytest.mark.parametrize("cfg", [2, 3])
def test_second_selection_round(oracle_run, cfg):
    """PAPER.md L46 (selection, then cuts); G26b: the clusters a rejected tracklet had won are
    released and go to accepted tracklets holding them.  Pinned against the sequential definition applied
    to the FIRST round's arrays, and by what must hold: same accepted set, nobody loses a cluster."""
    ev, r1 = oracle_run(cfg)
    ev, r2 = oracle_run(cfg, select_rounds=2)
    R = ev.geometry.n_rows
    assert np.array_equal(r1.hits, r2.hits) and np.array_equal(r1.nhits, r2.nhits)      # construction is untouched
    assert np.array_equal(r1.accepted, r2.accepted)
    acc = r1.accepted != 0
    assert np.all(r2.kept[acc] >= r1.kept[acc]) and np.all(r2.kept[~acc] == 0)
    kept, lists, owner = _second_round_reference(r1, R)
    assert np.array_equal(kept, r2.kept)
    assert len(r2.tracks) == acc.sum()
    for trk, t in zip(r2.tracks, np.nonzero(acc)[0]):
        cl = r2.track_cluster_ids[trk["first_cluster"]: trk["first_cluster"] + trk["n_clusters"]]
        assert cl.tolist() == lists[t]
    # every cluster of a first-round track is still in the same track; released clusters are either re-assigned
    # to an accepted tracklet that holds them or free (owner 0)
    ids1, ids2 = r1.track_cluster_ids, r2.track_cluster_ids
    assert len(np.unique(ids2)) == len(ids2) and set(ids1.tolist()) <= set(ids2.tolist())
    owned2 = np.nonzero(r2.owner)[0]
    assert set(owned2.tolist()) == set(owner.keys())
    if cfg == 2:
        assert len(ids2) > len(ids1)                                  # the dense sector does release clusters


@pytest.mark.parametrize("cfg", [2, 3])
def test_two_construction_passes_are_converged(oracle_run, event, cfg):
    """extrapolate, pick up, refit "until no more clusters are found".  DESIGN.md G22 stops after the up and
    the down pass; the oracle's diagnostic simulates a third pass for every tracklet: for the tracklets that become
    tracks it would add less than 0.1 % more clusters, even in the dense, kinked, lossy sector of config 2."""
    ev, r = oracle_run(cfg)
    o = Oracle.for_geometry(ev.geometry)
    o.run(ev.xyz, ev.row_start, fetch=False)
    g = o.third_pass_gain(ev.xyz, len(r.nhits)) & np.uint32(0x7fffffff)
    acc = r.accepted != 0
    assert g[acc].sum() < 1e-3 * r.nhits[acc].sum()
    # how many tracks would gain at least one cluster is a diagnostic, not a pin: no reading fixes a bound for it
    print(f"config {cfg}: {100 * (g[acc] > 0).mean():.2f} % of the tracks would gain a cluster in a third pass")
    assert g.sum() < 0.02 * r.nhits.sum()                           # all tracklets, including the ones selection drops
