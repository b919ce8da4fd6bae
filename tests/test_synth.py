"""Generator checks (inputs only): closed-form helix crossings, determinism, layout."""
import numpy as np

from tpcsynth import CONFIGS, NOISE_ID, generate_event, row_x_table


def test_row_radii_closed_form():
    # BASELINE.json configs[0]: 84.85 cm, 63 rows @0.75, 64 @1.0, 32 @1.5  (G1)
    x = row_x_table()
    assert x.size == 159
    assert abs(x[0] - 84.85) < 1e-12 and abs(x[62] - 131.35) < 1e-9
    assert abs(x[126] - 195.35) < 1e-9 and abs(x[158] - 243.35) < 1e-9
    assert np.all(np.diff(x) > 0)


def test_config1_matches_analytic_helix(event):
    ev = event(1)
    tr, tid = ev.tracks, ev.truth_id
    x = ev.xyz[:, 0].astype(np.float64)
    k, p0, tl = tr["kappa"][tid], tr["phi0"][tid], tr["tanl"][tid]
    sp = np.sin(p0) + k * x                      # sin(phi_k) = sin(phi_0) + kappa x_k
    ph = np.arcsin(sp)
    y = (np.cos(p0) - np.cos(ph)) / k
    z = tl * (ph - p0) / k
    assert np.abs(y - ev.true_y).max() < 1e-9
    assert np.abs(z - ev.true_z).max() < 1e-9
    assert np.abs(sp - ev.true_sinphi).max() < 1e-12
    # cluster radius: the point lies on the circle through the origin
    assert abs(np.std(ev.xyz[:, 1] - ev.true_y) - 0.1) < 0.01
    assert abs(np.std(ev.xyz[:, 2] - ev.true_z) - 0.1) < 0.01


def test_layout_and_determinism(event):
    for c in (1, 2, 3):
        ev = event(c)
        S, R = ev.geometry.n_sectors, ev.geometry.n_rows
        rs = ev.row_start.astype(np.int64)
        assert rs.size == S * R + 1 and rs[0] == 0 and rs[-1] == ev.n_clusters
        assert np.all(np.diff(rs) >= 0)
        rows = (np.searchsorted(rs, np.arange(ev.n_clusters), side="right") - 1) % R
        assert np.array_equal(ev.xyz[:, 0], ev.geometry.row_x[rows])
        ymax = ev.geometry.row_x[rows].astype(np.float64) * ev.geometry.tan_half_angle
        sig = ev.truth_id != NOISE_ID
        assert np.all(np.abs(ev.true_y[sig]) <= ymax[sig] * (1 + 1e-9))
    a, b = generate_event(3), generate_event(3)
    assert np.array_equal(a.xyz, b.xyz) and np.array_equal(a.row_start, b.row_start)
    c = generate_event(3, seed=99)
    assert c.n_clusters != a.n_clusters or not np.array_equal(a.xyz, c.xyz)


def test_sizes_match_design_table(event):
    # DESIGN.md "Input recipe" size table (from this generator; SURVEY §8 estimates in brackets)
    assert 12000 < event(1).n_clusters <= 15900
    assert 90000 < event(2).n_clusters < 140000
    assert 100000 < event(3).n_clusters < 140000
    n2 = np.diff(event(2).row_start.astype(np.int64))
    assert n2.max() > 900                       # the dense-row stress case
    assert CONFIGS[4].n_primaries == 20000 and CONFIGS[4].n_secondaries == 3000
