"""GPU parity on many seeded events and option combinations: the whole result of the CUDA path (tracks, cluster lists,
and the optional outputs) against the oracle, byte for byte, on events the other parity tests never see.

Each case draws an event configuration (pp-like with a random multiplicity and noise level, or the dense single sector
with a random number of tracks), a seed, a grid bin size and a set of options (chi2-weighted selection, second selection
round, iterated passes, global tracking, track merging) from a seeded generator, so the cases are the same on every run.
"""
from dataclasses import replace

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _case(i):
    from tpcsynth import CONFIGS
    rng = np.random.default_rng(1000 + i)
    if rng.random() < 0.6:
        cfg = replace(CONFIGS[3], n_primaries=int(rng.integers(100, 1500)), noise_frac=float(rng.choice([0.0, 0.02, 0.1])),
                      n_secondaries=int(rng.choice([0, 200])))
    else:
        cfg = replace(CONFIGS[2], n_primaries=int(rng.integers(50, 800)), drop_frac=float(rng.choice([0.0, 0.02, 0.08])),
                      noise_frac=float(rng.choice([0.0, 0.1, 0.3])))
    cuts = {}
    if rng.random() < 0.5:
        cuts["bin_y"], cuts["bin_z"] = float(rng.choice([0.8, 1.0, 2.5])), float(rng.choice([2.0, 4.0, 7.0]))
    if rng.random() < 0.4:
        cuts["select_mode"], cuts["alpha"] = 1, float(rng.choice([2.0, 6.0, 20.0]))
    if rng.random() < 0.4:
        cuts["select_rounds"] = 2
    if rng.random() < 0.3:
        cuts["max_row_gap"] = int(rng.choice([2, 6]))
    if rng.random() < 0.3:
        cuts["chi2_cut"] = float(rng.choice([6.0, 16.0]))
    if rng.random() < 0.4:
        cuts["merge_tracks"] = 1
    if rng.random() < 0.35:
        cuts["max_passes"] = int(rng.choice([3, 4, 7]))
    elif rng.random() < 0.5 and cfg.n_sectors == 36:
        cuts["global_tracking"] = 1
    return cfg, int(rng.integers(1, 10 ** 6)), cuts


@pytest.mark.parametrize("i", range(40))
def test_random_events_and_options_equal_the_oracle(i):
    import paper_1712_09407_b200 as t
    from oracle import Oracle
    from tpcsynth import generate_event
    cfg, seed, cuts = _case(i)
    ev = generate_event(cfg, seed)
    o = Oracle.for_geometry(ev.geometry, **cuts).run(ev.xyz, ev.row_start, n_threads=8)
    with t.SectorTracker(ev.geometry, max(ev.n_clusters, 1), max(4096, ev.n_clusters // 4), **cuts) as trk:
        r = trk.track_event(ev.xyz, ev.row_start)
        hits = trk.debug_fetch(t.TPCST_DBG_ROW_HITS).reshape(r.n_tracklets, -1)
        links = trk.debug_fetch(t.TPCST_DBG_LINKS).reshape(2, -1)
    assert np.array_equal(links[0], o.up) and np.array_equal(links[1], o.dn), (i, cuts)
    assert r.n_tracklets == len(o.nhits) and np.array_equal(hits, o.hits), (i, cuts)
    assert np.array_equal(r.cluster_ids, o.track_cluster_ids), (i, cuts)
    assert r.tracks.tobytes() == o.tracks.tobytes(), (i, cuts)
    if cuts.get("merge_tracks"):
        assert r.merge.tobytes() == o.merge.tobytes(), (i, cuts)
    if cuts.get("global_tracking"):
        assert r.global_ext.tobytes() == o.global_ext.tobytes() and np.array_equal(r.global_cluster_ids, o.global_cluster_ids), (i, cuts)
