"""The few values PAPER.md prints (tests/golden/paper_constants.txt, each with its citation) against the
defaults of the oracle, of the CUDA library and of the synthetic geometry."""
import os

import numpy as np

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "paper_constants.txt")


def _golden():
    out = {}
    for line in open(GOLDEN):
        line = line.split("#")[0].split()
        if len(line) == 2:
            out[line[0]] = float(line[1])
    return out


def test_paper_constants_are_the_defaults_on_both_sides():
    g = _golden()
    from oracle.oracle import DEFAULT_CUTS
    from tpcsynth import Geometry
    import paper_1712_09407_b200 as t
    c = t.tpcst_default_cuts()
    assert DEFAULT_CUTS["min_clusters"] == c.min_clusters == g["min_clusters"]
    assert DEFAULT_CUTS["alpha"] == c.alpha == g["alpha"]
    assert DEFAULT_CUTS["gt_max_rows"] == c.gt_max_rows == g["min_clusters"]      # L116 also sizes the global-tracking end region
    geo = Geometry(n_sectors=36)
    assert len(geo.row_x) == g["n_pad_rows"] and geo.n_sectors == g["n_sectors"]
    assert np.isclose(geo.tan_half_angle, np.tan(np.pi / (g["n_sectors"] / 2)))   # 18 sectors per ring: half angle 10 degrees


def test_every_oracle_track_has_at_least_the_papers_minimum_of_clusters(oracle_run):
    g = _golden()
    _, r = oracle_run(3, n_threads=4)
    assert len(r.tracks) > 1000 and r.tracks["n_clusters"].min() >= g["min_clusters"]
