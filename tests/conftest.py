import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


_EVENTS = {}
_ORACLE = {}


@pytest.fixture(scope="session")
def event():
    """event(config, seed=None) -> cached tpcsynth Event."""
    from tpcsynth import generate_event

    def get(config, seed=None):
        key = (config, seed)
        if key not in _EVENTS:
            _EVENTS[key] = generate_event(config, seed)
        return _EVENTS[key]
    return get


@pytest.fixture(scope="session")
def oracle_run(event):
    """oracle_run(config, seed=None, mode=0, **cuts) -> (Event, OracleResult), cached."""
    from oracle import Oracle

    def get(config, seed=None, mode=0, n_threads=1, **cuts):
        key = (config, seed, mode, tuple(sorted(cuts.items())))
        if key not in _ORACLE:
            ev = event(config, seed)
            o = Oracle.for_geometry(ev.geometry, **cuts)
            _ORACLE[key] = (ev, o.run(ev.xyz, ev.row_start, mode=mode, n_threads=n_threads))
        return _ORACLE[key]
    return get
