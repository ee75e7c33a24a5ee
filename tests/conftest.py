"""Shared fixtures.  ``-m "not gpu"`` runs here (CPU only); ``-m gpu`` needs a B200."""
import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200, sm_100a)")


@pytest.fixture(scope="session")
def geom():
    import synth
    return synth.make_geometry()


_cache = {}


def workload(config, n_events=None):
    """Cached (geometry, batch, params) for a BASELINE.json config."""
    import synth
    key = (config, n_events)
    if key not in _cache:
        _cache[key] = synth.make_workload(config, n_events=n_events)
    return _cache[key]


@pytest.fixture(scope="session")
def wl():
    return workload
