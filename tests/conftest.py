import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def geometry():
    from paper_1912_09161_b200 import workload

    return workload.geometry_g0()


_BATCH_CACHE = {}


@pytest.fixture(scope="session")
def batch_of():
    """batch_of(config, n_events) -> workload.Batch, cached per session."""
    from paper_1912_09161_b200 import workload

    def get(config, n_events=None, **kw):
        key = (config, n_events, tuple(sorted(kw.items())))
        if key not in _BATCH_CACHE:
            _BATCH_CACHE[key] = workload.generate(config, n_events=n_events, **kw)
        return _BATCH_CACHE[key]

    return get


_ORACLE_CACHE = {}


@pytest.fixture(scope="session")
def oracle_of(batch_of):
    """oracle_of(config, n_events) -> (batch, oracle.Result with pixel membership), cached per session."""
    import oracle

    def get(config, n_events=None, **kw):
        key = (config, n_events, tuple(sorted(kw.items())))
        if key not in _ORACLE_CACHE:
            b = batch_of(config, n_events, **kw)
            _ORACLE_CACHE[key] = (b, oracle.reconstruct(b.geometry, b.raw, b.event_offsets, with_pixels=True,
                                                        n_threads=os.cpu_count() or 1))
        return _ORACLE_CACHE[key]

    return get
