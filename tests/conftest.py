import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def workloads_cache():
    """Session cache of generated workloads (config 5's scene takes a few seconds)."""
    from paper_2607_04310_b200 import workloads as W
    cache = {}

    def get(idx, **kw):
        key = (idx, tuple(sorted(kw.items())))
        if key not in cache:
            cache[key] = W.make_config(idx, **kw)
        return cache[key]

    return get
