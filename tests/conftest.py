import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def impurities():
    """Lazily built, cached BASELINE.json impurities (configs 1-4; config 5 is built only on demand)."""
    from workloads import build_config_impurity
    cache = {}

    def get(cfg):
        if cfg not in cache:
            cache[cfg] = build_config_impurity(cfg)
        return cache[cfg]
    return get
