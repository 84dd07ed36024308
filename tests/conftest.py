import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")
    config.addinivalue_line("markers", "slow: long-running parity case (still part of -m gpu)")


@pytest.fixture(scope="session")
def config_cache():
    """Session cache of generated configurations (generation at 32^4 takes ~10 s)."""
    from paper_1206_0675_b200 import inputs

    cache = {}

    def get(name):
        if name not in cache:
            cache[name] = inputs.make_config(name)
        return cache[name]

    return get
