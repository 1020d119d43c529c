import os
import sys

import pytest

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "large: full-size C3-C5 parity samples (EMC_TEST_LARGE=1)")


@pytest.fixture(scope="session")
def inputs_cache():
    """Seeded workloads are deterministic; build each once per session."""
    from emc_inputs import make_inputs

    cache = {}

    def get(name, **kw):
        key = (name, tuple(sorted(kw.items())))
        if key not in cache:
            cache[key] = make_inputs(name, **kw)
        return cache[key]

    return get
