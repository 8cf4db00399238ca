import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def refs():
    """Oracle reference elements, built once per session."""
    from oracle.operators import ReferenceElement
    cache = {}

    def get(dim, N):
        if (dim, N) not in cache:
            cache[(dim, N)] = ReferenceElement(dim, N)
        return cache[(dim, N)]
    return get
