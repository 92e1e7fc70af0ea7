"""pytest configuration: the `gpu` marker, repo root on sys.path, the oracle built once."""
import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on the B200 box)")


@pytest.fixture(scope="session")
def oracle():
    import oracle as o
    o.lib()          # builds oracle/liboracle.so with g++ if it is stale
    return o


def golden_path(name):
    return os.path.join(ROOT, "tests", "golden", name)
