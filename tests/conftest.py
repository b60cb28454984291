import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


def pytest_sessionstart(session):
    """Compile libazint.so in-tree if it is missing or older than its sources (a build step: nvcc cross-compiles
    without a GPU; nothing here runs the product path)."""
    from paper_1412_6367_b200 import build
    build.build()


@pytest.fixture(scope="session")
def oracle():
    from oracle import oracle as O
    O.lib()
    return O


@pytest.fixture(scope="session")
def workloads():
    from paper_1412_6367_b200 import workloads as W
    return W
