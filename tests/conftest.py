import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def orc():
    """The serial CPU oracle (the definition)."""
    from oracle.oracle import Oracle
    return Oracle(omp=False)


@pytest.fixture(scope="session")
def orc_omp():
    """The OpenMP build of the same oracle source, for the larger lattices."""
    from oracle.oracle import Oracle
    return Oracle(omp=True)
