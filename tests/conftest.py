import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")
    # a fresh checkout has no libqcdmd.so (built artefacts are not in the history): compile it once, by path,
    # because the package refuses to import without it (no CPU fallback)
    lib = os.path.join(ROOT, "paper_1212_0785_b200", "libqcdmd.so")
    if not os.path.exists(lib):
        import importlib.util
        spec = importlib.util.spec_from_file_location("_qcdmd_build", os.path.join(ROOT, "paper_1212_0785_b200", "build.py"))
        mod = importlib.util.module_from_spec(spec)
        spec.loader.exec_module(mod)
        mod.build()


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
