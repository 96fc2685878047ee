import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _ensure_built():
    """Compile libkinnet.so (nvcc cross-compiles without a GPU) when it is missing
    or stale; build.py is loaded by path because the package refuses to import
    without the library."""
    import importlib.util

    path = os.path.join(ROOT, "paper_1409_5826_b200", "build.py")
    spec = importlib.util.spec_from_file_location("_kinnet_build", path)
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    mod.build()


def pytest_configure(config):
    _ensure_built()
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def hub150():
    from gen.configs import network

    return network("hub150")


@pytest.fixture(scope="session")
def g16():
    from gen.configs import network

    return network("g16")
