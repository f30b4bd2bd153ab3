import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session", autouse=True)
def _built_library():
    """(Re)build the in-tree CUDA library when it is missing or older than its sources."""
    import importlib.util
    spec = importlib.util.spec_from_file_location("awg_build", os.path.join(ROOT, "paper_2403_15582_b200", "build.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    mod.build()


@pytest.fixture(scope="session")
def awg():
    """The CUDA path's Python binding; GPU tests fail loudly if the extension is missing."""
    import paper_2403_15582_b200 as m

    return m
