import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def golden_dir():
    return os.path.join(ROOT, "tests", "golden")


@pytest.fixture(scope="session", autouse=True)
def _library_is_built():
    """Build csrc/libdarts.so for sm_100a if it is missing or stale (nvcc cross-compiles without a GPU).  This is the build step, not a
    fallback: if it fails the session fails, and the binding itself still refuses to import without the library."""
    from paper_2605_30859_b200 import build
    build.build()
