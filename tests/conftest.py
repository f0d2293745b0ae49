import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a real B200 (run with -m gpu under gpurun)")


@pytest.fixture(scope="session", autouse=True)
def _built_library():
    """The CUDA library is git-ignored: (re)build it in-tree when it is missing or older than its sources
    (nvcc cross-compiles without a GPU).  A failed build fails the session loudly; there is no fallback."""
    from paper_2511_22468_b200 import build as build_mod
    build_mod.build()
