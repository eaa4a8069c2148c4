import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a B200 (sm_100a) GPU; run with -m gpu on the GPU box")


@pytest.fixture(scope="session")
def built_lib():
    """Build libnbsdf.so (nvcc cross-compiles without a GPU) and return its path."""
    from paper_2406_17782_b200 import buildlib
    return buildlib.build()
