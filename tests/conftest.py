import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def oracle_mod():
    from oracle import oracle as O
    return O


def pytest_sessionstart(session):
    # a fresh checkout has no libnsgw.so (built files are git-ignored): build it once, in-tree, before any test loads it
    from paper_2509_04336_b200 import build
    if os.path.exists(os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")):
        build.build()
