import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


def pytest_sessionstart(session):
    """A checkout without the built library (it is git-ignored): compile it once with nvcc.  A build step,
    not a fallback: if nvcc fails the tests that need the library fail loudly."""
    from paper_2403_09990_b200 import build as build_mod
    if not os.path.exists(build_mod.LIB):
        build_mod.build_library()


@pytest.fixture(scope="session")
def golden_dir():
    return os.path.join(ROOT, "tests", "golden")
