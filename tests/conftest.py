import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


def pytest_sessionstart(session):
    """Make sure the in-tree native pieces exist (no-ops when up to date): the CUDA library (nvcc, sm_100a) and the
    oracle (g++).  A failure here is reported by the tests that need them, loudly -- there is no fallback."""
    try:
        from paper_1810_01609_b200 import build
        build.build()
    except Exception as e:  # pragma: no cover
        sys.stderr.write("conftest: building libmdwf.so failed: %s\n" % (e,))
    try:
        import oracle
        oracle.build()
    except Exception as e:  # pragma: no cover
        sys.stderr.write("conftest: building the oracle failed: %s\n" % (e,))


@pytest.fixture(scope="session")
def has_cuda():
    import torch
    return torch.cuda.is_available()
