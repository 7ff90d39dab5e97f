import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def oracle():
    """The CPU oracle (test infrastructure), built on demand with gcc."""
    sys.path.insert(0, os.path.join(ROOT, "oracle"))
    try:
        import hough_oracle
    finally:
        sys.path.pop(0)
    hough_oracle.lib()
    return hough_oracle
