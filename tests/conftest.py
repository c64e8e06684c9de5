import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "slow: parity at SURVEY.md 8(d)'s parity sizes / full sizes (minutes, not seconds)")


@pytest.fixture(scope="session")
def ora():
    """The oracle binding (compiles oracle/pic_oracle.c with gcc on first use)."""
    from oracle import ora as _ora
    _ora.lib()
    return _ora
