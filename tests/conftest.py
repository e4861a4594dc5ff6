"""pytest configuration: registers the `gpu` marker and puts the repo root on sys.path."""
import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")
    config.addinivalue_line("markers", "slow: longer-running case")


@pytest.fixture(scope="session")
def ref():
    """The CPU oracle binding (builds oracle/libmhd_ref.so on first use)."""
    from oracle import mhd_ref
    mhd_ref.lib()
    return mhd_ref
