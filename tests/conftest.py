import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def oracle_threads():
    """Use every core for the oracle's loops over cells (per-cell arithmetic is unchanged)."""
    from oracle import pyoracle as po
    return po.set_threads(0)
