import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "slow: full-size parity case (several minutes)")


@pytest.fixture(scope="session")
def oracle_c():
    """Make sure the C part of the oracle is built (tests that time out without it use this)."""
    from oracle import build as obuild
    obuild.build()
    from oracle import fdd_oracle
    return fdd_oracle
