import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")


@pytest.fixture(scope="session")
def O():
    """The CPU oracle (built on first use)."""
    from oracle import oracle
    oracle.lib()
    return oracle


@pytest.fixture(scope="session")
def W():
    from paper_2502_02294_b200 import workloads
    return workloads


@pytest.fixture(scope="session")
def IC():
    """The CPU oracle of the initial-condition map (oracle/ic.py)."""
    from oracle import ic
    return ic
