import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "slow: longer CPU test")


@pytest.fixture(scope="session")
def geo4():
    import oracle
    from paper_1810_11966_b200 import workloads as W
    return oracle.geometry(W.GEOMETRY_4)


@pytest.fixture(scope="session")
def geo6():
    import oracle
    from paper_1810_11966_b200 import workloads as W
    return oracle.geometry(W.GEOMETRY_6)
