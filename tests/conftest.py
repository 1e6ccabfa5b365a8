import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    from oracle import oracle as O
    O.build()          # the checker is plain C; gcc builds it in a second


@pytest.fixture(scope="session")
def O():
    from oracle import oracle as orc
    return orc


@pytest.fixture(scope="session")
def W():
    from paper_2511_17701_b200 import workloads
    return workloads
