import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_addoption(parser):
    parser.addoption("--full-parity", action="store_true", default=False,
                     help="GPU parity on the full SURVEY.md §8(d) parity set for g g > t t~ g g g as well "
                          "(first 16384 events + the 1024 hardest; ~10 minutes of oracle time)")


@pytest.fixture(scope="session")
def full_parity(request):
    return request.config.getoption("--full-parity")


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "slow: longer oracle runs (still CPU-only)")


@pytest.fixture(scope="session")
def oracle():
    from oracle import oracle as O
    return O.load(False)


@pytest.fixture(scope="session")
def oracle_ld():
    from oracle import oracle as O
    return O.load(True)
