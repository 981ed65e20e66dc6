import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "slow: minutes of CPU-oracle time (step-count parity at the configs' own sizes); "
                                       "part of -m gpu, deselect with -m 'gpu and not slow' while iterating")


@pytest.fixture(scope="session", autouse=True)
def _oracle_threads():
    from oracle import meg6_oracle as O
    O.set_threads(min(8, os.cpu_count() or 1))
    yield
