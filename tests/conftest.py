import os
import sys

import pytest

# The oracle's OpenMP threads sleep at the end of a parallel loop instead of spinning (read by libgomp when it is first
# loaded, hence here, before anything imports it): most oracle pins are tiny grids with thousands of short loops, and
# on a shared host whose cores are taken away now and then spinning threads made the CPU suite five to ten times slower.
# Timing is not what tests measure; bench.py's cpu_baseline does not go through here.
os.environ.setdefault("OMP_WAIT_POLICY", "passive")

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
