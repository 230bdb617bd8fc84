import os
import sys

import pytest

# The oracle's OpenMP threads must not spin at their barriers: on a shared or throttled host the default
# (active waiting, one thread per visible core) makes the CPU suite several times slower.  Set before
# libgomp is loaded; affects the tests only (bench.py times the oracle as it stands).
os.environ.setdefault("OMP_WAIT_POLICY", "passive")

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "slow: larger oracle runs")


@pytest.fixture(scope="session")
def oracle_mod():
    import oracle
    oracle.build()
    return oracle
