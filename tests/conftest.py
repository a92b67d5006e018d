import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session", autouse=True)
def _oracle_threads():
    # The oracle proper is single-threaded; its OpenMP loops are bit-identical for any
    # thread count (see oracle/grmhd_ref.cpp), so the CPU suite uses the host cores.
    from oracle import ref
    ref.set_num_threads(min(8, os.cpu_count() or 1))
    yield
