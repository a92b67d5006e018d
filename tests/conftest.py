import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_addoption(parser):
    parser.addoption("--parity-report", default=None, metavar="PATH",
                     help="write the measured GPU-vs-oracle parity errors to this JSON file")


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


# measured parity errors, appended to by tests/test_gpu_parity.py; written out only on request
PARITY_REPORT = []


def pytest_sessionfinish(session, exitstatus):
    path = session.config.getoption("--parity-report")
    if path and PARITY_REPORT:
        import json
        os.makedirs(os.path.dirname(os.path.abspath(path)), exist_ok=True)
        with open(path, "w") as f:
            json.dump(PARITY_REPORT, f, indent=1)


@pytest.fixture(scope="session", autouse=True)
def _oracle_threads():
    # The oracle proper is single-threaded; its OpenMP loops are bit-identical for any
    # thread count (see oracle/grmhd_ref.cpp), so the CPU suite uses the host cores.
    from oracle import ref
    ref.set_num_threads(min(32, os.cpu_count() or 1))
    yield
