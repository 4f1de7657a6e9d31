import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "slow: statistical pins that take tens of seconds")


@pytest.fixture(autouse=True, scope="session")
def _single_thread_blas():
    # multi-threaded OpenBLAS is slower than one thread on the small matmuls the oracle issues
    try:
        import threadpoolctl
        with threadpoolctl.threadpool_limits(1):
            yield
    except ImportError:
        yield
