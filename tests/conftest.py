import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session", autouse=True)
def _blas_threads():
    """OpenBLAS with one thread per core spins badly on the small matrices used here;
    cap the pool for the test session (the oracle itself is not changed)."""
    try:
        from threadpoolctl import threadpool_limits
        with threadpool_limits(limits=4):
            yield
    except ImportError:  # pragma: no cover
        yield


def have_cuda() -> bool:
    try:
        import torch
        return torch.cuda.is_available()
    except Exception:
        return False
