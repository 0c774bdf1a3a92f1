import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "slow: minutes of oracle time; left out with HAWKES_SKIP_SLOW_TESTS=1")


@pytest.fixture(scope="session")
def has_cuda():
    import torch
    return torch.cuda.is_available()
