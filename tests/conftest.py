import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "slow: full-size configuration, minutes on the GPU box")


@pytest.fixture(scope="session")
def cuda_device():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch.device("cuda:0")


def pytest_collection_modifyitems(config, items):
    """The hot-path parity tests run first (a launch trace of the first seconds of the GPU suite then shows the codec's own
    kernels rather than the calibration fit's eigen-solver steps); the order inside a file is kept."""
    items.sort(key=lambda it: 0 if "test_parity_gpu" in it.nodeid else 1)
