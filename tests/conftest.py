import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box via gpurun)")


@pytest.fixture(scope="session")
def cuda_lib():
    """The C-ABI library; GPU tests fail loudly (never skip to a fallback) if it is missing."""
    import torch
    from paper_2603_08593_b200 import load_library
    assert torch.cuda.is_available(), "gpu-marked test running without a CUDA device"
    return load_library()
