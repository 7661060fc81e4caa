import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def mori():
    """The CUDA path through its C ABI; fails loudly when there is no GPU / no built library."""
    import torch
    assert torch.cuda.is_available(), "gpu-marked test run without a CUDA device"
    from paper_2606_00866_b200 import binding
    binding.load()          # raises if libmori.so is missing
    return binding
