import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def cuda_lib():
    """The C-ABI library through its Python binding; fails loudly if it cannot run."""
    import torch
    from paper_1807_08116_b200 import binding
    assert torch.cuda.is_available(), "gpu-marked test started without a CUDA device"
    binding.load()
    return binding
