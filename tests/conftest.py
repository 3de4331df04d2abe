import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def have_gpu():
    import torch
    return torch.cuda.is_available()


@pytest.fixture(scope="session")
def nsm():
    """The CUDA package with libnsm.so built and loaded; skips without a GPU (the product has no CPU fallback)."""
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_2210_13641_b200 import build
    build.build()
    import paper_2210_13641_b200 as mod
    return mod
