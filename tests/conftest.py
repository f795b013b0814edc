import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "slow: full-size parity cases (minutes of host time)")


@pytest.fixture(scope="session")
def hot():
    """The CUDA library binding; skips when no GPU is visible (the -m gpu tests need one)."""
    import torch

    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1310_4502_b200 as hotlib

    return hotlib
