import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on a B200)")


@pytest.fixture(scope="session")
def gpu_lib():
    """The product's Python binding, loaded only for -m gpu tests; fails loudly when the extension is missing."""
    import torch

    if not torch.cuda.is_available():
        pytest.fail("-m gpu test selected but no CUDA device is visible")
    import paper_1902_04934_b200 as ile

    ile.load()
    return ile
