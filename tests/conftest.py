import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a real B200 (run with -m gpu)")


def pytest_collection_modifyitems(config, items):
    """GPU tests must never silently pass without a GPU: when one is collected
    without CUDA it is skipped with a loud reason (the driver selects them with
    -m gpu only on a B200 box)."""
    try:
        import torch
        has_cuda = torch.cuda.is_available()
    except Exception:  # pragma: no cover
        has_cuda = False
    if has_cuda:
        return
    skip = pytest.mark.skip(reason="no CUDA device: gpu-marked test not runnable here")
    for item in items:
        if "gpu" in item.keywords:
            item.add_marker(skip)
