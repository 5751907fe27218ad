import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")
    config.addinivalue_line("markers", "slow: about an hour of oracle time on the host cores; runs only with IA_RUN_SLOW=1")


def _have_gpu():
    try:
        import torch
        return torch.cuda.is_available()
    except Exception:
        return False


def pytest_collection_modifyitems(config, items):
    if os.environ.get("IA_RUN_SLOW", "0") != "1":
        skip_slow = pytest.mark.skip(reason="slow: set IA_RUN_SLOW=1")
        for item in items:
            if "slow" in item.keywords:
                item.add_marker(skip_slow)
    if _have_gpu():
        return
    skip = pytest.mark.skip(reason="no CUDA device")
    for item in items:
        if "gpu" in item.keywords:
            item.add_marker(skip)
