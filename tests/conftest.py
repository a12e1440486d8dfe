import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


def _has_cuda():
    try:
        import torch
        return torch.cuda.is_available()
    except Exception:
        return False


def pytest_collection_modifyitems(config, items):
    # a cooperative kernel that deadlocks would otherwise hang the whole session: every GPU test gets a time limit
    # (pytest-timeout, thread method: the process is ended with a stack dump)
    for it in items:
        if "gpu" in it.keywords and not any(m.name == "timeout" for m in it.iter_markers()):
            it.add_marker(pytest.mark.timeout(600, method="thread"))
    if _has_cuda():
        return
    skip = pytest.mark.skip(reason="no CUDA device")
    for it in items:
        if "gpu" in it.keywords:
            it.add_marker(skip)
