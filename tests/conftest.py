import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on a B200)")


def pytest_collection_modifyitems(config, items):
    # a GPU test on a box without a GPU is an error in how the suite was invoked, but the
    # CPU driver always passes -m "not gpu"; skip (loudly) if someone runs the bare suite here.
    try:
        import torch
        has_gpu = torch.cuda.is_available()
    except Exception:  # pragma: no cover
        has_gpu = False
    if has_gpu:
        return
    skip = pytest.mark.skip(reason="no CUDA device in this container")
    for item in items:
        if "gpu" in item.keywords:
            item.add_marker(skip)


@pytest.fixture(autouse=True)
def _device_errors_belong_to_their_test(request):
    """A kernel fault is reported asynchronously, at the next synchronising call: without this, a
    fault in one GPU test would surface in (and be blamed on) a later one."""
    yield
    if "gpu" in request.keywords:
        import torch

        if torch.cuda.is_available():
            torch.cuda.synchronize()
