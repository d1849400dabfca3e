import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


def pytest_collection_modifyitems(config, items):
    try:
        import torch
        has_gpu = torch.cuda.is_available()
    except Exception:
        has_gpu = False
    if has_gpu:
        return
    skip = pytest.mark.skip(reason="no CUDA device")
    for item in items:
        if "gpu" in item.keywords:
            item.add_marker(skip)


import time

_SESSION_T0 = time.time()


@pytest.fixture
def gpu_time_box():
    """Seconds this pytest session has been running.  The round-end GPU run has a 20-minute limit for the whole `-m gpu` suite;
    the one test that takes minutes on its own (BASELINE.json config 5) asks before it starts and skips, saying so, rather
    than let the limit kill the whole run."""
    return lambda: time.time() - _SESSION_T0
