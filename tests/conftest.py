import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)
HERE = os.path.dirname(os.path.abspath(__file__))
if HERE not in sys.path:
    sys.path.insert(0, HERE)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "slow: opt-in full-size oracle runs (MM_SLOW=1)")


def pytest_collection_modifyitems(config, items):
    if os.environ.get("MM_SLOW") == "1":
        return
    skip = pytest.mark.skip(reason="set MM_SLOW=1 to run full-size oracle comparisons")
    for it in items:
        if "slow" in it.keywords:
            it.add_marker(skip)
