import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "slow: long oracle run, skipped unless PRISM_SLOW=1")


def pytest_collection_modifyitems(config, items):
    if os.environ.get("PRISM_SLOW") == "1":
        return
    skip = pytest.mark.skip(reason="set PRISM_SLOW=1 to run")
    for item in items:
        if "slow" in item.keywords:
            item.add_marker(skip)
