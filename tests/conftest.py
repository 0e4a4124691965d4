import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (runs on the B200 box: pytest -m gpu)")
    config.addinivalue_line("markers", "slow: long oracle pin, only with LBMK_SLOW_PINS=1")


def pytest_collection_modifyitems(config, items):
    if os.environ.get("LBMK_SLOW_PINS") == "1":
        return
    skip = pytest.mark.skip(reason="set LBMK_SLOW_PINS=1 to re-run the N=512 paper pins (minutes)")
    for it in items:
        if "slow" in it.keywords:
            it.add_marker(skip)
