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


def pytest_sessionfinish(session, exitstatus):
    """GPU sessions: write the per-component parity figures the A16 gate recorded (tests/parity_metric.py) to
    gpurun_out/parity_table.{json,md} -- the folder that comes back from the GPU box."""
    try:
        import json
        import parity_metric as pm
    except Exception:
        return
    if not pm.ROWS:
        return
    out = os.path.join(ROOT, "gpurun_out")
    os.makedirs(out, exist_ok=True)
    with open(os.path.join(out, "parity_table.json"), "w") as fh:
        json.dump(pm.ROWS, fh, indent=0)
    with open(os.path.join(out, "parity_table.md"), "w") as fh:
        fh.write(pm.table_markdown(pm.ROWS))
