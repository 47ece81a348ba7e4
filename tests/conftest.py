import os
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "slow: full-size oracle runs (set SF_SLOW=1 to enable)")


def pytest_collection_modifyitems(config, items):
    if os.environ.get("SF_SLOW", "0") == "1":
        return
    skip = pytest.mark.skip(reason="full-size oracle run; set SF_SLOW=1")
    for item in items:
        if "slow" in item.keywords:
            item.add_marker(skip)
