import os
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")
    config.addinivalue_line("markers", "slow: long-running full-size check (enabled with MK_SLOW=1)")


def pytest_collection_modifyitems(config, items):
    if os.environ.get("MK_SLOW", "0") == "1":
        return
    skip = pytest.mark.skip(reason="set MK_SLOW=1 to run the long full-size checks")
    for it in items:
        if "slow" in it.keywords:
            it.add_marker(skip)
