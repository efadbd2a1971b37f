import os
import sys
import time

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


SESSION_START = time.time()      # tests that take minutes of oracle time look at how much of the run's budget is left


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "slow: full-size parity runs, enabled with SMCX_SLOW=1")


def pytest_collection_modifyitems(config, items):
    if os.environ.get("SMCX_SLOW", "0") == "1":
        return
    skip = pytest.mark.skip(reason="set SMCX_SLOW=1 to run full-size parity")
    for item in items:
        if "slow" in item.keywords:
            item.add_marker(skip)
