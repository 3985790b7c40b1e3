import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "soak: long randomised runs, opt-in: -m 'gpu and soak' (skipped otherwise)")


def pytest_collection_modifyitems(config, items):
    # soak tests run only when the marker expression names them
    if "soak" in (config.getoption("-m") or ""):
        return
    skip = pytest.mark.skip(reason="opt-in: -m 'gpu and soak'")
    for item in items:
        if "soak" in item.keywords:
            item.add_marker(skip)


@pytest.fixture(scope="session")
def oracle():
    from oracle import abm_oracle
    abm_oracle.lib()
    return abm_oracle
