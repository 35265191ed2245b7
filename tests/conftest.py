import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")
    config.addinivalue_line("markers", "slow: long oracle runs (still part of the default CPU suite unless deselected)")
    config.addinivalue_line("markers", "long: opt-in runs of many minutes (set BZ_LONG=1); no test carries it at present")


def pytest_collection_modifyitems(config, items):
    if os.environ.get("BZ_LONG") == "1":
        return
    skip = pytest.mark.skip(reason="opt-in: set BZ_LONG=1")
    for item in items:
        if item.get_closest_marker("long"):
            item.add_marker(skip)


@pytest.fixture(scope="session")
def golden_dir():
    return os.path.join(ROOT, "tests", "golden")
