import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


def pytest_collection_modifyitems(config, items):
    """Every GPU test gets a time limit (pytest-timeout, thread method: the whole process is ended, which also tears down a
    kernel that never returns -- a hung kernel must cost a test run minutes, not the box).  The largest GPU test takes ~10 s."""
    if not config.pluginmanager.hasplugin("timeout"):
        return
    for item in items:
        if item.get_closest_marker("gpu") and not item.get_closest_marker("timeout"):
            item.add_marker(pytest.mark.timeout(300, method="thread"))


@pytest.fixture(scope="session")
def c1():
    from paper_1302_4000_b200 import workloads
    return workloads.make_config("C1")
