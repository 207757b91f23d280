import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")


def pytest_collection_modifyitems(config, items):
    """A deadlocked kernel (mbarrier byte-count mismatch, a spin on a peer CTA) would otherwise hold the GPU box until
    the outer limit: every GPU test gets a hard per-test timeout (pytest-timeout, thread method = the process is
    killed) unless one is given on the command line."""
    if config.pluginmanager.hasplugin("timeout") and not config.getoption("timeout", None):
        for item in items:
            if item.get_closest_marker("gpu") is not None and item.get_closest_marker("timeout") is None:
                item.add_marker(pytest.mark.timeout(240, method="thread"))


@pytest.fixture(scope="session")
def repo_root():
    return ROOT
