import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


def pytest_collection_modifyitems(config, items):
    """GPU tests fail loudly (not skip) when selected on a box without the device or the library.
    A kernel that deadlocks must not hold the GPU box until the caller's limit: every GPU test gets a 15-minute
    timeout (pytest-timeout, thread method: the process exits even if it is blocked inside a CUDA call)."""
    try:
        import pytest_timeout  # noqa: F401
    except ImportError:
        return
    import pytest
    for item in items:
        if "gpu" in item.keywords and item.get_closest_marker("timeout") is None:
            item.add_marker(pytest.mark.timeout(900, method="thread"))
