import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu under gpurun")


def pytest_collection_modifyitems(config, items):
    """GPU tests fail loudly (not skip) on a box that has a GPU but no extension; on a
    CPU-only box `-m "not gpu"` deselects them."""
    return
