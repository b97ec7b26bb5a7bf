import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box via gpurun)")


def pytest_collection_modifyitems(config, items):
    # `-m gpu` on a box without CUDA should fail loudly, not silently pass: GPU tests assert on the device
    # themselves (helpers.require_cuda); nothing is auto-skipped here.
    return
