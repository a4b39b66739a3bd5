import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    # compile the oracle (g++) and the CUDA library (nvcc cross-compiles without a GPU) before
    # collection: test modules import the package at import time
    import __graft_entry__ as ge

    ge.build()
