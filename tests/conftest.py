import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    # The oracle (g++) is built first and on its own: its pins (test_oracle_pins.py) need neither
    # nvcc nor libskel.so. The CUDA library is built next (nvcc cross-compiles without a GPU); if
    # that fails, only the modules that import the product package fail, loudly, at import.
    import oracle

    oracle.build()
    try:
        import __graft_entry__ as ge

        ge.build_product()
    except Exception as e:  # noqa: BLE001
        sys.stderr.write(f"[conftest] libskel.so could not be built: {e}\n")
