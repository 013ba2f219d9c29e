import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "large: large-lattice GPU case (minutes, tens of GB)")
    config.addinivalue_line("markers", "faultinject: deliberately faults a kernel in a child process (MMU fault on the GPU); run with -m faultinject only")


def pytest_collection_modifyitems(config, items):
    """`-m gpu` must not raise MMU faults on a shared GPU: fault-injection tests run only when -m names them."""
    if "faultinject" in (config.getoption("-m") or ""):
        return
    skip = pytest.mark.skip(reason="faults a kernel on purpose: run with -m faultinject")
    for item in items:
        if "faultinject" in item.keywords:
            item.add_marker(skip)


@pytest.fixture(scope="session", autouse=True)
def _build_oracle():
    import oracle

    oracle.build()
    yield
