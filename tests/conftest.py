import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session", autouse=True)
def _built():
    """Make sure the oracle library and the C-ABI library exist (both compile without a GPU)."""
    from oracle import build as obuild
    obuild.build()
    from paper_1912_04197_b200 import build as pbuild
    try:
        pbuild.build()
    except FileNotFoundError:      # oracle-only checkout: no CUDA sources yet
        pass
    yield
