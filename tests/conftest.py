import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def boa():
    """The thin Python binding over the C ABI (loads libboa.so; builds it if missing)."""
    from paper_2511_11337_b200 import boa as _boa
    return _boa
